// cc_common.h -- definitions shared by the host plan code (cc_api.cu) and the
// fused device kernel (cc_fused.cuh).  Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

// Mixed-radix decomposition of the in-place FFTs (forward = decimation in
// frequency, natural order in -> "slot" order out; inverse = the transpose,
// slot order in -> natural order out).  N = r[0]*r[1]*r[2].
// Column FFTs (one thread per butterfly, NC columns in parallel) use large radices: fewer sweeps of S.
__host__ __device__ constexpr int cc_radix_col(int N, int p)
{
    return N == 64   ? (p == 0 ? 8 : p == 1 ? 8 : 1)
         : N == 128  ? (p == 0 ? 16 : p == 1 ? 8 : 1)
         : N == 256  ? (p == 0 ? 16 : p == 1 ? 16 : 1)
         : N == 512  ? (p == 0 ? 8 : p == 1 ? 8 : 8)
         : N == 1024 ? (p == 0 ? 16 : p == 1 ? 8 : 8)
                     : 0;
}
// Row FFTs (one warp per FFT) use radices small enough that a pass has >= 32 butterflies where possible:
// all lanes busy instead of N/16 of them.
__host__ __device__ constexpr int cc_radix_row(int N, int p)
{
    return N == 64   ? (p == 0 ? 8 : p == 1 ? 8 : 1)   // four row pairs per warp, 8 lanes each
         : N == 128  ? (p == 0 ? 4 : p == 1 ? 4 : 8)
         : N == 256  ? (p == 0 ? 16 : p == 1 ? 16 : 1)  // two row pairs per warp, 16 lanes each (cc_row_group)
         : N == 512  ? (p == 0 ? 8 : p == 1 ? 8 : 8)
         : N == 1024 ? (p == 0 ? 16 : p == 1 ? 8 : 8)
                     : 0;
}
// Row pairs a warp transforms side by side (32 / cc_row_group lanes each): two passes instead of three at N = 64, 256.
__host__ __device__ constexpr int cc_row_group(int N) { return N == 256 ? 2 : N == 64 ? 4 : 1; }
__host__ __device__ constexpr int cc_radix(int N, int p, bool row) { return row ? cc_radix_row(N, p) : cc_radix_col(N, p); }

// Frequency held by slot p after the forward FFT of length N:
// p = k1*(N/r0) + k2*(N/(r0 r1)) + k3  <->  k = k1 + r0*k2 + r0*r1*k3.
static inline int cc_freq_of_slot(int N, int p, bool row)
{
    int k = 0, mult = 1, L = N, rem = p;
    for (int i = 0; i < 3; ++i) {
        int r = cc_radix(N, i, row);
        if (r <= 1) break;
        L /= r;
        int d = rem / L;
        rem %= L;
        k += d * mult;
        mult *= r;
    }
    return k;
}

// TM1 split into vector chunks: widths 4,4,2 / 4,1 / ... ; chunk ci of thread-row tm1 sits at
// R1 * start(ci) + tm1 * width(ci) inside a staged k-row of MC1 floats.
__host__ __device__ constexpr int cc_tm1_nchunks(int tm1) { return tm1 == 10 ? 3 : (tm1 == 5 || tm1 == 8 || tm1 == 3) ? 2 : 1; }
__host__ __device__ constexpr int cc_tm1_width(int tm1, int ci)
{
    return tm1 == 10 ? (ci < 2 ? 4 : 2) : tm1 == 8 ? 4 : tm1 == 5 ? (ci == 0 ? 4 : 1) : tm1 == 3 ? (ci == 0 ? 2 : 1) : tm1;
}
__host__ __device__ constexpr int cc_tm1_start(int tm1, int ci)
{
    return ci == 0 ? 0 : ci == 1 ? cc_tm1_width(tm1, 0) : cc_tm1_width(tm1, 0) + cc_tm1_width(tm1, 1);
}

// Phases of the per-frame breakdown (cc_track_profile): 0 ingest + row FFT, 1 column FFT (x) conj(G) +
// column inverse, 2 row C2R + integer argmax, 3 fp64 integer polish, 4 upsampled stage 1 (last
// super-block), 5 upsampled stage 2, 6 sub-pixel argmax reduction, 7 fp64 sub-pixel polish.
#define CC_NPHASE 8

// Kernel parameters (passed by value).  All table pointers are device memory
// owned by the plan.
struct CcParams {
    const void *frames;  // batch * H * W pixels
    int batch;
    float *dx, *dy, *peak;  // peak may be null
    int *iy, *ix;           // may be null
    unsigned long long *phase_clk;  // optional [batch][CC_NPHASE] SM-clock cycles per phase, else null

    const float2 *tw;             // [NTW] (cos, -sin)(2 pi j / NTW), NTW = max(H, W)
    const uint16_t *row_slot;     // [W] slot holding row frequency k
    const float2 *Gt;             // [H][W/2]: conj(G[ky(p)][q]) / (H W), p = column slot; q = 0 unused
    const float4 *ab;             // [H]: conj(G)/(HW) of columns kx = 0 (DC bin zeroed) and kx = W/2, by slot
    const uint16_t *col_partner;  // [H]: slot of -ky for the frequency at slot p
    const float *blob;            // staged GEMM operand tiles (stage-1 even/odd Dirichlet tiles, stage-2 cos/sin tiles),
                                  // tile t at blob + t * tile_floats
    const float *eblob;           // TC variants: stage-1 operand tiles in UMMA layout, tile (sb, ks) at eblob + (sb * KS + ks) * 128 * N1:
                                  //   four tables [N1][8] (Ee_hi, Ee_lo, Eo_hi, Eo_lo), K-major 8-row x 16-byte core matrices
    int N1;                       // TC variants: offsets per super-block rounded up to a multiple of 16 (MMA N)
    const uint32_t *sched;        // [ntiles_frame] blob tile index of the i-th tile a frame consumes
    uint32_t sched_head[8];       // sched[i % ntiles_frame], i < 8: the initial burst of the operand ring
    const float *nyqc;            // [ne_pad] cos(pi e / u): Nyquist-column weight of stage 2
    float2 *Sg;                   // global spectrum scratch (variants with S in L2), else null
    // fp64 tables of the two argmax polish steps (exactly reduced integer phase numerators, built at plan time)
    const double2 *tw64;          // [W] (cos, sin)(2 pi j / W)
    const double *Dpol;           // [M][H] Dirichlet weights of grid row m for the physical rows (y0+j) mod H of the
                                  //        sum/difference layout: j = 0, H/2: D_H(t-j); 0 < j < H/2: even part; H-j: odd part
    const double *DpolPlain;      // [M][H] the same weights for S holding the plain Q: D_H((m - c)/u - j) for row (y0+j) mod H
                                  //        (tensor-core variants, which form the sums / differences while staging)
    const double2 *Xpol;          // [M][W/2] (cos, sin)(2 pi q (n - c) / (u W))
    const double *nyq64;          // [M] cos(pi (n - c) / u)
    const double2 *XpolR;         // latency variants with pol_smem: Xpol regrouped by cluster rank, [CS][M][NC], else null

    // real-time session (cc_rt_*): mapped host memory; null outside a session
    const volatile unsigned long long *rt_cmd;  // [0] sequence number of the newest command (~0: quit), [1] frame pointer | seq & 15
    float *rt_res;                              // dx, dy, peak, sequence number (as bits): one 16-byte record
    int *rt_alive;                              // cleared by the kernel when it exits
    unsigned long long rt_timeout_ns;           // the kernel exits after this long without a command

    // running reference image (Eq. (9)); ri_Fs == null outside that mode.  The kernel then
    // reads Gt / ab / the reference mean through L2 (ld.cg) and rewrites them after every frame.
    float2 *ri_Fs;             // [H][W/2] forward spectrum of the current frame, column-slot order (scratch)
    float4 *ri_Fab;            // [H] (DC column, Nyquist column) of the current frame's spectrum, by slot
    double *ri_emean;          // mean of the reference image when it lives on the device (else null: Emean below)
    // offline iteration (Eq. (8)): per-cluster sums of the aligned frame spectra; acc_G == null
    // outside that mode.  ri_Fs / ri_Fab then hold one copy per cluster and the reference is not rewritten.
    float2 *acc_G;             // [clusters][H][W/2]
    float4 *acc_ab;            // [clusters][H]
    double *acc_mean;          // [clusters] sum of the frame means
    const int16_t *col_freq;   // [H] signed row frequency ky of column-FFT slot p (-H/2 at the Nyquist slot)
    double ri_a0;              // a0 = 1 - exp(-T/tau); b1 = 1 - a0

    int u, M, c;        // upsample factor, grid size ceil(1.5 u), centre floor(M/2)
    int nd;             // c + 1: number of |offsets| d (and e) evaluated per axis
    int DS;             // offsets d owned per CTA per super-block (T holds 2*DS rows)
    int nsb;            // number of super-blocks
    int DSBp;           // DS*CS rounded up to a multiple of TM1: U columns of a stage-1 super-block
    int nch1;           // stage-1 column chunks per super-block
    int KT1;            // stage-1 k-tiles (of BK1 rows j)
    int nrc2, nnc2;     // stage-2 row chunks / e-column chunks
    int ntiles_frame;   // tiles consumed per frame
    int tile_floats;    // floats per staging slot
    int c0;             // integer constant subtracted from every pixel before the FFT (CC-U)
    // CC-SN: pixels become (I + sn_eps)^2 - sn_c0 (evaluated in fp64, rounded once to fp32) and the
    // plan's spectrum is that of -1/(E + sn_eps); peak_sign = -1 turns the maximised -S back into the sum S
    int sn;             // 0: CC-U, 1: CC-SN
    double sn_eps, sn_c0;
    double peak_sign;
    int u_bytes;        // bytes of the raw/scratch/T union region
    int pol_smem;       // latency variants: 1 = the fp64 polish tables (Dpol, this CTA's Xpol columns, nyq64) are copied
                        // into shared memory once per launch (they fit), 0 = read from global memory
    double Emean;       // mean of the reference image (DC add-back for `peak`)
};

// Launcher interface of one compiled kernel variant.
struct CcVariant {
    int H, W, CS, NT, dtype;  // dtype: 0 = u8, 1 = u16
    int TM1, TN1, TM2, TN2;
    int R1, Cn1, R2, Cn2, KS2;  // thread grids of the two GEMM stages (rows x cols [x k-split])
    int KS1;                    // k-split of stage 1
    int BK1, G2;                // stage-1 k-rows per tile; stage-2 groups of 4 k-rows per tile
    int s_global;  // 1: spectrum array lives in global memory (L2), 0: shared memory / DSMEM
    int NSTG;
    int lat;       // 1: small-batch (latency) variant
    int tc1;       // 1: stage 1 on the tensor cores
    size_t (*fixed_smem)();                 // bytes that do not depend on M (S, tables, misc), before U/stg
    int (*raw_scratch_bytes)();             // raw ring + FFT scratch (lower bound of the U region)
    cudaError_t (*prepare)(int smem_bytes);  // sets func attributes
    cudaError_t (*max_clusters)(int smem_bytes, int *n);
    cudaError_t (*launch)(const CcParams &p, int n_clusters, int smem_bytes, cudaStream_t st);
};

// cc_api.cu -- C-ABI boundary (include/cc.h): plan creation (reference
// spectrum and upsampling tables, fp64 on the host, rounded once to fp32),
// variant selection, launches.  Product code: shares nothing with oracle/.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <stdlib.h>
#include <time.h>

#include <algorithm>
#include <complex>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/cc.h"
#include "../../include/cc_bench.h"
#include "cc_common.h"
#include "cc_refupdate.h"

// ------------------------------------------------------------------ variants
#define CCV(name, H, W, CS, PIX, NT, TM1, TN1, TM2, TN2, SG, BK1, G2, R2, KS2, NSTG, PFD, KS1, TC) CcVariant cc_variant_##name();
#include "cc_variant_list.h"
#undef CCV

typedef CcVariant (*cc_variant_fn)();
static const cc_variant_fn g_variant_fns[] = {
#define CCV(name, H, W, CS, PIX, NT, TM1, TN1, TM2, TN2, SG, BK1, G2, R2, KS2, NSTG, PFD, KS1, TC) &cc_variant_##name,
#include "cc_variant_list.h"
#undef CCV
};

static thread_local std::string g_err;
static cc_status fail(cc_status s, const std::string &msg)
{
    g_err = msg;
    return s;
}
static cc_status fail_cuda(cudaError_t e, const char *what)
{
    g_err = std::string(what) + ": " + cudaGetErrorString(e);
    return CC_ERR_CUDA;
}
#define CK(call)                                         \
    do {                                                 \
        cudaError_t e_ = (call);                         \
        if (e_ != cudaSuccess) return fail_cuda(e_, #call); \
    } while (0)

static const int SMEM_LIMIT = 232448;  // 227 KB per CTA on sm_100

// Per-variant launch geometry and operand tiles derived from the plan (M etc.).
struct VarPlan {
    CcVariant v;
    int smem_bytes = 0, max_clusters = 0;
    int DS = 0, nsb = 0, DSBp = 0, nch1 = 0, KT1 = 0, nrc2 = 0, nnc2 = 0, KT2 = 0;
    int ntiles_frame = 0, tile_floats = 0, u_bytes = 0;
    int pol_smem = 0;           // latency variants: fp64 polish tables resident in shared memory
    int N1 = 0, KS1T = 0;       // tensor-core stage 1: MMA N (offsets per super-block, multiple of 16), 8-row k-steps
    float *eblob = nullptr;     // tensor-core stage 1: operand tiles in UMMA layout
    float *blob = nullptr;      // device: staged operand tiles
    uint32_t *sched = nullptr;  // device: per-frame tile order
    uint32_t sched_head[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    float *nyqc = nullptr;      // device: cos(pi e / u)
    float2 *Sg = nullptr;       // global spectrum scratch (s_global variants)
    double2 *XpolR = nullptr;   // pol_smem: Xpol regrouped by cluster rank [CS][M][NC] (one bulk copy per CTA)
    float2 *Sg_alt = nullptr;   // second copy, used by cc_track_host's second stream (allocated on first use)
    size_t sg_bytes = 0;
    bool ready = false;
};

struct cc_plan {
    int H = 0, W = 0, u = 0, M = 0, c = 0, dtype = 0;
    int c0 = 0;
    int sn = 0;            // 0: CC-U, 1: CC-SN
    double sn_eps = 0.0, sn_c0 = 0.0;
    double Emean = 0.0;
    // device tables
    float2 *tw = nullptr, *Gt = nullptr;
    uint16_t *row_slot = nullptr, *col_partner = nullptr;
    float4 *ab = nullptr;
    double2 *tw64 = nullptr, *Xpol = nullptr;  // fp64 tables of the argmax polish steps
    double *Dpol = nullptr, *nyq64 = nullptr;
    double *DpolPlain = nullptr;  // Dirichlet rows for S holding the plain Q (tensor-core variants)
    // running reference image (Eq. (9)): scratch spectrum of the current frame, running mean, slot -> frequency table
    float2 *ri_Fs = nullptr;
    float4 *ri_Fab = nullptr;
    double *ri_emean = nullptr;
    int16_t *col_freq = nullptr;
    double ri_a0 = 0.0;
    int keep_clusters = 0;        // copies of ri_Fs / ri_Fab allocated
    // offline iteration (Eq. (8)): per-cluster accumulators of the aligned spectra
    float2 *acc_G = nullptr;
    float4 *acc_ab = nullptr;
    double *acc_mean = nullptr;
    int acc_clusters = 0;
    long long acc_count = 0;      // frames accumulated since the last reference update
    // CC-SN with a moving reference image (R19): fp64 state G = F[E], created on first use from the caller's image
    CcSnState *sn_state = nullptr;
    std::vector<float> sn_ref;    // the caller's reference image (CC-SN plans only)
    size_t table_bytes = 0;
    VarPlan thr, lat;  // throughput variant, small-batch (latency) variant
    bool has_lat = false;
    // cc_track_host resources
    cudaStream_t hs[2] = {nullptr, nullptr};
    cudaEvent_t hev[2] = {nullptr, nullptr};
    void *dframes[2] = {nullptr, nullptr};
    float *dres = nullptr;  // [3][cap]
    int chunk_cap = 0, res_cap = 0;
    int host_chunk = 0;     // frames per cc_track_host chunk (0: about 64 MB of frames)
    // single-frame calls: the one-cluster launch of the small-batch variant as a pre-instantiated graph whose kernel
    // parameters are patched per call (launch + synchronise costs 7.3 us that way against 11.3 us for a plain launch)
    cudaGraph_t g1 = nullptr;
    cudaGraphExec_t ge1 = nullptr;
    cudaGraphNode_t gn1 = nullptr;
    cudaKernelNodeParams kp1{};
    const VarPlan *g1_vp = nullptr;
    mutable std::mutex g1_mu;
};

// ------------------------------------------------------------------ host fp64 FFT (plan time only)
static void fft1d(std::vector<std::complex<double>> &a, int n, int stride, size_t off, bool inv,
                  const std::vector<std::complex<double>> &w)  // w[j] = exp(-2 pi i j / n)
{
    // iterative radix-2, in place on a[off + i*stride]
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) std::swap(a[off + (size_t)i * stride], a[off + (size_t)j * stride]);
    }
    for (int len = 2; len <= n; len <<= 1) {
        const int step = n / len;
        for (int i = 0; i < n; i += len)
            for (int k = 0; k < len / 2; ++k) {
                std::complex<double> t = w[(size_t)k * step];
                if (inv) t = std::conj(t);
                const std::complex<double> x = a[off + (size_t)(i + k) * stride];
                const std::complex<double> y = a[off + (size_t)(i + k + len / 2) * stride] * t;
                a[off + (size_t)(i + k) * stride] = x + y;
                a[off + (size_t)(i + k + len / 2) * stride] = x - y;
            }
    }
}

static std::vector<std::complex<double>> unit_roots(int n)
{
    std::vector<std::complex<double>> w(n);
    for (int j = 0; j < n; ++j) {
        // exact octant values keep the table symmetric
        const double a = -2.0 * M_PI * (double)j / (double)n;
        w[j] = std::complex<double>(cos(a), sin(a));
    }
    return w;
}

static bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
static int round_up(int v, int m) { return (v + m - 1) / m * m; }

template <class T>
static cudaError_t upload(T **dptr, const std::vector<T> &h, size_t *acc)
{
    cudaError_t e = cudaMalloc((void **)dptr, h.size() * sizeof(T));
    if (e != cudaSuccess) return e;
    *acc += h.size() * sizeof(T);
    return cudaMemcpy(*dptr, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
}

// geometry of one variant for this plan; returns false if it cannot fit
static bool plan_variant(VarPlan &vp, int M, int W, int H)
{
    const CcVariant &v = vp.v;
    const int NC = W / 2 / v.CS;
    const int nd = M / 2 + 1;  // offsets d = 0..c (and e = 0..c)
    const int MC1 = v.R1 * v.TM1;
    const int T1F = v.tc1 ? 0 : v.BK1 * MC1, T2F = v.G2 * v.Cn2 * (16 + 4 * (v.TN2 - 4));
    vp.tile_floats = std::max(T1F, T2F);
    const int NSL = std::max(1, v.NT / NC);
    const int polish = 3 * H * 8 + 3 * NSL * NC * 16 + 3 * NC * 16 + 9 * NC * 8;
    const int lower = std::max(v.raw_scratch_bytes(), polish);
    const int red_bytes = std::max((v.KS2 - 1) * v.R2 * v.Cn2 * 2 * v.TM2 * v.TN2, (v.KS1 - 1) * v.R1 * v.Cn1 * v.TM1 * v.TN1) * 4;
    const long avail = (long)SMEM_LIMIT - (long)v.fixed_smem() - 32;
    if (avail < lower) return false;
    const int LDT = W + 4;
    int ds_cap = (int)((avail - red_bytes) / ((long)LDT * 4)) / 2;
    if (v.tc1) ds_cap = std::min(ds_cap, 128 / v.CS);  // four accumulator blocks of N1 <= 128 columns in the 512 columns of tensor memory
    if (ds_cap < 1) return false;
    int nsb = 1, DS;
    for (;; ++nsb) {
        const int per_sb = (nd + nsb - 1) / nsb;
        DS = (per_sb + v.CS - 1) / v.CS;
        if (DS <= ds_cap) break;
    }
    vp.DS = DS;
    vp.nsb = (nd + DS * v.CS - 1) / (DS * v.CS);
    vp.DSBp = round_up(DS * v.CS, v.TM1);
    vp.nch1 = (2 * vp.DSBp + MC1 - 1) / MC1;
    vp.KT1 = (H / 2 + 1 + v.BK1 - 1) / v.BK1;
    vp.nrc2 = (2 * DS + v.R2 * v.TM2 - 1) / (v.R2 * v.TM2);
    vp.nnc2 = (nd + v.Cn2 * v.TN2 - 1) / (v.Cn2 * v.TN2);
    vp.KT2 = W / (4 * v.G2);
    vp.ntiles_frame = vp.nsb * ((v.tc1 ? 0 : vp.nch1 * vp.KT1) + vp.nrc2 * vp.nnc2 * vp.KT2);
    vp.u_bytes = round_up(std::max(lower, 2 * DS * LDT * 4 + red_bytes), 16);
    if (v.tc1) {  // staging double buffer (2 x 4 x 4 KB) + 4 operand-ring slots of 4 tables [N1][8] floats, inside the U region
        vp.N1 = round_up(DS * v.CS, 16);
        vp.KS1T = (H / 2 + 1 + 7) / 8;
        vp.u_bytes = std::max(vp.u_bytes, 32768 + 4 * 4 * vp.N1 * 32);
    }
    vp.smem_bytes = (int)v.fixed_smem() + vp.u_bytes + 32;
    if (vp.smem_bytes > SMEM_LIMIT) return false;
    // latency variants: keep the fp64 polish tables in shared memory when they fit (two L2 round trips less per frame)
    const long pol_bytes = (long)M * H * 8 + (long)M * NC * 16 + (long)((M + 1) & ~1) * 8;
    vp.pol_smem = (v.lat && M > 2 && vp.smem_bytes + pol_bytes <= SMEM_LIMIT) ? 1 : 0;  // M == 2: u == 1, no tables
    if (vp.pol_smem) vp.smem_bytes += (int)pol_bytes;
    return true;
}

// D_H(t) = sin(pi t) cot(pi t / H) / H at t = tnum / u (periodic-sinc weight, Nyquist bin split half/half)
static double dirichlet_host(long long tnum, int u, int H)
{
    const long long den = (long long)u * H;
    const long long r = ((tnum % den) + den) % den;
    if (r == 0) return 1.0;
    const long long r2 = ((tnum % (2LL * u)) + 2LL * u) % (2LL * u);
    if (r2 == 0 || r2 == u) return 0.0;
    const double s1 = sin(M_PI * (double)r2 / (double)u);
    const double x = M_PI * (double)r / (double)den;
    return s1 * cos(x) / ((double)H * sin(x));
}

// ---- long-double versions for the fp64 polish tables
static const long double PI_L = 3.14159265358979323846264338327950288L;
static long double sinpi_frac_l(long long num, long long den)  // sin(pi num / den), phase reduced exactly
{
    long long r = num % (2 * den);
    if (r < 0) r += 2 * den;
    if (r == 0 || r == den) return 0.0L;
    return sinl(PI_L * (long double)r / (long double)den);
}
static long double dirichlet_l(long long tnum, int u, int H)
{
    const long long den = (long long)u * H;
    const long long r = ((tnum % den) + den) % den;
    if (r == 0) return 1.0L;
    const long double s1 = sinpi_frac_l(tnum, u);
    const long double x = PI_L * (long double)r / (long double)den;  // in (0, pi)
    return s1 * cosl(x) / ((long double)H * sinl(x));
}
// Even / odd parts of the Dirichlet weight about row offset j (0 < j < H/2), t = tnum / u, |t| < 1:
//   we = (D_H(t-j) + D_H(t+j)) / 2 = (-1)^j sin(pi t) sin(2x) / (2 H sin(x-y) sin(x+y)),
//   wo = (D_H(t-j) - D_H(t+j)) / 2 = (-1)^j sin(pi t) sin(2y) / (2 H sin(x-y) sin(x+y)),   x = pi t / H, y = pi j / H
static void dirichlet_pair_l(long long tnum, int j, int u, int H, double *we, double *wo)
{
    const long long den = (long long)u * H;
    const long double s = sinpi_frac_l(tnum, u);
    const long double sa = sinpi_frac_l(tnum - (long long)j * u, den), sb = sinpi_frac_l(tnum + (long long)j * u, den);
    const long double pref = ((j & 1) ? -s : s) / (2.0L * (long double)H * sa * sb);
    *we = (double)(pref * sinpi_frac_l(2 * tnum, den));
    *wo = (double)(pref * sinpi_frac_l(2LL * j, H));
}

// operand tiles of one variant: stage-1 even/odd Dirichlet tiles, stage-2 cos/sin tiles, the tile schedule
static cudaError_t build_tiles(VarPlan &vp, int H, int W, int u, int M, size_t *acc)
{
    const CcVariant &v = vp.v;
    const int c = M / 2, nd = c + 1;
    const int TF = vp.tile_floats, MC1 = v.R1 * v.TM1, DSB = vp.DS * v.CS;
    const int n1 = v.tc1 ? 0 : vp.nsb * vp.nch1 * vp.KT1, n2 = vp.nnc2 * vp.KT2;
    std::vector<float> blob((size_t)(n1 + n2) * TF, 0.f);
    // position inside a staged k-row -> logical [U|V] column of the chunk (cc_tm1_* chunk layout)
    std::vector<int> col_of_pos(MC1);
    for (int tm1 = 0; tm1 < v.R1; ++tm1)
        for (int ci = 0; ci < cc_tm1_nchunks(v.TM1); ++ci) {
            const int w = cc_tm1_width(v.TM1, ci), st = cc_tm1_start(v.TM1, ci);
            for (int i = 0; i < w; ++i) col_of_pos[v.R1 * st + tm1 * w + i] = tm1 * v.TM1 + st + i;
        }
    for (int sb = 0; sb < vp.nsb && !v.tc1; ++sb)
        for (int ch = 0; ch < vp.nch1; ++ch)
            for (int kt = 0; kt < vp.KT1; ++kt) {
                float *tile = blob.data() + (size_t)((sb * vp.nch1 + ch) * vp.KT1 + kt) * TF;
                for (int kk = 0; kk < v.BK1; ++kk) {
                    const int j = kt * v.BK1 + kk;
                    if (j > H / 2) continue;
                    for (int pos = 0; pos < MC1; ++pos) {
                        const int gc = ch * MC1 + col_of_pos[pos];
                        const bool isV = gc >= vp.DSBp;
                        const int dsb = gc - (isV ? vp.DSBp : 0);
                        const int d = sb * DSB + dsb;
                        if (dsb >= DSB || d >= nd) continue;
                        double val;
                        if (j == 0 || j == H / 2) {
                            val = isV ? 0.0 : dirichlet_host((long long)d - (long long)j * u, u, H);
                        } else {
                            const double dm = dirichlet_host((long long)d - (long long)j * u, u, H);
                            const double dp = dirichlet_host((long long)d + (long long)j * u, u, H);
                            val = isV ? 0.5 * (dm - dp) : 0.5 * (dm + dp);
                        }
                        tile[kk * MC1 + pos] = (float)val;
                    }
                }
            }
    const int X2 = v.TN2 - 4, GF2 = v.Cn2 * (16 + 4 * X2), NCOL2 = v.Cn2 * v.TN2;
    const long long denx = (long long)u * W;
    auto val2 = [&](int k, int e) -> float {
        if (e >= nd) return 0.f;
        if (k == 0) return 1.f;
        if (k == 1) return 0.f;  // Nyquist column: added in the stage-2 epilogue with nyqc
        const int q = k / 2;
        const long long num = ((long long)q * e) % denx;
        const double th = 2.0 * M_PI * (double)num / (double)denx;
        return (float)((k & 1) ? 2.0 * sin(th) : 2.0 * cos(th));
    };
    for (int nc2 = 0; nc2 < vp.nnc2; ++nc2)
        for (int kt = 0; kt < vp.KT2; ++kt) {
            float *tile = blob.data() + (size_t)(n1 + nc2 * vp.KT2 + kt) * TF;
            for (int g = 0; g < v.G2; ++g)
                for (int kk = 0; kk < 4; ++kk) {
                    const int k = (kt * v.G2 + g) * 4 + kk;
                    for (int col = 0; col < v.Cn2 * 4; ++col)
                        tile[g * GF2 + kk * v.Cn2 * 4 + col] = val2(k, nc2 * NCOL2 + col);
                    if (X2)
                        for (int tn = 0; tn < v.Cn2; ++tn)
                            tile[g * GF2 + 16 * v.Cn2 + tn * 4 + kk] = val2(k, nc2 * NCOL2 + 4 * v.Cn2 + tn);
                }
        }
    // tensor-core stage 1: per (super-block, 8-row k-step) four tables [N1][8] -- even weights hi / lo, odd weights hi / lo
    // (x = hi + lo: hi = the float with its low 13 mantissa bits cleared, lo = the rest of the float64 value, likewise
    // truncated to TF32) -- in the K-major core-matrix layout of the UMMA descriptors: element (d, k) of a table at float
    // (d / 8) * 64 + (k / 4) * 32 + (d % 8) * 4 + (k % 4)
    std::vector<float> eblob;
    if (v.tc1) {
        const int N1 = vp.N1, KS = vp.KS1T;
        auto hi13 = [](float x) {
            uint32_t b;
            memcpy(&b, &x, 4);
            b &= 0xffffe000u;
            memcpy(&x, &b, 4);
            return x;
        };
        eblob.assign((size_t)vp.nsb * KS * 4 * N1 * 8, 0.f);
        for (int sb = 0; sb < vp.nsb; ++sb)
            for (int ks = 0; ks < KS; ++ks) {
                float *tile = eblob.data() + ((size_t)sb * KS + ks) * 4 * N1 * 8;
                for (int dsb = 0; dsb < N1; ++dsb)
                    for (int k = 0; k < 8; ++k) {
                        const int j = ks * 8 + k, d = sb * DSB + dsb;
                        if (j > H / 2 || dsb >= DSB || d >= nd) continue;
                        double we, wo;
                        if (j == 0 || j == H / 2) {
                            we = dirichlet_host((long long)d - (long long)j * u, u, H), wo = 0.0;
                        } else {
                            const double dm = dirichlet_host((long long)d - (long long)j * u, u, H);
                            const double dp = dirichlet_host((long long)d + (long long)j * u, u, H);
                            we = 0.5 * (dm + dp), wo = 0.5 * (dm - dp);
                        }
                        const size_t off = (size_t)(dsb / 8) * 64 + (k / 4) * 32 + (dsb % 8) * 4 + (k % 4);
                        const float eh = hi13((float)we), oh = hi13((float)wo);
                        tile[off] = eh, tile[(size_t)N1 * 8 + off] = hi13((float)(we - (double)eh));
                        tile[(size_t)2 * N1 * 8 + off] = oh, tile[(size_t)3 * N1 * 8 + off] = hi13((float)(wo - (double)oh));
                    }
            }
    }
    std::vector<uint32_t> sched;
    for (int sb = 0; sb < vp.nsb; ++sb) {
        for (int ch = 0; ch < vp.nch1 && !v.tc1; ++ch)
            for (int kt = 0; kt < vp.KT1; ++kt) sched.push_back((uint32_t)((sb * vp.nch1 + ch) * vp.KT1 + kt));
        for (int rc = 0; rc < vp.nrc2; ++rc)
            for (int nc2 = 0; nc2 < vp.nnc2; ++nc2)
                for (int kt = 0; kt < vp.KT2; ++kt) sched.push_back((uint32_t)(n1 + nc2 * vp.KT2 + kt));
    }
    std::vector<float> nyq((size_t)vp.nnc2 * NCOL2, 0.f);
    for (int e = 0; e < nd; ++e) {
        const long long r2 = (long long)e % (2LL * u);
        nyq[e] = (float)cos(M_PI * (double)r2 / (double)u);
    }
    for (int i = 0; i < 8; ++i) vp.sched_head[i] = sched.empty() ? 0u : sched[(size_t)i % sched.size()];
    cudaError_t e = upload(&vp.blob, blob, acc);
    if (e == cudaSuccess && v.tc1) e = upload(&vp.eblob, eblob, acc);
    if (e == cudaSuccess) e = upload(&vp.sched, sched, acc);
    if (e == cudaSuccess) e = upload(&vp.nyqc, nyq, acc);
    return e;
}

static cc_status check_device()
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(CC_ERR_ARCH, std::string("no CUDA device: ") + cudaGetErrorString(e));
    int major = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return fail_cuda(e, "cudaDeviceGetAttribute");
    if (major != 10) return fail(CC_ERR_ARCH, "device is not compute capability 10.x (sm_100a kernels only; no fallback)");
    return CC_OK;
}

static void fill_params(const cc_plan *pl, const VarPlan &vp, CcParams &p);

// One-cluster launch of the single-frame variant, captured once; cc_track(batch = 1) patches its parameters.
static cudaError_t build_single_frame_graph(cc_plan *pl)
{
    const VarPlan *vp = pl->has_lat ? &pl->lat : &pl->thr;
    cudaStream_t cs = nullptr;
    cudaError_t e = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking);
    if (e != cudaSuccess) return e;
    CcParams p{};
    fill_params(pl, *vp, p);
    p.batch = 1;
    e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
        const cudaError_t le = vp->v.launch(p, 1, vp->smem_bytes, cs);
        e = cudaStreamEndCapture(cs, &pl->g1);
        if (e == cudaSuccess) e = le;
    }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&pl->ge1, pl->g1, 0);
    size_t n = 1;
    if (e == cudaSuccess) e = cudaGraphGetNodes(pl->g1, &pl->gn1, &n);
    if (e == cudaSuccess && n != 1) e = cudaErrorUnknown;
    if (e == cudaSuccess) e = cudaGraphKernelNodeGetParams(pl->gn1, &pl->kp1);
    if (e == cudaSuccess) pl->g1_vp = vp;
    cudaStreamDestroy(cs);
    return e;
}

extern "C" cc_status cc_plan_destroy(cc_plan *plan)
{
    if (!plan) return CC_OK;
    cudaFree(plan->tw), cudaFree(plan->Gt), cudaFree(plan->row_slot), cudaFree(plan->col_partner);
    cudaFree(plan->ab);
    cudaFree(plan->tw64), cudaFree(plan->Xpol), cudaFree(plan->Dpol), cudaFree(plan->nyq64), cudaFree(plan->DpolPlain);
    cudaFree(plan->ri_Fs), cudaFree(plan->ri_Fab), cudaFree(plan->ri_emean), cudaFree(plan->col_freq);
    cudaFree(plan->acc_G), cudaFree(plan->acc_ab), cudaFree(plan->acc_mean);
    cc_sn_state_destroy(plan->sn_state);
    for (VarPlan *vp : {&plan->thr, &plan->lat})
        cudaFree(vp->Sg), cudaFree(vp->Sg_alt), cudaFree(vp->blob), cudaFree(vp->sched), cudaFree(vp->nyqc), cudaFree(vp->XpolR), cudaFree(vp->eblob);
    for (int i = 0; i < 2; ++i) {
        if (plan->hs[i]) cudaStreamDestroy(plan->hs[i]);
        if (plan->hev[i]) cudaEventDestroy(plan->hev[i]);
        cudaFree(plan->dframes[i]);
    }
    cudaFree(plan->dres);
    if (plan->ge1) cudaGraphExecDestroy(plan->ge1);
    if (plan->g1) cudaGraphDestroy(plan->g1);
    delete plan;
    return CC_OK;
}

extern "C" cc_status cc_plan_create(cc_plan **out, int H, int W, cc_dtype dtype, int upsample, const float *reference)
{
    return cc_plan_create_weighted(out, H, W, dtype, upsample, reference, CC_METHOD_U, 0.f);
}

extern "C" cc_status cc_plan_create_weighted(cc_plan **out, int H, int W, cc_dtype dtype, int upsample, const float *reference,
                                             cc_method method, float epsilon)
{
    if (method != CC_METHOD_U && method != CC_METHOD_SN) return fail(CC_ERR_INVALID_ARG, "cc_plan_create_weighted: bad method");
    if (method == CC_METHOD_SN && !(epsilon >= 0.f)) return fail(CC_ERR_INVALID_ARG, "cc_plan_create_weighted: epsilon must be >= 0");
    if (!out || !reference || H <= 0 || W <= 0 || upsample < 1 || (dtype != CC_U8 && dtype != CC_U16))
        return fail(CC_ERR_INVALID_ARG, "cc_plan_create: bad argument");
    if (upsample > 4096) return fail(CC_ERR_UNSUPPORTED, "upsample factor above 4096");
    if (!is_pow2(H) || !is_pow2(W) || cc_radix_col(H, 0) == 0 || cc_radix_row(W, 0) == 0)
        return fail(CC_ERR_UNSUPPORTED, "frame sides must be powers of two in 64..1024");
    cc_status st = check_device();
    if (st != CC_OK) return st;

    cc_plan *pl = new (std::nothrow) cc_plan();
    if (!pl) return fail(CC_ERR_NOMEM, "host allocation failed");
    pl->H = H, pl->W = W, pl->u = upsample, pl->dtype = (int)dtype;
    pl->M = (3 * upsample + 1) / 2;  // ceil(1.5 u)
    pl->c = pl->M / 2;
    const int M = pl->M, c = pl->c, u = upsample;
    (void)c;

    // ---- variants: smallest cluster = throughput variant, largest = small-batch (latency) variant
    {
        std::vector<VarPlan> fits;
        for (cc_variant_fn fn : g_variant_fns) {
            VarPlan vp;
            vp.v = fn();
            if (vp.v.H != H || vp.v.W != W || vp.v.dtype != (int)dtype) continue;
            if (plan_variant(vp, M, W, H)) fits.push_back(vp);
        }
        if (fits.empty()) {
            delete pl;
            return fail(CC_ERR_UNSUPPORTED, "no kernel variant for this frame shape / pixel type");
        }
        std::sort(fits.begin(), fits.end(), [](const VarPlan &a, const VarPlan &b) { return a.v.CS < b.v.CS; });
        pl->thr = fits.front();
        if (fits.back().v.CS != fits.front().v.CS) pl->lat = fits.back(), pl->has_lat = true;
    }

    // ---- reference image to the host
    std::vector<float> ref((size_t)H * W);
    {
        cudaError_t e = cudaMemcpy(ref.data(), reference, ref.size() * sizeof(float), cudaMemcpyDefault);
        if (e != cudaSuccess) {
            delete pl;
            return fail_cuda(e, "copy of the reference image");
        }
    }

    // ---- G = DFT2(E) in fp64 (row pass, column pass)
    std::vector<std::complex<double>> G((size_t)H * W);
    if (method == CC_METHOD_SN) {
        // CC-SN, Eqs. (5)-(7): correlate I'^2 with 1/E', E' = E + eps; chi^2 is minimised, so the kernel maximises the
        // correlation with -1/E' (R15, R16).  sn_c0 = the mean of E'^2 rounded to an integer: the constant
        // taken off every transformed pixel (an exact no-op for the argmax; restored in `peak`).
        double m2 = 0.0;
        for (size_t i = 0; i < G.size(); ++i) {
            const double ep = (double)ref[i] + (double)epsilon;
            if (!(ep > 0.0)) {
                delete pl;
                return fail(CC_ERR_INVALID_ARG, "CC-SN needs reference + epsilon > 0 in every pixel");
            }
            G[i] = std::complex<double>(-1.0 / ep, 0.0);
            m2 += ep * ep;
        }
        pl->sn = 1, pl->sn_eps = (double)epsilon, pl->sn_c0 = nearbyint(m2 / (double)G.size());
        pl->sn_ref = ref;
    } else {
        for (size_t i = 0; i < G.size(); ++i) G[i] = std::complex<double>((double)ref[i], 0.0);
    }
    {
        const auto wW = unit_roots(W), wH = unit_roots(H);
        for (int y = 0; y < H; ++y) fft1d(G, W, 1, (size_t)y * W, false, wW);
        for (int x = 0; x < W; ++x) fft1d(G, H, W, (size_t)x, false, wH);
    }
    const double HW = (double)H * (double)W;
    pl->Emean = G[0].real() / HW;
    pl->c0 = (int)std::min(65535.0, std::max(0.0, nearbyint(pl->Emean)));

    // ---- tables
    const int NTW = std::max(H, W);
    std::vector<float2> tw(NTW);
    for (int j = 0; j < NTW; ++j) {
        const double a = 2.0 * M_PI * (double)j / (double)NTW;
        tw[j] = make_float2((float)cos(a), (float)(-sin(a)));
    }
    std::vector<uint16_t> row_slot(W), col_slot(H), col_partner(H);
    for (int p = 0; p < W; ++p) row_slot[cc_freq_of_slot(W, p, true)] = (uint16_t)p;
    for (int p = 0; p < H; ++p) col_slot[cc_freq_of_slot(H, p, false)] = (uint16_t)p;
    for (int p = 0; p < H; ++p) col_partner[p] = col_slot[(H - cc_freq_of_slot(H, p, false)) % H];

    const int Wh = W / 2;
    std::vector<float2> Gt((size_t)H * Wh);
    std::vector<float4> ab(H);
    for (int p = 0; p < H; ++p) {
        const int ky = cc_freq_of_slot(H, p, false);
        for (int q = 1; q < Wh; ++q) {
            const std::complex<double> g = std::conj(G[(size_t)ky * W + q]) / HW;
            Gt[(size_t)p * Wh + q] = make_float2((float)g.real(), (float)g.imag());
        }
        Gt[(size_t)p * Wh] = make_float2(0.f, 0.f);
        // packed column: DC bin of the reference zeroed (shift-independent constant; R10)
        std::complex<double> g0 = (ky == 0) ? std::complex<double>(0.0, 0.0) : std::conj(G[(size_t)ky * W]) / HW;
        std::complex<double> gn = std::conj(G[(size_t)ky * W + Wh]) / HW;
        ab[p] = make_float4((float)g0.real(), (float)g0.imag(), (float)gn.real(), (float)gn.imag());
    }

    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = upload(&pl->tw, tw, &pl->table_bytes);
    if (e == cudaSuccess) e = upload(&pl->row_slot, row_slot, &pl->table_bytes);
    if (e == cudaSuccess) e = upload(&pl->col_partner, col_partner, &pl->table_bytes);
    if (e == cudaSuccess) e = upload(&pl->Gt, Gt, &pl->table_bytes);
    if (e == cudaSuccess) e = upload(&pl->ab, ab, &pl->table_bytes);
    // ---- fp64 tables of the polish steps (R9): every phase from an exactly reduced integer numerator
    {
        std::vector<double2> tw64(W);
        for (int j = 0; j < W; ++j) tw64[j] = make_double2((double)cosl(2.0L * PI_L * j / W), (double)sinl(2.0L * PI_L * j / W));
        if (e == cudaSuccess) e = upload(&pl->tw64, tw64, &pl->table_bytes);
    }
    if (u > 1) {
        std::vector<double> Dpol((size_t)M * H), nyq64((size_t)(M + 1) & ~(size_t)1, 0.0);  // even length: copied in 16-byte units
        std::vector<double2> Xpol((size_t)M * Wh);
        const long long denx = (long long)u * W;
        for (int m = 0; m < M; ++m) {
            const long long tnum = m - c;  // t = tnum / u, |t| < 1
            double *row = Dpol.data() + (size_t)m * H;
            row[0] = (double)dirichlet_l(tnum, u, H);
            row[H / 2] = (double)dirichlet_l(tnum - (long long)(H / 2) * u, u, H);
            for (int j = 1; j < H / 2; ++j) dirichlet_pair_l(tnum, j, u, H, &row[j], &row[H - j]);
            nyq64[m] = (double)cosl(PI_L * (long double)(((tnum % (2LL * u)) + 2LL * u) % (2LL * u)) / (long double)u);
            for (int q = 0; q < Wh; ++q) {
                const long long num = (((long long)q * tnum) % denx + denx) % denx;
                const long double th = 2.0L * PI_L * (long double)num / (long double)denx;
                Xpol[(size_t)m * Wh + q] = make_double2((double)cosl(th), (double)sinl(th));
            }
        }
        if (e == cudaSuccess) e = upload(&pl->Dpol, Dpol, &pl->table_bytes);
        if (pl->thr.v.tc1 || (pl->has_lat && pl->lat.v.tc1)) {
            std::vector<double> Dplain((size_t)M * H);
            for (int m = 0; m < M; ++m)
                for (int j = 0; j < H; ++j) Dplain[(size_t)m * H + j] = (double)dirichlet_l((long long)(m - c) - (long long)j * u, u, H);
            if (e == cudaSuccess) e = upload(&pl->DpolPlain, Dplain, &pl->table_bytes);
        }
        if (e == cudaSuccess) e = upload(&pl->Xpol, Xpol, &pl->table_bytes);
        if (e == cudaSuccess) e = upload(&pl->nyq64, nyq64, &pl->table_bytes);
        if (e == cudaSuccess) e = build_tiles(pl->thr, H, W, u, M, &pl->table_bytes);
        if (e == cudaSuccess && pl->has_lat) e = build_tiles(pl->lat, H, W, u, M, &pl->table_bytes);
        for (VarPlan *vp : {&pl->thr, &pl->lat}) {
            if (e != cudaSuccess || !vp->pol_smem) continue;
            const int CS = vp->v.CS, NC = Wh / CS;
            std::vector<double2> xr((size_t)M * Wh);
            for (int r = 0; r < CS; ++r)
                for (int m = 0; m < M; ++m)
                    for (int ql = 0; ql < NC; ++ql) xr[((size_t)r * M + m) * NC + ql] = Xpol[(size_t)m * Wh + r * NC + ql];
            e = upload(&vp->XpolR, xr, &pl->table_bytes);
        }
    }

    // ---- kernel attributes, occupancy, scratch
    VarPlan *vps[2] = {&pl->thr, pl->has_lat ? &pl->lat : nullptr};
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
        VarPlan *vp = vps[i];
        if (!vp) continue;
        e = vp->v.prepare(vp->smem_bytes);
        if (e == cudaSuccess) e = vp->v.max_clusters(vp->smem_bytes, &vp->max_clusters);
        if (e == cudaSuccess && vp->max_clusters < 1) {
            cc_plan_destroy(pl);
            return fail(CC_ERR_UNSUPPORTED, "kernel variant cannot be made resident (cluster occupancy 0)");
        }
        if (e == cudaSuccess && vp->v.s_global) {
            vp->sg_bytes = (size_t)vp->max_clusters * vp->v.CS * ((size_t)H * (W / 2 / vp->v.CS)) * sizeof(float2);
            e = cudaMalloc((void **)&vp->Sg, vp->sg_bytes);
        }
        vp->ready = (e == cudaSuccess);
    }
    if (e == cudaSuccess) e = build_single_frame_graph(pl);
    if (e != cudaSuccess) {
        cc_status s = (e == cudaErrorMemoryAllocation) ? fail(CC_ERR_NOMEM, "device allocation failed") : fail_cuda(e, "plan setup");
        cc_plan_destroy(pl);
        return s;
    }
    *out = pl;
    return CC_OK;
}

static void fill_params(const cc_plan *pl, const VarPlan &vp, CcParams &p)
{
    p.tw = pl->tw, p.row_slot = pl->row_slot, p.Gt = pl->Gt, p.ab = pl->ab, p.col_partner = pl->col_partner;
    p.blob = vp.blob, p.sched = vp.sched, p.nyqc = vp.nyqc, p.Sg = vp.Sg, p.eblob = vp.eblob, p.N1 = vp.N1;
    for (int i = 0; i < 8; ++i) p.sched_head[i] = vp.sched_head[i];
    p.tw64 = pl->tw64, p.Dpol = pl->Dpol, p.DpolPlain = pl->DpolPlain, p.Xpol = pl->Xpol, p.nyq64 = pl->nyq64, p.XpolR = vp.XpolR;
    p.u = pl->u, p.M = pl->M, p.c = pl->c, p.nd = pl->c + 1;
    p.DS = vp.DS, p.nsb = vp.nsb, p.DSBp = vp.DSBp, p.nch1 = vp.nch1, p.KT1 = vp.KT1, p.nrc2 = vp.nrc2, p.nnc2 = vp.nnc2;
    p.ntiles_frame = pl->u > 1 ? vp.ntiles_frame : 0, p.tile_floats = vp.tile_floats;
    p.c0 = pl->c0, p.u_bytes = vp.u_bytes, p.pol_smem = vp.pol_smem, p.Emean = pl->Emean;
    p.ri_emean = pl->ri_emean;  // null while the reference mean is the host constant Emean
    if (pl->ri_a0 > 0.0 && !pl->sn) {  // CC-U: Eq. (9) inside the fused kernel; CC-SN: separate fp64 kernels (cc_refupdate.cu)
        p.ri_Fs = pl->ri_Fs, p.ri_Fab = pl->ri_Fab, p.col_freq = pl->col_freq, p.ri_a0 = pl->ri_a0;
    }
    p.sn = pl->sn, p.sn_eps = pl->sn_eps, p.sn_c0 = pl->sn_c0, p.peak_sign = pl->sn ? -1.0 : 1.0;
}

static cc_status track_impl(const cc_plan *plan, const void *frames, int batch, float *dx, float *dy, float *peak,
                            int *iy, int *ix, unsigned long long *phase_clk, void *stream, int sg_slot = 0)
{
    if (!plan || batch < 0) return fail(CC_ERR_INVALID_ARG, "cc_track: bad plan or batch");
    if (batch == 0) return CC_OK;
    if (!frames || !dx || !dy) return fail(CC_ERR_INVALID_ARG, "cc_track: null pointer");
    if (((uintptr_t)frames & 15u) != 0) return fail(CC_ERR_INVALID_ARG, "cc_track: frames must be 16-byte aligned");
    const VarPlan *vp = &plan->thr;
    const bool ri = plan->ri_a0 > 0.0;  // running reference image: frames strictly in order, one cluster
    if (plan->has_lat && (ri || (batch <= plan->lat.max_clusters && batch * plan->lat.v.CS <= plan->thr.max_clusters * plan->thr.v.CS)))
        vp = &plan->lat;
    CcParams p{};
    fill_params(plan, *vp, p);
    p.frames = frames, p.batch = batch, p.dx = dx, p.dy = dy, p.peak = peak, p.iy = iy, p.ix = ix, p.phase_clk = phase_clk;
    if (sg_slot == 1 && vp->Sg_alt) p.Sg = vp->Sg_alt;  // cc_track_host's second stream: its own spectrum scratch
    if (ri && plan->sn) {
        // CC-SN with the running reference image (R19): one frame per launch against the current weight
        // spectrum, then the fp64 update kernels rewrite it from the new state (Eq. (9) on the raw images)
        const size_t fbytes = (size_t)plan->H * plan->W * (plan->dtype == CC_U8 ? 1 : 2);
        const CcSnTables t{plan->Gt, plan->ab, plan->ri_emean, plan->col_freq};
        for (int i = 0; i < batch; ++i) {
            const void *fi = (const unsigned char *)frames + (size_t)i * fbytes;
            p.frames = fi, p.batch = 1, p.dx = dx + i, p.dy = dy + i, p.peak = peak ? peak + i : nullptr;
            p.iy = iy ? iy + i : nullptr, p.ix = ix ? ix + i : nullptr;
            p.phase_clk = phase_clk ? phase_clk + (size_t)i * CC_NPHASE : nullptr;
            cudaError_t e = vp->v.launch(p, 1, vp->smem_bytes, (cudaStream_t)stream);
            if (e == cudaSuccess) e = cc_sn_update_eq9(plan->sn_state, fi, dy + i, dx + i, plan->ri_a0, t, (cudaStream_t)stream);
            if (e != cudaSuccess) return fail_cuda(e, "CC-SN frame + reference update");
        }
        return CC_OK;
    }
    const int ncl = ri ? 1 : std::min(batch, vp->max_clusters);
    if (ncl == 1 && vp == plan->g1_vp && plan->ge1 && sg_slot == 0) {  // single frame: the pre-instantiated graph
        std::lock_guard<std::mutex> lk(plan->g1_mu);
        cudaKernelNodeParams kp = plan->kp1;
        void *args[1] = {&p};
        kp.kernelParams = args;
        kp.extra = nullptr;
        cudaError_t e = cudaGraphExecKernelNodeSetParams(plan->ge1, plan->gn1, &kp);
        if (e == cudaSuccess) e = cudaGraphLaunch(plan->ge1, (cudaStream_t)stream);
        if (e != cudaSuccess) return fail_cuda(e, "single-frame graph launch");
        return CC_OK;
    }
    cudaError_t e = vp->v.launch(p, ncl, vp->smem_bytes, (cudaStream_t)stream);
    if (e != cudaSuccess) return fail_cuda(e, "kernel launch");
    return CC_OK;
}

extern "C" cc_status cc_track_debug(const cc_plan *plan, const void *frames, int batch, float *dx, float *dy, float *peak,
                                    int *iy, int *ix, void *stream)
{
    return track_impl(plan, frames, batch, dx, dy, peak, iy, ix, nullptr, stream);
}

extern "C" cc_status cc_track_profile(const cc_plan *plan, const void *frames, int batch, float *dx, float *dy,
                                      float *peak, unsigned long long *phase_cycles, void *stream)
{
    if (!phase_cycles) return fail(CC_ERR_INVALID_ARG, "cc_track_profile: null pointer");
    return track_impl(plan, frames, batch, dx, dy, peak, nullptr, nullptr, phase_cycles, stream);
}

extern "C" cc_status cc_track(const cc_plan *plan, const void *frames, int batch, float *dx, float *dy, float *peak,
                              void *stream)
{
    return track_impl(plan, frames, batch, dx, dy, peak, nullptr, nullptr, nullptr, stream);
}

// ------------------------------------------------------------------ cc_track_static: the same launch, no allocation anywhere
// The spectrum scratch of the shapes whose spectrum block lives in global memory (the 1024 x 1024 variants, Cfg::SG)
// comes from this file-scope array instead of the plan's cudaMalloc'ed one.  In HOST code the name is only a handle:
// the device address is resolved once per device by cudaGetSymbolAddress (static_scratch_setup) and that pointer is
// what the kernel receives.  Every GPU that loads the library holds the array until the process exits.
static __device__ __align__(256) unsigned char cc_static_scratch[CC_STATIC_SCRATCH_BYTES];

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
void *g_static_ptr[kMaxDevices] = {};  // device address of cc_static_scratch, per device ordinal

// Set-up, once per device, with that device current: resolve the device address of the array.
cc_status static_scratch_setup(void **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, "cudaGetDevice");
    if (dev < 0 || dev >= kMaxDevices) return fail(CC_ERR_UNSUPPORTED, "cc_track_static: device ordinal above 63");
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, cc_static_scratch);
        if (e != cudaSuccess || !ptr) return fail_cuda(e != cudaSuccess ? e : cudaErrorInvalidSymbol, "cudaGetSymbolAddress(cc_static_scratch)");
        g_static_ptr[dev] = ptr;
    }
    *out = g_static_ptr[dev];
    return CC_OK;
}
}  // namespace

extern "C" cc_status cc_track_static(const cc_plan *plan, const void *frames, int batch, float *dx, float *dy, float *peak,
                                     void *stream)
{
    if (!plan || batch < 0) return fail(CC_ERR_INVALID_ARG, "cc_track_static: bad plan or batch");
    if (batch == 0) return CC_OK;
    if (!frames || !dx || !dy) return fail(CC_ERR_INVALID_ARG, "cc_track_static: null pointer");
    if (((uintptr_t)frames & 15u) != 0) return fail(CC_ERR_INVALID_ARG, "cc_track_static: frames must be 16-byte aligned");
    if (plan->ri_a0 > 0.0)
        return fail(CC_ERR_UNSUPPORTED, "cc_track_static: the plan updates its reference image (Eq. (9)); that path uses "
                                        "plan-owned scratch and, for CC-SN, separate kernels: use cc_track");
    // the variant cc_track would take, launched plainly (no graph object, no plan-owned scratch)
    const VarPlan *vp = &plan->thr;
    if (plan->has_lat && batch <= plan->lat.max_clusters && batch * plan->lat.v.CS <= plan->thr.max_clusters * plan->thr.v.CS)
        vp = &plan->lat;
    const int ncl = std::min(batch, vp->max_clusters);
    CcParams p{};
    fill_params(plan, *vp, p);
    p.frames = frames, p.batch = batch, p.dx = dx, p.dy = dy, p.peak = peak;
    p.Sg = nullptr;
    if (vp->v.s_global) {
        // one spectrum block (H x W/2 complex64) per cluster in flight.  The kernel writes every element of its block
        // (row-FFT scatter) before it reads any, so nothing has to be cleared between calls.
        const size_t need = (size_t)ncl * plan->H * (size_t)(plan->W / 2) * sizeof(float2);
        if (need > (size_t)CC_STATIC_SCRATCH_BYTES) {
            char msg[256];
            snprintf(msg, sizeof msg,
                     "cc_track_static: batch %d needs %zu bytes of spectrum scratch (%d frames in flight), the static array holds "
                     "%zu: at %d x %d the largest batch is %zu (use cc_track for more)",
                     batch, need, ncl, (size_t)CC_STATIC_SCRATCH_BYTES, plan->H, plan->W,
                     (size_t)CC_STATIC_SCRATCH_BYTES / ((size_t)plan->H * (size_t)(plan->W / 2) * sizeof(float2)));
            return fail(CC_ERR_UNSUPPORTED, msg);
        }
        void *scratch = nullptr;
        const cc_status st = static_scratch_setup(&scratch);
        if (st != CC_OK) return st;
        p.Sg = reinterpret_cast<float2 *>(scratch);
    }
    const cudaError_t e = vp->v.launch(p, ncl, vp->smem_bytes, (cudaStream_t)stream);
    if (e != cudaSuccess) return fail_cuda(e, "kernel launch");
    return CC_OK;
}

extern "C" cc_status cc_plan_set_host_chunk(cc_plan *plan, int frames_per_chunk)
{
    if (!plan || frames_per_chunk < 0) return fail(CC_ERR_INVALID_ARG, "cc_plan_set_host_chunk: bad plan or chunk");
    plan->host_chunk = frames_per_chunk;
    return CC_OK;
}

extern "C" cc_status cc_track_host(cc_plan *plan, const void *frames, int batch, float *dx, float *dy, float *peak)
{
    if (!plan || batch < 0) return fail(CC_ERR_INVALID_ARG, "cc_track_host: bad plan or batch");
    if (batch == 0) return CC_OK;
    if (!frames || !dx || !dy) return fail(CC_ERR_INVALID_ARG, "cc_track_host: null pointer");
    const size_t fbytes = (size_t)plan->H * plan->W * (plan->dtype == CC_U8 ? 1 : 2);
    // chunk: about 64 MB of frames, at least one wave of clusters (or what cc_plan_set_host_chunk asked for)
    int chunk = plan->host_chunk > 0 ? plan->host_chunk
                                     : (int)std::max<size_t>((size_t)plan->thr.max_clusters, (size_t)(64u << 20) / fbytes);
    chunk = std::min(chunk, batch);
    if (!plan->hs[0]) {
        for (int i = 0; i < 2; ++i) {
            CK(cudaStreamCreateWithFlags(&plan->hs[i], cudaStreamNonBlocking));
            CK(cudaEventCreateWithFlags(&plan->hev[i], cudaEventDisableTiming));
        }
    }
    if (chunk > plan->chunk_cap) {
        for (int i = 0; i < 2; ++i) {
            cudaFree(plan->dframes[i]);
            plan->dframes[i] = nullptr;
            plan->chunk_cap = 0;
            CK(cudaMalloc(&plan->dframes[i], (size_t)chunk * fbytes));
        }
        plan->chunk_cap = chunk;
    }
    if (batch > plan->res_cap) {
        cudaFree(plan->dres);
        plan->dres = nullptr;
        plan->res_cap = 0;
        CK(cudaMalloc((void **)&plan->dres, (size_t)3 * batch * sizeof(float)));
        plan->res_cap = batch;
    }
    // variants that keep the spectrum block in plan-owned global scratch (1024 x 1024): the kernels of the two streams
    // overlap, so the second stream gets a scratch of its own
    for (VarPlan *vp : {&plan->thr, &plan->lat})
        if (vp->ready && vp->v.s_global && !vp->Sg_alt) CK(cudaMalloc((void **)&vp->Sg_alt, vp->sg_bytes));
    float *ddx = plan->dres, *ddy = plan->dres + plan->res_cap, *dpk = plan->dres + 2 * (size_t)plan->res_cap;
    const int nchunks = (batch + chunk - 1) / chunk;
    cc_status st = CC_OK;
    cudaError_t ce = cudaSuccess;
    for (int ci = 0; ci < nchunks && st == CC_OK && ce == cudaSuccess; ++ci) {
        // with the running reference image (Eq. (9)) the chunks must run in order: one stream, one staging buffer
        const int b = plan->ri_a0 > 0.0 ? 0 : (ci & 1), f0 = ci * chunk, n = std::min(chunk, batch - f0);
        cudaStream_t s = plan->hs[b];
        ce = cudaMemcpyAsync(plan->dframes[b], (const unsigned char *)frames + (size_t)f0 * fbytes, (size_t)n * fbytes,
                             cudaMemcpyHostToDevice, s);
        if (ce != cudaSuccess) break;
        st = track_impl(plan, plan->dframes[b], n, ddx + f0, ddy + f0, dpk + f0, nullptr, nullptr, nullptr, (void *)s, b);
        if (st != CC_OK) break;
        ce = cudaMemcpyAsync(dx + f0, ddx + f0, (size_t)n * sizeof(float), cudaMemcpyDeviceToHost, s);
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(dy + f0, ddy + f0, (size_t)n * sizeof(float), cudaMemcpyDeviceToHost, s);
        if (ce == cudaSuccess && peak) ce = cudaMemcpyAsync(peak + f0, dpk + f0, (size_t)n * sizeof(float), cudaMemcpyDeviceToHost, s);
    }
    // drain both streams on every path: no copy into or out of the caller's buffers is in flight after the return
    const cudaError_t s0 = cudaStreamSynchronize(plan->hs[0]), s1 = cudaStreamSynchronize(plan->hs[1]);
    if (st != CC_OK) return st;
    if (ce != cudaSuccess) return fail_cuda(ce, "cc_track_host: copy");
    if (s0 != cudaSuccess) return fail_cuda(s0, "cc_track_host: stream 0");
    if (s1 != cudaSuccess) return fail_cuda(s1, "cc_track_host: stream 1");
    return CC_OK;
}

extern "C" cc_status cc_track_latency_probe(const cc_plan *plan, const void *frames, int n, float *dx, float *dy,
                                            float *peak, double *lat_us, void *stream)
{
    if (!plan || n < 0) return fail(CC_ERR_INVALID_ARG, "cc_track_latency_probe: bad plan or n");
    if (n == 0) return CC_OK;
    if (!frames || !dx || !dy || !lat_us) return fail(CC_ERR_INVALID_ARG, "cc_track_latency_probe: null pointer");
    const size_t fbytes = (size_t)plan->H * plan->W * (plan->dtype == CC_U8 ? 1 : 2);
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaStreamSynchronize(st));
    for (int i = 0; i < n; ++i) {
        struct timespec t0, t1;
        clock_gettime(CLOCK_MONOTONIC, &t0);
        cc_status s = cc_track(plan, (const unsigned char *)frames + (size_t)i * fbytes, 1, dx + i, dy + i,
                               peak ? peak + i : nullptr, stream);
        if (s != CC_OK) return s;
        cudaError_t e = cudaStreamSynchronize(st);
        clock_gettime(CLOCK_MONOTONIC, &t1);
        if (e != cudaSuccess) return fail_cuda(e, "cudaStreamSynchronize");
        lat_us[i] = (double)(t1.tv_sec - t0.tv_sec) * 1e6 + (double)(t1.tv_nsec - t0.tv_nsec) * 1e-3;
    }
    return CC_OK;
}

// ------------------------------------------------------------------ real-time session
struct cc_rt {
    cc_plan *plan = nullptr;
    const VarPlan *vp = nullptr;
    cudaStream_t stream = nullptr;
    void *hbox = nullptr;                      // mapped host memory: [0,16) command, [64,80) result, [128,132) alive
    volatile unsigned long long *cmd = nullptr;
    volatile uint32_t *res = nullptr;
    volatile int *alive = nullptr;
    void *dbox = nullptr;                      // device view of hbox
    unsigned long long seq = 0;                // sequence number of the last submitted frame
    const void *pending = nullptr;             // frame of that submission (for a restart)
    bool in_flight = false;
    unsigned long long timeout_ns = 0;
    float2 *Sg = nullptr;                      // the session's own spectrum scratch (s_global variants)
};

static double mono_us()
{
    struct timespec t;
    clock_gettime(CLOCK_MONOTONIC, &t);
    return (double)t.tv_sec * 1e6 + (double)t.tv_nsec * 1e-3;
}

static cc_status rt_launch(cc_rt *rt)
{
    if (rt->plan->sn && rt->plan->ri_a0 > 0.0)
        return fail(CC_ERR_UNSUPPORTED, "a real-time session cannot serve a CC-SN plan with the Eq. (9) update: its reference is "
                                        "rewritten by separate kernels between frames (use cc_track)");
    // a fresh kernel starts counting at sequence 0: rebase the mailbox
    CK(cudaStreamSynchronize(rt->stream));
    rt->seq = 0;
    rt->cmd[0] = 0, rt->cmd[1] = 0;
    rt->res[3] = 0;
    *rt->alive = 1;
    __sync_synchronize();
    CcParams p{};
    fill_params(rt->plan, *rt->vp, p);
    p.batch = 0;
    p.rt_cmd = (const volatile unsigned long long *)rt->dbox;
    p.rt_res = (float *)((char *)rt->dbox + 64);
    p.rt_alive = (int *)((char *)rt->dbox + 128);
    p.rt_timeout_ns = rt->timeout_ns;
    if (rt->Sg) p.Sg = rt->Sg;  // not the plan's: cc_track(batch 1) on the same plan may run beside the session
    cudaError_t e = rt->vp->v.launch(p, 1, rt->vp->smem_bytes, rt->stream);
    if (e != cudaSuccess) {
        *rt->alive = 0;
        return fail_cuda(e, "session kernel launch");
    }
    return CC_OK;
}

extern "C" cc_status cc_rt_close(cc_rt *rt)
{
    if (!rt) return CC_OK;
    if (rt->cmd) {
        rt->cmd[0] = ~0ull;  // quit
        __sync_synchronize();
    }
    if (rt->stream) {
        cudaStreamSynchronize(rt->stream);
        cudaStreamDestroy(rt->stream);
    }
    if (rt->hbox) cudaFreeHost(rt->hbox);
    cudaFree(rt->Sg);
    delete rt;
    return CC_OK;
}

extern "C" cc_status cc_rt_open(cc_plan *plan, int idle_timeout_ms, cc_rt **out)
{
    if (!plan || !out) return fail(CC_ERR_INVALID_ARG, "cc_rt_open: null pointer");
    cc_rt *rt = new (std::nothrow) cc_rt();
    if (!rt) return fail(CC_ERR_NOMEM, "host allocation failed");
    rt->plan = plan;
    rt->vp = plan->has_lat ? &plan->lat : &plan->thr;
    rt->timeout_ns = (unsigned long long)(idle_timeout_ms > 0 ? idle_timeout_ms : 1000) * 1000000ull;
    cudaError_t e = cudaHostAlloc(&rt->hbox, 256, cudaHostAllocMapped | cudaHostAllocPortable);
    if (e == cudaSuccess) {
        memset(rt->hbox, 0, 256);
        e = cudaHostGetDevicePointer(&rt->dbox, rt->hbox, 0);
    }
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&rt->stream, cudaStreamNonBlocking);
    if (e == cudaSuccess && rt->vp->v.s_global)
        e = cudaMalloc((void **)&rt->Sg, (size_t)rt->vp->v.CS * ((size_t)plan->H * (plan->W / 2 / rt->vp->v.CS)) * sizeof(float2));
    if (e != cudaSuccess) {
        cc_status s = fail_cuda(e, "cc_rt_open");
        if (rt->hbox) cudaFreeHost(rt->hbox);
        if (rt->stream) cudaStreamDestroy(rt->stream);
        cudaFree(rt->Sg);
        delete rt;
        return s;
    }
    rt->cmd = (volatile unsigned long long *)rt->hbox;
    rt->res = (volatile uint32_t *)((char *)rt->hbox + 64);
    rt->alive = (volatile int *)((char *)rt->hbox + 128);
    cc_status s = rt_launch(rt);
    if (s != CC_OK) {
        rt->cmd = nullptr;
        cc_rt_close(rt);
        return s;
    }
    *out = rt;
    return CC_OK;
}

extern "C" cc_status cc_rt_submit(cc_rt *rt, const void *frame)
{
    if (!rt || !frame) return fail(CC_ERR_INVALID_ARG, "cc_rt_submit: null pointer");
    if (((uintptr_t)frame & 15u) != 0) return fail(CC_ERR_INVALID_ARG, "cc_rt_submit: frame must be 16-byte aligned");
    if (rt->in_flight) return fail(CC_ERR_INVALID_ARG, "cc_rt_submit: a frame is already in flight");
    if (!*rt->alive) {  // the kernel left after its idle timeout: start it again
        cc_status s = rt_launch(rt);
        if (s != CC_OK) return s;
    }
    rt->pending = frame;
    ++rt->seq;
    rt->cmd[1] = (unsigned long long)(uintptr_t)frame | (rt->seq & 15ull);  // tag: low 4 bits of the sequence number
    __atomic_store_n((unsigned long long *)&rt->cmd[0], rt->seq, __ATOMIC_RELEASE);
    rt->in_flight = true;
    return CC_OK;
}

extern "C" cc_status cc_rt_wait(cc_rt *rt, float *dx, float *dy, float *peak)
{
    if (!rt || !dx || !dy) return fail(CC_ERR_INVALID_ARG, "cc_rt_wait: null pointer");
    if (!rt->in_flight) return fail(CC_ERR_INVALID_ARG, "cc_rt_wait: no frame submitted");
    int restarts = 0;
    double t0 = mono_us();
    for (;;) {
        if (__atomic_load_n((uint32_t *)&rt->res[3], __ATOMIC_ACQUIRE) == (uint32_t)rt->seq) break;
#if defined(__x86_64__) || defined(__i386__)
        __builtin_ia32_pause();  // spin-wait hint: the result arrives by a PCIe write into this cache line
#endif
        if (mono_us() - t0 > 2.0e5) {  // 200 ms without an answer
            // the kernel may have hit its idle timeout just as the frame was submitted: restart once
            if (!*rt->alive && restarts == 0) {
                const void *frame = rt->pending;
                rt->in_flight = false;
                cc_status s = rt_launch(rt);
                if (s == CC_OK) s = cc_rt_submit(rt, frame);
                if (s != CC_OK) return s;
                ++restarts;
                t0 = mono_us();
                continue;
            }
            rt->in_flight = false;
            cudaError_t e = cudaStreamQuery(rt->stream);
            return fail(CC_ERR_CUDA, std::string("cc_rt_wait: no answer from the session kernel (") +
                                         cudaGetErrorString(e == cudaErrorNotReady ? cudaSuccess : e) + ")");
        }
    }
    union { uint32_t u; float f; } c;
    c.u = rt->res[0], *dx = c.f;
    c.u = rt->res[1], *dy = c.f;
    c.u = rt->res[2];
    if (peak) *peak = c.f;
    rt->in_flight = false;
    return CC_OK;
}

extern "C" cc_status cc_rt_track(cc_rt *rt, const void *frame, float *dx, float *dy, float *peak)
{
    cc_status s = cc_rt_submit(rt, frame);
    if (s != CC_OK) return s;
    return cc_rt_wait(rt, dx, dy, peak);
}

extern "C" cc_status cc_rt_latency_probe(cc_rt *rt, const void *frames, int n, float *dx, float *dy, float *peak,
                                         double *lat_us)
{
    if (!rt || n < 0) return fail(CC_ERR_INVALID_ARG, "cc_rt_latency_probe: bad session or n");
    if (n == 0) return CC_OK;
    if (!frames || !dx || !dy || !lat_us) return fail(CC_ERR_INVALID_ARG, "cc_rt_latency_probe: null pointer");
    const size_t fbytes = (size_t)rt->plan->H * rt->plan->W * (rt->plan->dtype == CC_U8 ? 1 : 2);
    for (int i = 0; i < n; ++i) {
        const double t0 = mono_us();
        cc_status s = cc_rt_track(rt, (const unsigned char *)frames + (size_t)i * fbytes, dx + i, dy + i, peak ? peak + i : nullptr);
        lat_us[i] = mono_us() - t0;
        if (s != CC_OK) return s;
    }
    return CC_OK;
}

// ------------------------------------------------------------------ running reference image
// scratch for the frames' forward spectra (one copy per cluster), the slot -> frequency table, the device-resident mean
static cc_status ensure_spectrum_scratch(cc_plan *plan, int clusters)
{
    const int H = plan->H, W = plan->W;
    cudaError_t e = cudaSuccess;
    if (!plan->col_freq) {
        std::vector<int16_t> cf(H);
        for (int p = 0; p < H; ++p) {
            const int ky = cc_freq_of_slot(H, p, false);
            cf[p] = (int16_t)(2 * ky < H ? ky : ky - H);  // Nyquist slot: -H/2
        }
        e = upload(&plan->col_freq, cf, &plan->table_bytes);
        if (e == cudaSuccess) e = cudaMalloc((void **)&plan->ri_emean, sizeof(double));
        if (e == cudaSuccess) e = cudaMemcpy(plan->ri_emean, &plan->Emean, sizeof(double), cudaMemcpyHostToDevice);
    }
    if (e == cudaSuccess && clusters > plan->keep_clusters) {
        cudaFree(plan->ri_Fs), cudaFree(plan->ri_Fab);
        plan->ri_Fs = nullptr, plan->ri_Fab = nullptr, plan->keep_clusters = 0;
        e = cudaMalloc((void **)&plan->ri_Fs, (size_t)clusters * H * (W / 2) * sizeof(float2));
        if (e == cudaSuccess) e = cudaMalloc((void **)&plan->ri_Fab, (size_t)clusters * H * sizeof(float4));
        if (e == cudaSuccess) plan->keep_clusters = clusters;
    }
    if (e != cudaSuccess)
        return e == cudaErrorMemoryAllocation ? fail(CC_ERR_NOMEM, "device allocation failed") : fail_cuda(e, "spectrum scratch setup");
    return CC_OK;
}

// CC-SN plans: the fp64 state G = F[E] (created from the caller's reference image on first use)
static cc_status ensure_sn_state(cc_plan *plan)
{
    cc_status st = ensure_spectrum_scratch(plan, 0);
    if (st != CC_OK || plan->sn_state) return st;
    cudaError_t e = cc_sn_state_create(&plan->sn_state, plan->H, plan->W, plan->u, plan->dtype, plan->sn_eps, plan->sn_ref.data());
    if (e != cudaSuccess)
        return e == cudaErrorMemoryAllocation ? fail(CC_ERR_NOMEM, "device allocation failed") : fail_cuda(e, "CC-SN reference state");
    return CC_OK;
}

extern "C" cc_status cc_plan_enable_reference_update(cc_plan *plan, double a0)
{
    if (!plan || !(a0 >= 0.0 && a0 <= 1.0)) return fail(CC_ERR_INVALID_ARG, "cc_plan_enable_reference_update: bad plan or a0");
    CK(cudaDeviceSynchronize());
    if (a0 == 0.0) {
        plan->ri_a0 = 0.0;
        return CC_OK;
    }
    cc_status st = plan->sn ? ensure_sn_state(plan) : ensure_spectrum_scratch(plan, 1);
    if (st != CC_OK) return st;
    plan->ri_a0 = a0;
    return CC_OK;
}

// the state of a CC-SN plan as a half spectrum (H x (W/2+1) complex128); creates the state on first use
static cc_status sn_half_spectrum(cc_plan *plan, std::vector<double> &half)
{
    cc_status st = ensure_sn_state(plan);
    if (st != CC_OK) return st;
    const int H = plan->H, W = plan->W, Wh = W / 2;
    std::vector<double> full((size_t)H * W * 2);
    int flag = 0;
    CK(cc_sn_read_state(plan->sn_state, full.data(), &flag));
    if (flag) return fail(CC_ERR_INVALID_ARG, "CC-SN: reference + epsilon became non-positive in some pixel during the updates");
    half.resize((size_t)H * (Wh + 1) * 2);
    for (int ky = 0; ky < H; ++ky)
        memcpy(&half[(size_t)ky * (Wh + 1) * 2], &full[(size_t)ky * W * 2], (size_t)(Wh + 1) * 2 * sizeof(double));
    return CC_OK;
}

extern "C" cc_status cc_plan_get_reference_spectrum_f64(const cc_plan *plan, double *out)
{
    if (!plan || !out) return fail(CC_ERR_INVALID_ARG, "cc_plan_get_reference_spectrum_f64: null pointer");
    const int H = plan->H, Wh = plan->W / 2;
    const size_t n = (size_t)H * (Wh + 1);
    if (plan->sn) {
        std::vector<double> half;
        cc_status st = sn_half_spectrum(const_cast<cc_plan *>(plan), half);
        if (st != CC_OK) return st;
        memcpy(out, half.data(), n * 2 * sizeof(double));
        return CC_OK;
    }
    std::vector<float> f(n * 2);
    cc_status st = cc_plan_get_reference_spectrum(plan, f.data());
    if (st != CC_OK) return st;
    for (size_t i = 0; i < n * 2; ++i) out[i] = (double)f[i];
    return CC_OK;
}

extern "C" cc_status cc_plan_get_reference_spectrum(const cc_plan *plan, float *out)
{
    if (!plan || !out) return fail(CC_ERR_INVALID_ARG, "cc_plan_get_reference_spectrum: null pointer");
    const int H = plan->H, W = plan->W, Wh = W / 2;
    if (plan->sn) {  // CC-SN: the plan's tables hold the weight spectrum; F[E] is the fp64 state
        std::vector<double> half;
        cc_status st = sn_half_spectrum(const_cast<cc_plan *>(plan), half);
        if (st != CC_OK) return st;
        for (size_t i = 0; i < half.size(); ++i) out[i] = (float)half[i];
        return CC_OK;
    }
    CK(cudaDeviceSynchronize());
    std::vector<float2> Gt((size_t)H * Wh);
    std::vector<float4> ab(H);
    double emean = plan->Emean;
    CK(cudaMemcpy(Gt.data(), plan->Gt, Gt.size() * sizeof(float2), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(ab.data(), plan->ab, ab.size() * sizeof(float4), cudaMemcpyDeviceToHost));
    if (plan->ri_emean) CK(cudaMemcpy(&emean, plan->ri_emean, sizeof(double), cudaMemcpyDeviceToHost));
    const double HW = (double)H * (double)W;
    for (int p = 0; p < H; ++p) {
        const int ky = cc_freq_of_slot(H, p, false);
        float *row = out + (size_t)ky * (Wh + 1) * 2;
        for (int q = 1; q < Wh; ++q) {  // stored: conj(G) / (HW)
            row[2 * q] = (float)((double)Gt[(size_t)p * Wh + q].x * HW);
            row[2 * q + 1] = (float)(-(double)Gt[(size_t)p * Wh + q].y * HW);
        }
        row[0] = ky == 0 ? (float)(emean * HW) : (float)((double)ab[p].x * HW);  // the DC bin is kept as the mean
        row[1] = ky == 0 ? 0.f : (float)(-(double)ab[p].y * HW);
        row[2 * Wh] = (float)((double)ab[p].z * HW);
        row[2 * Wh + 1] = (float)(-(double)ab[p].w * HW);
    }
    return CC_OK;
}

// ------------------------------------------------------------------ offline iteration (Eq. (8))
extern "C" cc_status cc_track_accumulate(cc_plan *plan, const void *frames, int batch, float *dx, float *dy, float *peak,
                                         void *stream)
{
    if (!plan || batch < 0) return fail(CC_ERR_INVALID_ARG, "cc_track_accumulate: bad plan or batch");
    if (plan->ri_a0 > 0.0) return fail(CC_ERR_INVALID_ARG, "cc_track_accumulate: switch the Eq. (9) update off first");
    if (batch == 0) return CC_OK;
    if (!frames || !dx || !dy) return fail(CC_ERR_INVALID_ARG, "cc_track_accumulate: null pointer");
    if (((uintptr_t)frames & 15u) != 0) return fail(CC_ERR_INVALID_ARG, "cc_track_accumulate: frames must be 16-byte aligned");
    if (plan->sn) {
        // CC-SN (R19): plain tracking of the batch against the current weight, then the aligned RAW spectra
        // are summed in fp64 (frame order: deterministic)
        cc_status st = ensure_sn_state(plan);  // first use: may synchronise
        if (st == CC_OK) st = track_impl(plan, frames, batch, dx, dy, peak, nullptr, nullptr, nullptr, stream);
        if (st != CC_OK) return st;
        cudaError_t e = cc_sn_accumulate(plan->sn_state, frames, batch, dy, dx, (cudaStream_t)stream);
        if (e != cudaSuccess)
            return e == cudaErrorMemoryAllocation ? fail(CC_ERR_NOMEM, "device allocation failed") : fail_cuda(e, "CC-SN accumulation");
        plan->acc_count += batch;
        return CC_OK;
    }
    const VarPlan *vp = &plan->thr;
    const int H = plan->H, W = plan->W, ncmax = vp->max_clusters;
    if (plan->acc_clusters < ncmax) {  // first use: may synchronise
        CK(cudaDeviceSynchronize());
        cc_status st = ensure_spectrum_scratch(plan, ncmax);
        if (st != CC_OK) return st;
        cudaFree(plan->acc_G), cudaFree(plan->acc_ab), cudaFree(plan->acc_mean);
        plan->acc_G = nullptr, plan->acc_ab = nullptr, plan->acc_mean = nullptr, plan->acc_clusters = 0, plan->acc_count = 0;
        cudaError_t e = cudaMalloc((void **)&plan->acc_G, (size_t)ncmax * H * (W / 2) * sizeof(float2));
        if (e == cudaSuccess) e = cudaMalloc((void **)&plan->acc_ab, (size_t)ncmax * H * sizeof(float4));
        if (e == cudaSuccess) e = cudaMalloc((void **)&plan->acc_mean, (size_t)ncmax * sizeof(double));
        if (e == cudaSuccess) e = cudaMemset(plan->acc_G, 0, (size_t)ncmax * H * (W / 2) * sizeof(float2));
        if (e == cudaSuccess) e = cudaMemset(plan->acc_ab, 0, (size_t)ncmax * H * sizeof(float4));
        if (e == cudaSuccess) e = cudaMemset(plan->acc_mean, 0, (size_t)ncmax * sizeof(double));
        if (e != cudaSuccess)
            return e == cudaErrorMemoryAllocation ? fail(CC_ERR_NOMEM, "device allocation failed") : fail_cuda(e, "accumulator setup");
        plan->acc_clusters = ncmax;
    }
    CcParams p{};
    fill_params(plan, *vp, p);
    p.frames = frames, p.batch = batch, p.dx = dx, p.dy = dy, p.peak = peak;
    p.ri_Fs = plan->ri_Fs, p.ri_Fab = plan->ri_Fab, p.col_freq = plan->col_freq, p.ri_a0 = 0.0;
    p.acc_G = plan->acc_G, p.acc_ab = plan->acc_ab, p.acc_mean = plan->acc_mean;
    const int ncl = std::min(batch, ncmax);
    cudaError_t e = vp->v.launch(p, ncl, vp->smem_bytes, (cudaStream_t)stream);
    if (e != cudaSuccess) return fail_cuda(e, "kernel launch");
    plan->acc_count += batch;
    return CC_OK;
}

// Gt <- conj(sum over clusters) / (N HW), clusters in index order (deterministic); accumulators cleared
__global__ void cc_reduce_reference_kernel(float2 *acc_G, float4 *acc_ab, double *acc_mean, int ncl, int H, int Wh,
                                           const int16_t *col_freq, float2 *Gt, float4 *ab, double *emean, double inv, double invN)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    const size_t plane = (size_t)H * Wh;
    if (idx < H * Wh && idx % Wh != 0) {
        double sx = 0.0, sy = 0.0;
        for (int c = 0; c < ncl; ++c) {
            const float2 v = acc_G[c * plane + idx];
            sx += (double)v.x, sy += (double)v.y;
            acc_G[c * plane + idx] = make_float2(0.f, 0.f);
        }
        Gt[idx] = make_float2((float)(sx * inv), (float)(-sy * inv));
    }
    if (idx < H) {
        double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
        for (int c = 0; c < ncl; ++c) {
            const float4 v = acc_ab[(size_t)c * H + idx];
            a0 += (double)v.x, a1 += (double)v.y, a2 += (double)v.z, a3 += (double)v.w;
            acc_ab[(size_t)c * H + idx] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        const bool dc = col_freq[idx] == 0;  // the DC bin of the reference stays zero (R10)
        ab[idx] = make_float4(dc ? 0.f : (float)(a0 * inv), dc ? 0.f : (float)(-a1 * inv), (float)(a2 * inv), (float)(-a3 * inv));
    }
    if (idx == 0) {
        double m = 0.0;
        for (int c = 0; c < ncl; ++c) m += acc_mean[c], acc_mean[c] = 0.0;
        *emean = m * invN;
    }
}

extern "C" cc_status cc_plan_update_reference_from_accumulator(cc_plan *plan, void *stream)
{
    if (!plan) return fail(CC_ERR_INVALID_ARG, "cc_plan_update_reference_from_accumulator: null plan");
    if (plan->sn && plan->acc_count > 0 && plan->sn_state) {
        const CcSnTables t{plan->Gt, plan->ab, plan->ri_emean, plan->col_freq};
        cudaError_t e = cc_sn_finish_pass(plan->sn_state, plan->acc_count, t, (cudaStream_t)stream);
        if (e != cudaSuccess) return fail_cuda(e, "CC-SN reference update");
        plan->acc_count = 0;
        return CC_OK;
    }
    if (plan->acc_count <= 0 || !plan->acc_G) return fail(CC_ERR_INVALID_ARG, "nothing accumulated: call cc_track_accumulate first");
    const int H = plan->H, Wh = plan->W / 2;
    const double invN = 1.0 / (double)plan->acc_count, inv = invN / ((double)H * (double)plan->W);
    const int threads = 256, blocks = (H * Wh + threads - 1) / threads;
    cc_reduce_reference_kernel<<<blocks, threads, 0, (cudaStream_t)stream>>>(plan->acc_G, plan->acc_ab, plan->acc_mean,
                                                                             plan->acc_clusters, H, Wh, plan->col_freq, plan->Gt,
                                                                             plan->ab, plan->ri_emean, inv, invN);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "reference reduction launch");
    plan->acc_count = 0;
    return CC_OK;
}

// ------------------------------------------------------------------ drift correction
// One warp: the lanes fetch 32 samples at a time (coalesced), lane 0 runs the recurrence of Eqs. (10)-(12) in fp64
// with separately rounded multiplies and adds (no contraction: the same roundings as a plain C evaluation), the
// lanes store the 32 corrected samples.
__global__ void __launch_bounds__(32, 1) cc_drift_kernel(const float *dx, const float *dy, int n, double a0, double max_step,
                                                         double *state, float *dxc, float *dyc)
{
    const int lane = threadIdx.x;
    const double b1 = 1.0 - a0, b1m1 = b1 - 1.0;
    double Rx = state[0], Ry = state[1];
    for (int base = 0; base < n; base += 32) {
        const int i = base + lane;
        const float fx = i < n ? dx[i] : 0.f, fy = i < n ? dy[i] : 0.f;
        float ox = 0.f, oy = 0.f;
        const int cnt = min(32, n - base);
        for (int k = 0; k < cnt; ++k) {
            const double rx = (double)__shfl_sync(0xffffffffu, fx, k), ry = (double)__shfl_sync(0xffffffffu, fy, k);
            if (max_step > 0.0) {
                const double ex = __dadd_rn(__dmul_rn(a0, rx), __dmul_rn(b1m1, Rx));  // Eq. (11)
                const double ey = __dadd_rn(__dmul_rn(a0, ry), __dmul_rn(b1m1, Ry));
                const double norm = __dsqrt_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)));
                if (norm > max_step) {  // Eq. (12), first case
                    Rx = __dadd_rn(Rx, __dmul_rn(max_step, __ddiv_rn(ex, norm)));
                    Ry = __dadd_rn(Ry, __dmul_rn(max_step, __ddiv_rn(ey, norm)));
                } else {
                    Rx = __dadd_rn(Rx, ex);
                    Ry = __dadd_rn(Ry, ey);
                }
            } else {  // Eq. (10)
                Rx = __dadd_rn(__dmul_rn(a0, rx), __dmul_rn(b1, Rx));
                Ry = __dadd_rn(__dmul_rn(a0, ry), __dmul_rn(b1, Ry));
            }
            if (lane == k) ox = (float)(rx - Rx), oy = (float)(ry - Ry);
        }
        if (i < n) dxc[i] = ox, dyc[i] = oy;
    }
    if (lane == 0) state[0] = Rx, state[1] = Ry;
}

extern "C" cc_status cc_drift_correct(const float *dx, const float *dy, int n, double a0, double max_step, double *state,
                                      float *dxc, float *dyc, void *stream)
{
    if (n < 0 || !(a0 >= 0.0 && a0 <= 1.0)) return fail(CC_ERR_INVALID_ARG, "cc_drift_correct: bad n or a0");
    if (n == 0) return CC_OK;
    if (!dx || !dy || !state || !dxc || !dyc) return fail(CC_ERR_INVALID_ARG, "cc_drift_correct: null pointer");
    cc_status st = check_device();
    if (st != CC_OK) return st;
    cc_drift_kernel<<<1, 32, 0, (cudaStream_t)stream>>>(dx, dy, n, a0, max_step, state, dxc, dyc);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "drift kernel launch");
    return CC_OK;
}

extern "C" cc_status cc_plan_info(const cc_plan *plan, cc_plan_info_t *info)
{
    if (!plan || !info) return fail(CC_ERR_INVALID_ARG, "cc_plan_info: null pointer");
    memset(info, 0, sizeof(*info));
    info->H = plan->H, info->W = plan->W, info->upsample = plan->u, info->dtype = plan->dtype, info->grid_M = plan->M;
    info->cluster_size = plan->thr.v.CS, info->threads = plan->thr.v.NT, info->smem_bytes = plan->thr.smem_bytes;
    info->max_clusters = plan->thr.max_clusters;
    info->lat_cluster_size = plan->has_lat ? plan->lat.v.CS : 0;
    info->lat_max_clusters = plan->has_lat ? plan->lat.max_clusters : 0;
    info->scratch_bytes = (long long)(plan->thr.sg_bytes + (plan->has_lat ? plan->lat.sg_bytes : 0));
    info->table_bytes = (long long)plan->table_bytes;
    info->super_blocks = plan->thr.nsb, info->offsets_per_cta = plan->thr.DS;
    info->tensor_core_stage1 = plan->thr.v.tc1;
    return CC_OK;
}

// ------------------------------------------------------------------ FP32 peak probes (include/cc_bench.h)
namespace {
struct DevBuf {  // freed on every return path
    void *p = nullptr;
    ~DevBuf() { cudaFree(p); }
};
struct EvPair {
    cudaEvent_t a = nullptr, b = nullptr;
    ~EvPair()
    {
        if (a) cudaEventDestroy(a);
        if (b) cudaEventDestroy(b);
    }
};
}  // namespace

__global__ void __launch_bounds__(1024, 1) cc_ffma_probe_kernel(float *out, int iters)
{
    float a0 = threadIdx.x * 1e-3f, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f, a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f,
          a7 = a0 + 7.f;
    const float b = 0.999f, c = 1e-3f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            a0 = fmaf(a0, b, c), a1 = fmaf(a1, b, c), a2 = fmaf(a2, b, c), a3 = fmaf(a3, b, c);
            a4 = fmaf(a4, b, c), a5 = fmaf(a5, b, c), a6 = fmaf(a6, b, c), a7 = fmaf(a7, b, c);
        }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
}

extern "C" cc_status cc_fp32_peak_probe(double *tflops, void *stream)
{
    if (!tflops) return fail(CC_ERR_INVALID_ARG, "cc_fp32_peak_probe: null pointer");
    cc_status st = check_device();
    if (st != CC_OK) return st;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int blocks = sms * 2, threads = 1024, iters = 4096;
    DevBuf ob;
    EvPair ev;
    CK(cudaMalloc(&ob.p, (size_t)blocks * threads * sizeof(float)));
    float *out = (float *)ob.p;
    CK(cudaEventCreate(&ev.a));
    CK(cudaEventCreate(&ev.b));
    const cudaEvent_t e0 = ev.a, e1 = ev.b;
    cudaStream_t s = (cudaStream_t)stream;
    cc_ffma_probe_kernel<<<blocks, threads, 0, s>>>(out, 64);
    float best = 1e30f;
    for (int r = 0; r < 3; ++r) {
        CK(cudaEventRecord(e0, s));
        cc_ffma_probe_kernel<<<blocks, threads, 0, s>>>(out, iters);
        CK(cudaEventRecord(e1, s));
        CK(cudaEventSynchronize(e1));
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        best = std::min(best, ms);
    }
    const double flops = 2.0 * 8.0 * 16.0 * (double)iters * (double)blocks * (double)threads;
    *tflops = flops / ((double)best * 1e-3) / 1e12;
    return CC_OK;
}

__global__ void __launch_bounds__(256, 1) cc_ffma_tile_probe_kernel(float *out, const float *in, int iters)
{
    float a[8], b[8], acc[8][8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = in[threadIdx.x + i], b[i] = in[threadIdx.x + 8 + i];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
        a[0] += 1e-9f, b[7] -= 1e-9f;  // keeps the loop from being hoisted (2 FADD per 64 FFMA)
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) s += acc[i][j];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

extern "C" cc_status cc_fp32_tile_probe(double *tflops, void *stream)
{
    if (!tflops) return fail(CC_ERR_INVALID_ARG, "cc_fp32_tile_probe: null pointer");
    cc_status st = check_device();
    if (st != CC_OK) return st;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int blocks = sms, threads = 256, iters = 20000;  // 8 warps per SM, as the fused kernel runs
    DevBuf ob, ib;
    EvPair ev;
    CK(cudaMalloc(&ob.p, (size_t)blocks * threads * sizeof(float)));
    CK(cudaMalloc(&ib.p, 4096));
    float *out = (float *)ob.p, *in = (float *)ib.p;
    CK(cudaMemset(in, 0, 4096));
    CK(cudaEventCreate(&ev.a));
    CK(cudaEventCreate(&ev.b));
    const cudaEvent_t e0 = ev.a, e1 = ev.b;
    cudaStream_t s = (cudaStream_t)stream;
    cc_ffma_tile_probe_kernel<<<blocks, threads, 0, s>>>(out, in, 64);
    float best = 1e30f;
    for (int r = 0; r < 3; ++r) {
        CK(cudaEventRecord(e0, s));
        cc_ffma_tile_probe_kernel<<<blocks, threads, 0, s>>>(out, in, iters);
        CK(cudaEventRecord(e1, s));
        CK(cudaEventSynchronize(e1));
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        best = std::min(best, ms);
    }
    *tflops = 2.0 * 64.0 * (double)iters * (double)blocks * (double)threads / ((double)best * 1e-3) / 1e12;
    return CC_OK;
}

extern "C" const char *cc_status_string(cc_status s)
{
    switch (s) {
        case CC_OK: return "CC_OK";
        case CC_ERR_INVALID_ARG: return "CC_ERR_INVALID_ARG";
        case CC_ERR_UNSUPPORTED: return "CC_ERR_UNSUPPORTED";
        case CC_ERR_NOMEM: return "CC_ERR_NOMEM";
        case CC_ERR_CUDA: return "CC_ERR_CUDA";
        case CC_ERR_ARCH: return "CC_ERR_ARCH";
    }
    return "CC_ERR_UNKNOWN";
}

extern "C" const char *cc_last_error(void) { return g_err.c_str(); }

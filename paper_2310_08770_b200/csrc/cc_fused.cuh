// cc_fused.cuh -- the fused per-frame displacement kernel for sm_100a.
//
// One thread-block cluster of CS CTAs processes one frame at a time
// (persistent over the batch).  Steps (PAPER.md citations in
// include/cc.h and DESIGN.md):
//   a1 ingest    : cp.async.bulk (TMA) of raw u8/u16 rows into shared memory
//   a2 fwd FFT   : two real rows per complex row FFT (per warp), results
//                  scattered to the column owners through DSMEM; column FFT
//   a3 product   : fused into the last forward / first inverse column pass
//   a4 inv FFT   : column inverse -> Q[y][kx] (kept: it feeds a6), row C2R
//   a5 argmax    : streamed out of the row C2R, never stored; fp64 3x3 polish
//   a6 upsampled : both upsampling matrices are even/odd-symmetric about the window centre, so
//                  stage 1  [T(c+d) + T(c-d), T(c+d) - T(c-d)] = [Ee, Eo] * [Q(y0+j) + Q(y0-j), Q(y0+j) - Q(y0-j)]
//                  stage 2  [C(m,c+e) + C(m,c-e), C(m,c-e) - C(m,c+e)] / 2 = [T_re * cos, T_im * sin]
//                  (FP32 register-tiled GEMMs with half the multiply-adds of the plain products);
//                  operand tiles stream L2 -> smem through a TMA ring refilled by the last warp to release a slot
//   a7 argmax    : streamed out of stage 2, fp64 3x3 hill-climb polish, compose
// Product code: shares nothing with oracle/.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "cc_common.h"

namespace ccf {
namespace cg = cooperative_groups;

constexpr int XN = 10;    // doubles per cluster-exchange record

// ------------------------------------------------------------------ schedule fuzzing (build.py --fuzz: -DCC_FUZZ)
// compute-sanitizer is closed on the pool this was developed on, so the race check is done by perturbation: in the fuzz
// build every synchronisation point (mbarrier waits, ring acquire / release, cluster exchanges, CTA / cluster barriers,
// warp-level FFT passes) is preceded by a pseudo-random per-LANE delay of up to ~2 us.  A missing barrier or a slot
// released too early then shows up as results that change from run to run or differ from the plain build
// (paper_2310_08770_b200/selftest.py --compare-fuzz; profiles/sanitizer_r2.md).
#ifdef CC_FUZZ
__device__ __forceinline__ void cc_jitter()
{
    unsigned c = (unsigned)clock64();
    unsigned h = (c ^ (threadIdx.x * 2654435761u) ^ (blockIdx.x * 40503u)) * 2246822519u;
    h ^= h >> 15;
    if ((h & 7u) == 0u) __nanosleep((h >> 8) & 2047u);
}
#define CC_JITTER() cc_jitter()
#define __syncthreads() (cc_jitter(), __syncthreads())
#else
#define CC_JITTER() ((void)0)
#endif

// ------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *b, uint32_t cnt)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(cnt) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *b, uint32_t parity)
{
    CC_JITTER();
    uint32_t ok;
    const uint32_t a = smem_u32(b);
    do {
        asm volatile(
            "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
            : "=r"(ok)
            : "r"(a), "r"(parity)
            : "memory");
    } while (!ok);
}
// TMA 1D bulk copy global -> shared, completion on an mbarrier
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void *src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
// address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa_u32(uint32_t saddr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
// 8-byte store into a peer CTA's shared memory that completes 8 tx-bytes on the peer's mbarrier
__device__ __forceinline__ void st_async_b64(uint32_t raddr, uint64_t v, uint32_t rbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];" ::"r"(raddr), "l"(v), "r"(rbar)
                 : "memory");
}
// 16-byte flavour (four floats)
__device__ __forceinline__ void st_async_v4(uint32_t raddr, float4 v, uint32_t rbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1, %2, %3, %4}, [%5];" ::"r"(raddr),
                 "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "r"(rbar)
                 : "memory");
}
__device__ __forceinline__ void ld_sys_v2u64(const volatile unsigned long long *p, uint64_t &a, uint64_t &b)
{
    unsigned long long x, y;
    asm volatile("ld.volatile.global.v2.u64 {%0, %1}, [%2];" : "=l"(x), "=l"(y) : "l"(p) : "memory");
    a = x, b = y;
}
__device__ __forceinline__ uint64_t globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// ---- 5th-generation tensor cores (tcgen05): shared-memory matrix descriptor (no swizzle, K-major: 8-row x 16-byte core
// matrices; lbo = byte distance of the two 16-byte K chunks, sbo = byte distance of successive 8-row groups; version 1)
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo)
{
    return (uint64_t)((saddr >> 4) & 0x3fffu) | ((uint64_t)((lbo >> 4) & 0x3fffu) << 16) | ((uint64_t)((sbo >> 4) & 0x3fffu) << 32) |
           (1ull << 46);
}
// D[tmem] (+)= A[smem] B[smem]^T, A: 128 x 8, B: N x 8, TF32 operands, FP32 accumulator; issued by ONE thread
__device__ __forceinline__ void umma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}\n" ::"r"(d_tmem),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t *bar)  // the mbarrier completes when every MMA issued so far has
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xffffe000u); }
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&r)[8])  // 32 lanes x 8 columns, lane = thread
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr)
                 : "memory");
}

// packed FP32 pairs (Blackwell FFMA2: two fused multiply-adds per instruction, each IEEE-rounded like fmaf)
__device__ __forceinline__ unsigned long long pack2(float x, float y)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(x), "f"(y));
    return r;
}
__device__ __forceinline__ void unpack2(unsigned long long v, float &x, float &y) { asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(v)); }
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}

// complex add / subtract as one packed instruction each (IEEE per lane, same results as two scalar adds)
__device__ __forceinline__ float2 cadd2(float2 a, float2 b)
{
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pack2(a.x, a.y)), "l"(pack2(b.x, b.y)));
    float2 r;
    unpack2(d, r.x, r.y);
    return r;
}
__device__ __forceinline__ float2 csub2(float2 a, float2 b)
{
    unsigned long long d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pack2(a.x, a.y)), "l"(pack2(b.x, b.y)));
    float2 r;
    unpack2(d, r.x, r.y);
    return r;
}

// ------------------------------------------------------------------ small complex helpers
__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) { return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }  // a*conj(b)

__device__ __forceinline__ float c16(int t)  // cos(2 pi t / 16)
{
    switch (t & 15) {
        case 0: return 1.f;
        case 1: return 0.92387953251128674f;
        case 2: return 0.70710678118654752f;
        case 3: return 0.38268343236508977f;
        case 4: return 0.f;
        case 5: return -0.38268343236508977f;
        case 6: return -0.70710678118654752f;
        case 7: return -0.92387953251128674f;
        case 8: return -1.f;
        case 9: return -0.92387953251128674f;
        case 10: return -0.70710678118654752f;
        case 11: return -0.38268343236508977f;
        case 12: return 0.f;
        case 13: return 0.38268343236508977f;
        case 14: return 0.70710678118654752f;
        default: return 0.92387953251128674f;
    }
}
__device__ __forceinline__ float s16(int t) { return c16(t - 4); }  // sin(2 pi t / 16)

__host__ __device__ constexpr int ilog2c(int v) { return v <= 1 ? 0 : 1 + ilog2c(v >> 1); }
__host__ __device__ constexpr int brev(int k, int bits)
{
    int r = 0;
    for (int i = 0; i < bits; ++i) r |= ((k >> i) & 1) << (bits - 1 - i);
    return r;
}

// In-register DFT of size R (2..16) by radix-2 DIF stages; X[k] ends up in
// v[brev(k)].  INV selects exp(+i...).  Fully unrolled: all twiddles are
// compile-time constants.
template <int R, bool INV>
__device__ __forceinline__ void dft_reg(float2 (&v)[R])
{
#pragma unroll
    for (int span = R / 2; span >= 1; span >>= 1) {
#pragma unroll
        for (int i = 0; i < R; ++i) {
            if ((i & span) == 0) {
                const int j = i | span;
                const float2 a = v[i], b = v[j];
                v[i] = cadd2(a, b);
                const float2 d = csub2(a, b);
                const int t16 = (i & (span - 1)) * (8 / span);  // twiddle angle in units of 2 pi / 16
                if (t16 == 0) {
                    v[j] = d;
                } else if (t16 == 4) {
                    v[j] = INV ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x);
                } else {
                    const float c = c16(t16), s = s16(t16);
                    v[j] = INV ? make_float2(d.x * c - d.y * s, d.y * c + d.x * s)
                               : make_float2(d.x * c + d.y * s, d.y * c - d.x * s);
                }
            }
        }
    }
}

// One radix-R butterfly of an in-place FFT pass.  addr(i) -> float2* of the
// i-th element; twf(i) -> twiddle w^(i*twstep) = (cos, -sin), i = 1..R-1.
// Forward (DIF): DFT then twiddle; inverse (DIT): conj twiddle then inverse DFT.
template <int R, bool INV, bool TW, class Addr, class Twf>
__device__ __forceinline__ void fft_bfly(Addr addr, Twf twf)
{
    float2 v[R];
#pragma unroll
    for (int i = 0; i < R; ++i) v[i] = *addr(i);
    if (INV && TW) {
#pragma unroll
        for (int i = 1; i < R; ++i) v[i] = cmulc(v[i], twf(i));
    }
    dft_reg<R, INV>(v);
    constexpr int bits = ilog2c(R);
#pragma unroll
    for (int k = 0; k < R; ++k) {
        float2 o = v[brev(k, bits)];
        if (!INV && TW && k > 0) o = cmul(o, twf(k));
        *addr(k) = o;
    }
}
// The same butterfly with separate load / store functors: ld(i) -> float2 input i, st(k, value) output k.
template <int R, bool INV, bool TW, class Ld, class St, class Twf>
__device__ __forceinline__ void fft_bfly_io(Ld ld, St st, Twf twf)
{
    float2 v[R];
#pragma unroll
    for (int i = 0; i < R; ++i) v[i] = ld(i);
    if (INV && TW) {
#pragma unroll
        for (int i = 1; i < R; ++i) v[i] = cmulc(v[i], twf(i));
    }
    dft_reg<R, INV>(v);
    constexpr int bits = ilog2c(R);
#pragma unroll
    for (int k = 0; k < R; ++k) {
        float2 o = v[brev(k, bits)];
        if (!INV && TW && k > 0) o = cmul(o, twf(k));
        st(k, o);
    }
}
// twiddles from the table tw[j] = (cos, -sin)(2 pi j / NTW)
template <int R, bool INV, bool TW, int NTW, class Addr>
__device__ __forceinline__ void fft_bfly(Addr addr, int twstep, const float2 *tw)
{
    fft_bfly<R, INV, TW>(addr, [&](int i) { return tw[(i * twstep) & (NTW - 1)]; });
}

// Index into a padded scratch row of a length-N row FFT: one float2 of padding per 16, and for the long rows one more
// per 128 (N = 512) / per 256 (N = 1024).  With the first term alone the untangle / C2R accesses at the slots of
// consecutive frequencies (stride N / r0 = 64) met only 4 distinct bank groups -- 4.5 wavefronts per access at
// N = 1024 by ncu's source counters; a bank simulation of every access pattern of the row passes gives 720 -> 416
// wavefronts per row pair at N = 1024 (ideal 384) and 352 -> 272 at N = 512 (with the lane order of pass 1 below).
template <int N>
__device__ __forceinline__ int padi(int i)
{
    return i + (i >> 4) + (N == 1024 ? (i >> 8) : N == 512 ? (i >> 7) : 0);
}

// Slot holding frequency k after the forward row FFT of length N (cc_common.h: k = k1 + r0 k2 + r0 r1 k3  <->
// p = k1 N/r0 + k2 N/(r0 r1) + k3): powers of two throughout, so a few shifts instead of a table lookup.
template <int N>
__device__ __forceinline__ int row_slot_of(int k)
{
    constexpr int r0 = cc_radix_row(N, 0), r1 = cc_radix_row(N, 1);
    return (k % r0) * (N / r0) + ((k / r0) % r1) * (N / (r0 * r1)) + k / (r0 * r1);
}

// Per-lane twiddles of the warp-level row FFT of length N: a lane handles the same butterflies of every row, so
// its twiddles are loaded from the shared table once per phase and stay in registers (the inverse conjugates).
template <int N, int NTW>
struct RowTw {
    static constexpr int R0 = cc_radix_row(N, 0), R1 = cc_radix_row(N, 1), R2 = cc_radix_row(N, 2);
    static constexpr int LP = 32 / cc_row_group(N);              // lanes that share one row pair
    static constexpr int NB0 = (N / R0 + LP - 1) / LP;           // pass-0 butterflies per lane, b = g
    static constexpr int L1 = N / R0, ST1 = L1 / R1;
    static constexpr int NB1 = (N / R1 + LP - 1) / LP;
    static constexpr int S1 = ST1 <= 1 ? 0 : (ST1 <= LP ? 1 : NB1);  // pass-1 twiddle sets (b = g % ST1 repeats when ST1 | LP)
    float2 t0[NB0 * (R0 - 1)];
    float2 t1[S1 > 0 ? S1 * (R1 - 1) : 1];
    __device__ __forceinline__ void load(const float2 *tw, int lane)
    {
        const int gl = lane % LP;
#pragma unroll
        for (int n = 0; n < NB0; ++n) {
            const int b = (gl + LP * n) % (N / R0);
#pragma unroll
            for (int i = 1; i < R0; ++i) t0[n * (R0 - 1) + i - 1] = tw[(i * b * (NTW / N)) & (NTW - 1)];
        }
#pragma unroll
        for (int n = 0; n < S1; ++n) {
            const int b = (gl + LP * n) % ST1;
#pragma unroll
            for (int i = 1; i < R1; ++i) t1[n * (R1 - 1) + i - 1] = tw[(i * b * (NTW / L1)) & (NTW - 1)];
        }
    }
};

// One pass (sub-FFT length L, radix R) of a length-N FFT held by LP lanes of a warp in a padded scratch row
// (gl = lane % LP; the other lanes of the warp work on their own rows); rt = the lane's twiddles (SETS sets of
// R-1), unused when the pass has none (L == R).
template <int N, int L, int R, bool INV, int SETS, int LP>
__device__ __forceinline__ void warp_fft_pass(float2 *sc, const float2 *rt, int gl)
{
    constexpr int ST = L / R, NB = (N / R + LP - 1) / LP;
    CC_JITTER();
#pragma unroll
    for (int n = 0; n < NB; ++n) {
        int g = gl + LP * n;
        // N = 1024, pass 1 (blocks of 64, 8 lanes each): a half-warp takes blocks (0, 2) / (1, 3) instead of (0, 1) /
        // (2, 3) -- their scratch offsets differ by half the bank window, so its 16 accesses meet 32 distinct banks
        if constexpr (N == 1024 && L == 64 && LP == 32) g = (g & ~0x18) | ((g & 0x08) << 1) | ((g & 0x10) >> 1);
        if (g < N / R) {
            const int blk = g / ST, b = g % ST;
            const int base = blk * L + b;
            fft_bfly<R, INV, (ST > 1)>([&](int i) { return sc + padi<N>(base + i * ST); },
                                       [&](int i) { return rt[(SETS > 1 ? n : 0) * (R - 1) + i - 1]; });
        }
    }
    __syncwarp();
}

template <int N, bool INV, int NTW>
__device__ __forceinline__ void warp_fft(float2 *sc, const RowTw<N, NTW> &rt, int gl)
{
    using T = RowTw<N, NTW>;
    constexpr int R0 = T::R0, R1 = T::R1, R2 = T::R2, LP = T::LP;
    if (!INV) {
        warp_fft_pass<N, N, R0, false, T::NB0, LP>(sc, rt.t0, gl);
        if constexpr (R1 > 1) warp_fft_pass<N, N / R0, R1, false, T::S1, LP>(sc, rt.t1, gl);
        if constexpr (R2 > 1) warp_fft_pass<N, N / (R0 * R1), R2, false, 1, LP>(sc, rt.t1, gl);
    } else {
        if constexpr (R2 > 1) warp_fft_pass<N, N / (R0 * R1), R2, true, 1, LP>(sc, rt.t1, gl);
        if constexpr (R1 > 1) warp_fft_pass<N, N / R0, R1, true, T::S1, LP>(sc, rt.t1, gl);
        warp_fft_pass<N, N, R0, true, T::NB0, LP>(sc, rt.t0, gl);
    }
}

// Forward warp FFT whose first pass reads input x from in(x) (the decoded pixels: no staging store + reload).
template <int N, int NTW, class In>
__device__ __forceinline__ void warp_fft_fwd_from(float2 *sc, const RowTw<N, NTW> &rt, int gl, In in)
{
    using T = RowTw<N, NTW>;
    constexpr int R0 = T::R0, R1 = T::R1, R2 = T::R2, LP = T::LP, ST = N / R0;
#pragma unroll
    for (int n = 0; n < T::NB0; ++n) {
        const int g = gl + LP * n;
        if (g < ST)
            fft_bfly_io<R0, false, true>([&](int i) { return in(g + i * ST); }, [&](int k, float2 o) { sc[padi<N>(g + k * ST)] = o; },
                                         [&](int i) { return rt.t0[n * (R0 - 1) + i - 1]; });
    }
    __syncwarp();
    if constexpr (R1 > 1) warp_fft_pass<N, N / R0, R1, false, T::S1, LP>(sc, rt.t1, gl);
    if constexpr (R2 > 1) warp_fft_pass<N, N / (R0 * R1), R2, false, 1, LP>(sc, rt.t1, gl);
}
// Inverse warp FFT whose last pass hands output x to out(x, value) (streamed into the argmax: no store + reload).
template <int N, int NTW, class Out>
__device__ __forceinline__ void warp_fft_inv_to(float2 *sc, const RowTw<N, NTW> &rt, int gl, Out out)
{
    using T = RowTw<N, NTW>;
    constexpr int R0 = T::R0, R1 = T::R1, R2 = T::R2, LP = T::LP, ST = N / R0;
    if constexpr (R2 > 1) warp_fft_pass<N, N / (R0 * R1), R2, true, 1, LP>(sc, rt.t1, gl);
    if constexpr (R1 > 1) warp_fft_pass<N, N / R0, R1, true, T::S1, LP>(sc, rt.t1, gl);
#pragma unroll
    for (int n = 0; n < T::NB0; ++n) {
        const int g = gl + LP * n;
        if (g < ST)
            fft_bfly_io<R0, true, true>([&](int i) { return sc[padi<N>(g + i * ST)]; }, [&](int k, float2 o) { out(g + k * ST, o); },
                                        [&](int i) { return rt.t0[n * (R0 - 1) + i - 1]; });
    }
    __syncwarp();
}

// argmax record: larger value wins; equal values -> smaller index wins.
struct Best {
    float v;
    int i;
};
__device__ __forceinline__ bool better(float v1, int i1, float v2, int i2) { return v1 > v2 || (v1 == v2 && i1 < i2); }
// Over a warp: two hardware reductions (redux.sync) instead of five shuffle rounds -- the maximum of an order-preserving
// integer image of the value (-0 folded into +0 so that equal values have equal keys), then the smallest index among the
// lanes that hold it.
__device__ __forceinline__ Best warp_best(Best b)
{
    const uint32_t u = __float_as_uint(b.v + 0.0f);
    const uint32_t key = (u & 0x80000000u) ? ~u : (u | 0x80000000u);
    const uint32_t kmax = __reduce_max_sync(0xffffffffu, key);
    const int imin = __reduce_min_sync(0xffffffffu, key == kmax ? b.i : 0x7fffffff);
    return Best{__uint_as_float((kmax & 0x80000000u) ? (kmax & 0x7fffffffu) : ~kmax), imin};
}

// ------------------------------------------------------------------ the kernel
template <int H_, int W_, int CS_, typename PIX_, int NT_, int TM1_, int TN1_, int TM2_, int TN2_, bool SG_, int BK1_, int G2_,
          int R2_, int KS2_, int NSTG_, int PFD_, int KS1_, int TC_ = 0>
struct Cfg {
    static constexpr bool TC1 = TC_ != 0;       // stage 1 of the upsampled DFT on the tensor cores (tcgen05, 3 x TF32)
    static constexpr int NSTG = NSTG_;  // staging ring depth
    static constexpr int MINB = (H_ * W_ <= 64 * 64 && CS_ == 1) ? 2 : 1;  // CTAs per SM the register budget is set for
    static constexpr int NBARS = NSTG + 16;  // full[NSTG], raw ring [2], cluster exchange [2], rt command [1], row scatter [1], polish
                                             // tables [1], tensor-core stage 1: operand ring [4], MMA completion [2], staged [2]; T rows [1]
    static constexpr bool LAT = PFD_ > 4;       // small-batch (latency) variant: whole-frame operand prefetch, fp64 twiddles in smem
    static constexpr int H = H_, W = W_, CS = CS_, NT = NT_;
    static constexpr int TM1 = TM1_, TN1 = TN1_, TM2 = TM2_, TN2 = TN2_;
    static constexpr int BK1 = BK1_, G2 = G2_, R2 = R2_, KS2 = KS2_, KS1 = KS1_;
    static constexpr bool SG = SG_;
    using PIX = PIX_;
    static constexpr int NC = W / 2 / CS;   // spectrum columns per CTA (column 0 of rank 0 packs DC + Nyquist)
    static constexpr int NR = H / CS;       // frame rows per CTA
    static constexpr int NWARP = NT / 32;
    static constexpr int NTW = H > W ? H : W;
    static constexpr int PADW = W + W / 16 + (W == 1024 ? W / 256 : W == 512 ? W / 128 : 0);  // padi<W>(W)
    static constexpr int rch0 = 16384 / (W * (int)sizeof(PIX));
    static constexpr int RG = cc_row_group(W);  // row pairs per warp in the row FFT phases
    static constexpr int LP = 32 / RG;
    static constexpr int rch1 = rch0 > 2 * NWARP * RG ? rch0 : 2 * NWARP * RG;
    static constexpr int RCH = NR < rch1 ? NR : rch1;  // rows per raw chunk
    static constexpr int NCHK = NR / RCH;
    static constexpr int CHB = RCH * W * (int)sizeof(PIX);
    static constexpr int RAWB = (NCHK > 1 ? 2 : 1) * CHB;
    static constexpr int SCRB = NWARP * RG * PADW * 8;
    // stage 1: thread grid R1 (rows of [U|V]) x Cn1 (groups of TN1 spectrum floats) x KS1 (k-split); a warp covers
    // WR1 x WC1 threads of one k-slice
    static constexpr int Cn1 = 2 * NC / TN1;
    static constexpr int R1 = NT / (Cn1 * KS1);
    static constexpr int WC1 = Cn1 < 8 ? Cn1 : 8;
    static constexpr int WR1 = 32 / WC1;
    static constexpr int WG1C = Cn1 / WC1;
    static constexpr int MC1 = R1 * TM1;          // [U|V] columns per stage-1 chunk
    static constexpr int T1F = TC1 ? 0 : BK1 * MC1;  // floats of a stage-1 tile (TC1: stage-1 operands have their own ring)
    // stage 2: thread grid R2 x Cn2 x KS2 (k-split); a warp covers WR2 x WC2 threads of one k-slice
    static constexpr int Cn2 = NT / (R2 * KS2);
    static constexpr int WC2 = Cn2 < 8 ? Cn2 : 8;
    static constexpr int WR2 = 32 / WC2;
    static constexpr int WG2C = Cn2 / WC2;
    static constexpr int WG2R = R2 / WR2;
    static constexpr int X2 = TN2 - 4;                  // 0 or 1 extra e-column per thread
    static constexpr int GF2 = Cn2 * (16 + 4 * X2);      // floats of one group of 4 k-rows
    static constexpr int T2F = G2 * GF2;                 // floats of a stage-2 tile
    static constexpr int NCOL2 = Cn2 * TN2;              // e-columns per stage-2 chunk
    static constexpr int TILEF = T1F > T2F ? T1F : T2F;  // floats per staging slot
    static constexpr int RED2_FLOATS = (KS2 - 1) * R2 * Cn2 * 2 * TM2 * TN2;
    static constexpr int RED1_FLOATS = (KS1 - 1) * R1 * Cn1 * TM1 * TN1;
    static constexpr int RED_FLOATS = RED1_FLOATS > RED2_FLOATS ? RED1_FLOATS : RED2_FLOATS;
    static constexpr int LDT = W + 4;  // row stride (floats) of the T buffer
    static constexpr size_t S_BYTES = SG ? 0 : (size_t)H * NC * 8;
    static constexpr size_t MISC_BYTES = 8 * NBARS + 8 * (2 * CS * XN) + 16 * NWARP + 64 + 16 + 4 * NSTG + 16;
    static constexpr size_t FIXED_BYTES =
        S_BYTES + (size_t)NSTG * TILEF * 4 + (size_t)NTW * 8 + (size_t)W * 2 + MISC_BYTES + (LAT ? (size_t)W * 16 + 16 : 0);
    static_assert(NC >= 1 && NR >= 2 && (NR % 2) == 0, "bad split");
    static_assert(NR % RCH == 0 && RCH % 2 == 0 && (RCH / 2) % RG == 0 && (NR / 2) % RG == 0, "bad raw chunking");
    static_assert((2 * NC) % TN1 == 0 && NT % (Cn1 * KS1) == 0 && TN1 % 4 == 0 && Cn1 % WC1 == 0 && 32 % WC1 == 0, "bad stage-1 tiling");
    static_assert(R1 % 4 == 0 && R1 % WR1 == 0 && (R1 / WR1) * WG1C * KS1 == NWARP && BK1 % KS1 == 0, "bad stage-1 warp grid");
    static_assert(TM1 == 1 || TM1 == 2 || TM1 == 3 || TM1 == 4 || TM1 == 5 || TM1 == 8 || TM1 == 10, "TM1 chunking");
    static_assert(R2 * Cn2 * KS2 == NT && Cn2 % WC2 == 0 && 32 % WC2 == 0 && R2 % WR2 == 0, "bad stage-2 tiling");
    static_assert(WG2R * WG2C * KS2 == NWARP && (TN2 == 4 || TN2 == 5) && G2 % KS2 == 0 && W % (4 * G2) == 0, "bad stage-2 tiling");
    static_assert(TILEF % 4 == 0 && MC1 % 4 == 0, "tile alignment");
    static_assert(NT % NC == 0 || NC % NT == 0, "threads vs columns");
    static_assert(NSTG <= 8, "ring (sched_head carries 8 entries)");
    static_assert(!TC1 || (2 * NC == 128 && NT == 256), "tensor-core stage 1: 128 spectrum floats per CTA (MMA N = 128), 8 warps");
};

template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB) cc_fused_kernel(const CcParams p)
{
    constexpr int H = C::H, W = C::W, CS = C::CS, NT = C::NT, NC = C::NC, NR = C::NR;
    constexpr int NWARP = C::NWARP, NTW = C::NTW, PADW = C::PADW;
    constexpr int LDT = C::LDT;
    constexpr bool SG = C::SG;
    constexpr int NSTG = C::NSTG, NBARS = C::NBARS;
    using PIX = typename C::PIX;

    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long t_entry = clock64();
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (CS > 1) ? (int)cluster.block_rank() : 0;
    const int cid = blockIdx.x / CS, ncl = gridDim.x / CS;
    constexpr int RG = C::RG, LP = C::LP;
    const int gl = lane % LP, gp = lane / LP;  // lane within its row pair, row pair within the warp

    // ---- loads whose latency the whole setup hides: the plan's twiddle tables (all variants) and, in the latency
    // variants whose CTA slice is one raw chunk, the pixels of the first frame straight into registers (a plain
    // coalesced load arrives in about a third of the time of a TMA copy + mbarrier round trip)
    constexpr int NI_TW = (C::NTW + NT - 1) / NT, NI_W = (W + NT - 1) / NT;
    float2 r_tw[NI_TW];
    double2 r_64[C::LAT ? NI_W : 1];
#pragma unroll
    for (int e = 0; e < NI_TW; ++e)
        if (tid + e * NT < C::NTW) r_tw[e] = __ldg(&p.tw[tid + e * NT]);
    if constexpr (C::LAT) {
#pragma unroll
        for (int e = 0; e < NI_W; ++e)
            if (tid + e * NT < W) r_64[e] = __ldg(&p.tw64[tid + e * NT]);
    }
    constexpr bool DIRECT = C::LAT && C::NCHK == 1 && (C::RCH / 2) <= C::NWARP * RG;
    constexpr int NPX = W / LP;  // pixels per row per lane in the decode
    PIX pxa[DIRECT ? NPX : 1], pxb[DIRECT ? NPX : 1];
    bool direct_first = false;   // the first frame's pixels ride in registers instead of the raw ring
    if constexpr (DIRECT) {
        direct_first = !p.rt_cmd && cid < p.batch;
        const int jp = warp * RG + gp;
        if (direct_first && jp < C::RCH / 2) {
            const PIX *fb = reinterpret_cast<const PIX *>(p.frames) + (size_t)cid * H * W + (size_t)rank * C::NR * W;
            const PIX *ga = fb + (size_t)jp * W, *gb = fb + (size_t)(jp + C::RCH / 2) * W;
#pragma unroll
            for (int i = 0; i < NPX; ++i) pxa[i] = __ldg(ga + gl + i * LP), pxb[i] = __ldg(gb + gl + i * LP);
        }
    }

    // ---- shared memory carve-up
    float2 *const Ssm = reinterpret_cast<float2 *>(smem);
    float *const stg = reinterpret_cast<float *>(smem + C::S_BYTES);        // [NSTG][TILEF] operand ring
    unsigned char *const U = reinterpret_cast<unsigned char *>(stg + NSTG * C::TILEF);
    float2 *const tw = reinterpret_cast<float2 *>(U + p.u_bytes);
    uint16_t *const rslot = reinterpret_cast<uint16_t *>(tw + NTW);
    unsigned char *misc = reinterpret_cast<unsigned char *>(rslot + W);
    misc = reinterpret_cast<unsigned char *>(((uintptr_t)misc + 15) & ~(uintptr_t)15);
    uint64_t *const bars = reinterpret_cast<uint64_t *>(misc);         // full[NSTG], empty[NSTG], raw ring [2]
    uint64_t *const bfull = bars, *const braw = bars + NSTG, *const xbar = braw + 2, *const cbar = xbar + 2;
    uint64_t *const sbar = cbar + 1, *const pbar = sbar + 1;   // sbar: the peers' rows of the row-FFT scatter have landed
    uint64_t *const ebar = pbar + 1, *const mdone = ebar + 4, *const afull = mdone + 2;  // tensor-core stage 1: operand ring,
                                                                                         // MMA completion, operands staged
    uint64_t *const trow = afull + 2;                          // the peers' rows of T (stage-1 output) have landed
    double *const xchg = reinterpret_cast<double *>(bars + NBARS);     // [2][CS][XN]
    float *const wv = reinterpret_cast<float *>(xchg + 2 * CS * XN);    // [NWARP]
    int *const wi = reinterpret_cast<int *>(wv + NWARP);               // [NWARP]
    float *const f00 = reinterpret_cast<float *>(wi + NWARP);          // [1]
    uint64_t *const cmdslot = reinterpret_cast<uint64_t *>(((uintptr_t)(f00 + 1) + 7) & ~(uintptr_t)7);  // [2] rt command (seq, frame)
    uint32_t *const relcnt = reinterpret_cast<uint32_t *>(cmdslot + 2);  // [NSTG] releases of each ring slot (mod NWARP)
    uint32_t *const tmem_slot = relcnt + NSTG;                           // [1] base address of the tensor-memory allocation

    float2 *const scr = reinterpret_cast<float2 *>(U + C::RAWB) + (warp * RG + gp) * PADW;
    float *const Tb = reinterpret_cast<float *>(U);

    // local spectrum block S[y][ql], y in [0,H), ql in [0,NC)
    float2 *const Sl = SG ? p.Sg + ((size_t)cid * CS + rank) * ((size_t)H * NC) : Ssm;
    auto Sof = [&](int r) -> float2 * {
        if constexpr (SG) return p.Sg + ((size_t)cid * CS + r) * ((size_t)H * NC);
        if constexpr (CS > 1) return cluster.map_shared_rank(Ssm, r);
        return Ssm;
    };
    // Cluster barriers.  csync(): release / acquire at cluster scope -- a MEMBAR.ALL.GPU per warp, measured at 430
    // cycles with nothing outstanding, 1000 after global stores and 1300-2000 after remote shared-memory stores (the
    // fence waits for their acknowledgements).  It is kept where GLOBAL data crosses CTAs (the L2-resident spectrum of
    // the SG variants).  Remote shared-memory data travels by st.async instead: the bytes complete on an mbarrier of the
    // receiving CTA (sbar, trow, the exchange barriers), one-way latency and no fence.  What is left is control:
    // csync_ctl() = CTA barrier (this CTA's shared-memory accesses are performed) + relaxed arrive + wait, 120 cycles:
    // "my peers may now read what I wrote into MY shared memory" / "I no longer touch the region you are about to fill".
    auto csync = [&]() {
        CC_JITTER();
        if constexpr (CS > 1) cluster.sync();
        else __syncthreads();
    };
    auto csync_ctl = [&]() {
        CC_JITTER();
        __syncthreads();
        if constexpr (CS > 1) asm volatile("barrier.cluster.arrive.relaxed.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    };

    PIX *const raw = reinterpret_cast<PIX *>(U);
    // raw-pixel ring: the first (up to two) chunks of frame f and an L2 prefetch of the cluster's next frame
    auto issue_raw_head = [&](const void *frames, int f) {  // thread 0 only
        const PIX *fbase = reinterpret_cast<const PIX *>(frames) + (size_t)f * H * W + (size_t)rank * NR * W;
        fence_proxy_async();
        for (int ck = 0; ck < (C::NCHK > 1 ? 2 : 1); ++ck) {
            mbar_expect_tx(&braw[ck], C::CHB);
            bulk_g2s(raw + (size_t)ck * C::RCH * W, fbase + (size_t)ck * C::RCH * W, C::CHB, &braw[ck]);
        }
        if (f + ncl < p.batch) {  // pull the next frame of this cluster into L2
            const PIX *nb = fbase + (size_t)ncl * H * W;
            constexpr uint32_t tot = (uint32_t)NR * W * sizeof(PIX);
            for (uint32_t o = 0; o < tot; o += 32768u)
                bulk_prefetch_l2(reinterpret_cast<const unsigned char *>(nb) + o, tot - o < 32768u ? tot - o : 32768u);
        }
    };

    // ---- operand ring: every frame consumes the same p.ntiles_frame tiles of p.blob in the order of
    // p.sched; the NSTG slots always hold the next NSTG tiles (landed or in flight), also across frames and
    // phases.  A slot is refilled, with the tile NSTG positions ahead, by whichever warp is the LAST to release
    // it (shared-memory release counter): the copy is issued at the first moment the slot is free, whatever the
    // relative progress of the warps -- no dedicated producer, no CTA barrier inside the GEMM loops.
    const uint32_t my_frames = p.batch > cid ? (uint32_t)((p.batch - cid + ncl - 1) / ncl) : 0u;
    // real-time session: frames arrive one by one for as long as the session lives; the ring runs ahead freely
    const uint32_t total_tiles = p.rt_cmd ? (p.ntiles_frame ? 0xffffffffu : 0u) : my_frames * (uint32_t)p.ntiles_frame;
    uint32_t g_cons = 0;                       // tiles consumed so far (saturating in a session)
    uint32_t c_slot = 0, c_par = 0;            // current ring slot and the parity of its full barrier
    uint32_t r_idx = (uint32_t)(p.ntiles_frame > 0 ? NSTG % p.ntiles_frame : 0);  // schedule position of tile g_cons + NSTG
    uint32_t refill_ti = 0u;                   // its blob index, fetched at acquire time (lane 0)
    auto ring_acquire = [&]() -> const float * {
        if (lane == 0) refill_ti = __ldg(&p.sched[r_idx]);  // latency overlaps the tile's compute
        mbar_wait(&bfull[c_slot], c_par);
        return stg + (size_t)c_slot * C::TILEF;
    };
    auto ring_release = [&]() {
        CC_JITTER();
        __syncwarp();
        if (lane == 0) {
            // (every value the warp loaded from the slot has been consumed by an FMA above, so the loads have completed;
            //  a __threadfence_block() here also waited for the refill_ti load in flight: 5-8 % of the GEMM phases)
            const uint32_t old = atomicAdd(&relcnt[c_slot], 1u);
            if ((old + 1u) % (uint32_t)NWARP == 0u && (total_tiles == 0xffffffffu || g_cons + (uint32_t)NSTG < total_tiles)) {
                fence_proxy_async();  // generic-proxy reads of the slot before the async-proxy write
                mbar_expect_tx(&bfull[c_slot], (uint32_t)C::TILEF * 4u);
                bulk_g2s(stg + (size_t)c_slot * C::TILEF, p.blob + (size_t)refill_ti * C::TILEF, (uint32_t)C::TILEF * 4u,
                         &bfull[c_slot]);
            }
        }
        if (g_cons != 0xffffffffu) ++g_cons;
        if (++c_slot == NSTG) c_slot = 0, c_par ^= 1u;
        if (++r_idx == (uint32_t)p.ntiles_frame) r_idx = 0;
    };

    // ---- one-time setup.  Thread 0 initialises the mbarriers and at once puts in flight (TMA bulk copies) the plan
    // tables (FFT twiddles, slot table; fp64 twiddles and -- where they fit -- the fp64 polish tables of the latency
    // variants), the first NSTG operand tiles and the first frame's raw rows.  The cluster barrier that makes the
    // mbarriers of all CTAs visible is split: arrive here, wait just before the first remote access (after the first
    // raw chunk has landed), so neither the table latency nor the barrier latency is exposed.
    const double2 *tw64 = p.tw64;  // (cos, sin)(2 pi j / W) in fp64; the latency variants keep a copy in shared memory
    double2 *const t64s = reinterpret_cast<double2 *>(((uintptr_t)(relcnt + NSTG + 4) + 15) & ~(uintptr_t)15);   // [W] (LAT)
    // resident polish tables (p.pol_smem): Dpol [M][H], this CTA's columns of Xpol [M][NC], nyq64 [M rounded up to even]
    double *const DpolS = reinterpret_cast<double *>(t64s + (C::LAT ? W : 0));
    double2 *const XpolS = reinterpret_cast<double2 *>(DpolS + (size_t)p.M * H);
    double *const nyqS = reinterpret_cast<double *>(XpolS + (size_t)p.M * NC);
    const bool POLS = C::LAT && p.pol_smem != 0;
    static_assert(NBARS <= 32, "one lane of warp 0 per mbarrier");
    if (tid < NBARS) {  // one barrier per lane (a single thread took 900 cycles over them); thread 0 also the raw ring's
        uint64_t *const b = bars + tid;
        const bool is_raw = b == &braw[0] || b == &braw[1];
        // counts: the two MMA-issuing threads commit to mdone[]; the four staging warps arrive on afull[]; else 1
        const uint32_t cnt = (b == &mdone[0] || b == &mdone[1]) ? 2u : (b == &afull[0] || b == &afull[1]) ? 128u : 1u;
        if (!is_raw) mbar_init(b, cnt);
        if (tid < NSTG) relcnt[tid] = 0u;
        if (tid == 0) mbar_init(&braw[0], 1), mbar_init(&braw[1], 1);
        fence_mbar_init();
        if (tid == 0 && !p.rt_cmd && cid < p.batch && !direct_first) issue_raw_head(p.frames, cid);
    }
#pragma unroll
    for (int e = 0; e < NI_TW; ++e)
        if (tid + e * NT < NTW) tw[tid + e * NT] = r_tw[e];
    if constexpr (C::LAT) {
#pragma unroll
        for (int e = 0; e < NI_W; ++e)
            if (tid + e * NT < W) t64s[tid + e * NT] = r_64[e];
    }
    if constexpr (C::LAT) tw64 = t64s;
    if constexpr (C::TC1) {  // all 512 columns of tensor memory (one CTA per SM): accumulators U and V of stage 1
        if (warp == 1) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    }
    __syncthreads();  // the mbarrier inits are visible to every thread of the CTA
    uint32_t tmem = 0, mph[2] = {0u, 0u}, aph[2] = {0u, 0u}, e_issued = 0u, e_cons = 0u;  // TC1: tensor-memory base, completed waits on mdone[],
                                                                        // stage-1 operand tiles requested / consumed (thread 0)
    if constexpr (C::TC1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        tmem = *tmem_slot;
    }
    // the copies nobody waits for yet are issued by other warps, beside the first phase: the operand ring ...
    if (tid == 32 && total_tiles > 0) {  // the first schedule entries ride in the kernel parameters: no load latency
#pragma unroll
        for (int i = 0; i < NSTG; ++i)
            if ((uint32_t)i < total_tiles) {
                mbar_expect_tx(&bfull[i], (uint32_t)C::TILEF * 4u);
                bulk_g2s(stg + (size_t)i * C::TILEF, p.blob + (size_t)p.sched_head[i] * C::TILEF, (uint32_t)C::TILEF * 4u, &bfull[i]);
            }
    }
    // ... and the resident fp64 polish tables (Dpol, this CTA's slice of the rank-major copy of Xpol, nyq64)
    if (tid == 64 && POLS) {
        const uint32_t db = (uint32_t)p.M * H * 8u, xb = (uint32_t)p.M * NC * 16u, nb = (uint32_t)((p.M + 1) & ~1) * 8u;
        mbar_expect_tx(pbar, db + xb + nb);
        for (uint32_t o = 0; o < db; o += 32768u)
            bulk_g2s(reinterpret_cast<unsigned char *>(DpolS) + o, reinterpret_cast<const unsigned char *>(p.Dpol) + o,
                     db - o < 32768u ? db - o : 32768u, pbar);
        bulk_g2s(XpolS, p.XpolR + (size_t)rank * p.M * NC, xb, pbar);
        bulk_g2s(nyqS, p.nyq64, nb, pbar);
    }
    bool csync_pending = false;  // the cluster half of the setup barrier: arrive now, wait before the first remote access
    if constexpr (CS > 1) {
        // relaxed: what the peers need (the mbarrier inits) was published by fence.mbarrier_init.release.cluster
        asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");
        csync_pending = true;
    }
    auto setup_cluster_wait = [&]() {
        if constexpr (CS > 1) {
            if (csync_pending) {
                asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
                csync_pending = false;
            }
        }
    };
    bool pol_pending = POLS;
    uint32_t sph = 0u, tph1 = 0u;  // phase parities of sbar and trow
    uint32_t ph = 0;   // phase parity bits of the raw ring
    int xpar = 0;      // exchange buffer parity
    uint32_t xph = 0;  // phase parity bits of the two exchange barriers

    const int u = p.u, M = p.M, cM = p.c;
    const double c0d = p.sn ? p.sn_c0 : (double)p.c0;  // constant subtracted from every (transformed) pixel

    // Cluster-wide exchanges: every CTA stores its record into every peer with st.async, which completes
    // tx-bytes on the PEER's mbarrier: a one-way DSMEM latency instead of remote stores + a full cluster barrier.
    // Two buffers/barriers alternate; a CTA cannot run two exchanges ahead of a peer because each exchange needs
    // that peer's record.
    // one exchange round: arm the barrier of buffer xpar (thread 0), wait for every rank's record, flip
    auto xchg_arm = [&](int bytes_per_rank) {
        if constexpr (CS > 1) mbar_expect_tx(&xbar[xpar], (uint32_t)(CS * bytes_per_rank));
    };
    auto xchg_send = [&](int k, uint64_t bits, int r) {  // my record word k -> rank r
        CC_JITTER();
        if constexpr (CS > 1) {
            const uint32_t dst = mapa_u32(smem_u32(xchg + ((size_t)xpar * CS + rank) * XN + k), (uint32_t)r);
            st_async_b64(dst, bits, mapa_u32(smem_u32(&xbar[xpar]), (uint32_t)r));
        } else {
            reinterpret_cast<uint64_t *>(xchg)[(size_t)xpar * XN + k] = bits;
        }
    };
    auto xchg_wait = [&]() -> const double * {
        const double *res = xchg + (size_t)xpar * CS * XN;
        if constexpr (CS > 1) {
            mbar_wait(&xbar[xpar], (xph >> xpar) & 1u);
            xph ^= 1u << xpar;
        } else {
            __syncthreads();
        }
        xpar ^= 1;
        return res;
    };
    // cluster-wide argmax: warp shuffles -> warp 0 over the warp records -> one 8-byte record (value, index) per
    // rank to every peer.  The same (larger value, then smaller index) rule at every level; result in all threads.
    auto cluster_best = [&](Best b) -> Best {
        b = warp_best(b);
        if (lane == 0) {
            wv[warp] = b.v;
            wi[warp] = b.i;
        }
        __syncthreads();  // also: all reads of the exchange buffer used two rounds ago are done
        if (warp == 0) {
            Best c{-INFINITY, 0x7fffffff};
            if (lane < NWARP) c.v = wv[lane], c.i = wi[lane];
            c = warp_best(c);
            if (lane == 0) xchg_arm(8);
            if (lane < CS) xchg_send(0, (uint64_t)__float_as_uint(c.v) | ((uint64_t)(uint32_t)c.i << 32), lane);
        }
        const uint64_t *res = reinterpret_cast<const uint64_t *>(xchg_wait());
        Best g{-INFINITY, 0x7fffffff};
#pragma unroll
        for (int r = 0; r < CS; ++r) {
            const uint64_t w = res[r * XN];
            const float v = __uint_as_float((uint32_t)w);
            const int i = (int)(uint32_t)(w >> 32);
            if (better(v, i, g.v, g.i)) g.v = v, g.i = i;
        }
        return g;
    };

    auto bar_wait = [&](int b) {  // raw ring barriers
        mbar_wait(&braw[b], (ph >> b) & 1u);
        ph ^= 1u << b;
    };

    // 3x3 evaluation in fp64 of  sum_q w_q Re( R[a][q] * (cs + i sn)(b, q) )  over this CTA's columns,
    // summed over the cluster in rank order.  Eight lanes (sub = 0..7) serve each (a, ql): getR(a, ql, sub)
    // returns R[a][ql] to all of them (it may shuffle inside the 8-lane group); lanes sub = b < 3 then form the
    // term of column phase b.  The packed column (rank 0, ql 0) holds (dc, nyq) and uses nyq_c[b].
    // phase(b, q) -> (cos, sin) of the column phase from the plan's fp64 tables.  Scratch `terms` =
    // double[9][NC].  Result: lane k < 9 of every warp of every CTA returns the value of candidate k = a*3+b (other
    // lanes: 0).  Summation order is fixed.
    auto xeval9 = [&](auto getR, auto phase, const double *nyq_c, double *terms) -> double {
        static_assert((24 * NC) % 32 == 0, "whole warps per (a, ql) group sweep");
        constexpr int XIT = (24 * NC + NT - 1) / NT;
#pragma unroll
        for (int it = 0; it < XIT; ++it) {  // unrolled: the table loads of all trips go out together
            const int t = tid + it * NT;
            if (t >= 24 * NC) break;       // warp-uniform (24 NC and NT are multiples of 32)
            const int o = t >> 3, sub = t & 7;
            const int a = o / NC, ql = o % NC;
            const int q = rank * NC + ql;
            double2 cs = make_double2(1.0, 0.0);
            if (sub < 3 && q != 0) cs = phase(sub, q);  // issued before the group sum: the latency overlaps
            const double2 r = getR(a, ql, sub);
            if (sub < 3) {
                double v;
                if (q == 0) v = r.x + r.y * (sub == 0 ? nyq_c[0] : sub == 1 ? nyq_c[1] : nyq_c[2]);
                else v = 2.0 * (r.x * cs.x - r.y * cs.y);
                terms[(a * 3 + sub) * NC + ql] = v;
            }
        }
        __syncthreads();  // terms complete; all reads of the exchange buffer used two rounds ago are done
        if (tid == 0) xchg_arm(72);
        if (tid < 96) {  // three whole warps: 8 lanes per output k = a*3+b (k >= 9: idle groups)
            const int k = tid >> 3, sub = tid & 7;
            double sum = 0.0;
            if (k < 9)
                for (int ql = sub; ql < NC; ql += 8) sum += terms[k * NC + ql];
            sum += __shfl_xor_sync(0xffffffffu, sum, 1);
            sum += __shfl_xor_sync(0xffffffffu, sum, 2);
            sum += __shfl_xor_sync(0xffffffffu, sum, 4);
            if (k < 9 && sub < CS) {  // lane sub sends this CTA's k-th sum to rank sub (CS <= 8)
                for (int r = sub; r < CS; r += 8) xchg_send(k, (uint64_t)__double_as_longlong(sum), r);
            }
        }
        const double *res = xchg_wait();
        double mine = 0.0;  // lane k < 9 of every warp: sum over the ranks, in rank order
        if (lane < 9)
            for (int r = 0; r < CS; ++r) mine += res[r * XN + lane];
        return mine;
    };
    // The decision over the nine candidates: lane k < 9 holds (value, index, valid); larger value wins, then the smaller
    // index -- a 16-lane butterfly instead of nine broadcasts and a nine-way compare chain (this code runs once per
    // launch in the single-frame variants, from a cold instruction cache: its size is its cost).  All lanes return the
    // winner's value and candidate number.
    auto best9 = [&](double v, int idx, bool valid, double &bv, int &bk) {
        if (!valid || lane >= 9) v = -INFINITY, idx = 0x7fffffff;
        int k = lane;
#pragma unroll
        for (int o = 8; o >= 1; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, v, o);
            const int oi = __shfl_xor_sync(0xffffffffu, idx, o), ok = __shfl_xor_sync(0xffffffffu, k, o);
            if (ov > v || (ov == v && oi < idx)) v = ov, idx = oi, k = ok;
        }
        bv = __shfl_sync(0xffffffffu, v, 0);
        bk = __shfl_sync(0xffffffffu, k, 0);
    };

    long long tph = t_entry;  // the first frame's phase 0 includes the kernel setup
    auto stamp = [&](int k, int f) {  // optional per-phase cycle counts (rank 0, thread 0)
        if (p.phase_clk && rank == 0 && tid == 0) {
            const long long now = clock64();
            p.phase_clk[(size_t)f * CC_NPHASE + k] = (unsigned long long)(now - tph);
            tph = now;
        }
    };

    // results of one frame (rank 0, thread 0): batch arrays, or the session's mapped host record
    const bool RT = p.rt_cmd != nullptr;
    const bool ACC = p.acc_G != nullptr;              // offline iteration, Eq. (8): accumulate the aligned spectra
    const bool RI = p.ri_Fs != nullptr;               // the frame's spectrum is kept: Eq. (9) update, or Eq. (8) accumulation
    // this cluster's copy of the frame spectrum (computed at the use sites: no registers held through the GEMM phases)
    auto Fs_of = [&]() { return p.ri_Fs + (size_t)cid * H * (W / 2); };
    auto Fab_of = [&]() { return p.ri_Fab + (size_t)cid * H; };
    uint64_t rt_seq = 0;    // sequence number of the command being served
    uint32_t cph = 0;       // phase parity of the command barrier
    auto emit = [&](int f, float dyv, float dxv, float pkv, int wyv, int wxv) {
        if (__builtin_expect(!RT, true)) {
            p.dy[f] = dyv;
            p.dx[f] = dxv;
            if (p.peak) p.peak[f] = pkv;
            if (p.iy) p.iy[f] = wyv;
            if (p.ix) p.ix[f] = wxv;
        } else {  // one 16-byte store; the sequence number is the last word
            asm volatile("st.volatile.global.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p.rt_res), "f"(dxv), "f"(dyv), "f"(pkv),
                         "f"(__uint_as_float((uint32_t)rt_seq))
                         : "memory");
            __threadfence_system();
        }
    };

    // ---- running reference image, Eq. (9): F[E_i] = a0 F[I_i(r + d_i)] + b1 F[E_{i-1}] (R18).  d = (ny, nx) / u.
    // In the plan's storage (conj(G)/(HW), column-slot order): Gt <- b1 Gt + (a0/HW) conj(F exp(i theta)),
    // theta = 2 pi (fy ny / (u H) + kx nx / (u W)); cos(pi d) replaces the phase factor on the Nyquist row / column.
    // Every CTA rewrites exactly the columns it reads in the product, so no cluster barrier is involved.
    auto ri_update = [&](long long ny, long long nx) {
        const double a0 = p.ri_a0, b1 = 1.0 - a0;
        const float b1f = (float)b1, scf = (float)(a0 / ((double)H * (double)W));
        const double cnx = cospi((double)(((nx % (2LL * u)) + 2LL * u) % (2LL * u)) / (double)u);  // cos(pi dx)
        const double cny = cospi((double)(((ny % (2LL * u)) + 2LL * u) % (2LL * u)) / (double)u);  // cos(pi dy)
        // exp(i theta) = wy(slot) * wx(kx): H + W/2 phase factors per frame (exactly reduced phase numerators, fp64
        // sincospi, rounded once) in the free U region instead of one evaluation per spectrum element
        float2 *const wyt = reinterpret_cast<float2 *>(U), *const wxt = wyt + H;
        for (int i = tid; i < H + W / 2; i += NT) {
            double sn, cs;
            if (i < H) {
                const int fy = (int)p.col_freq[i];
                if (2 * fy == -H) {  // Nyquist row: the real interpolant multiplies by cos(pi dy)
                    cs = cny, sn = 0.0;
                } else {
                    const long long dy_den = (long long)u * H;
                    long long num = ((long long)fy * ny) % dy_den;
                    if (num < 0) num += dy_den;
                    sincospi(2.0 * (double)num / (double)dy_den, &sn, &cs);
                }
                wyt[i] = make_float2((float)cs, (float)sn);
            } else {
                const long long dx_den = (long long)u * W;
                long long num = ((long long)(i - H) * nx) % dx_den;
                if (num < 0) num += dx_den;
                sincospi(2.0 * (double)num / (double)dx_den, &sn, &cs);
                wxt[i - H] = make_float2((float)cs, (float)sn);
            }
        }
        __syncthreads();
        for (int idx = tid; idx < H * NC; idx += NT) {
            const int ps = idx / NC, q = rank * NC + idx % NC;
            if (q == 0) continue;
            const size_t gi = (size_t)ps * (W / 2) + q;
            const float2 Fp = cmul(__ldcg(&Fs_of()[gi]), cmul(wyt[ps], wxt[q]));
            if (ACC) {  // Eq. (8): this cluster's running sum of the aligned spectra
                float2 *a = p.acc_G + (size_t)cid * H * (W / 2) + gi;
                const float2 av = __ldcg(a);
                __stcg(a, make_float2(av.x + Fp.x, av.y + Fp.y));
            } else {
                const float2 Gv = __ldcg(&p.Gt[gi]);
                __stcg(const_cast<float2 *>(&p.Gt[gi]), make_float2(fmaf(b1f, Gv.x, scf * Fp.x), fmaf(b1f, Gv.y, -scf * Fp.y)));
            }
        }
        if (rank == 0) {
            for (int ps = tid; ps < H; ps += NT) {
                const int fy = (int)p.col_freq[ps];
                const float4 Fv = __ldcg(&Fab_of()[ps]);
                const float2 wy = wyt[ps];
                const float2 Fa = cmul(make_float2(Fv.x, Fv.y), wy);
                const float2 Fb = cmul(make_float2(Fv.z, Fv.w), make_float2(wy.x * (float)cnx, wy.y * (float)cnx));
                if (ACC) {
                    float4 *a = p.acc_ab + (size_t)cid * H + ps;
                    const float4 av = __ldcg(a);
                    __stcg(a, make_float4(av.x + Fa.x, av.y + Fa.y, av.z + Fb.x, av.w + Fb.y));
                    continue;
                }
                const float4 Gv = __ldcg(&p.ab[ps]);
                float4 o;
                o.x = fy == 0 ? 0.f : fmaf(b1f, Gv.x, scf * Fa.x);  // the DC bin of the reference stays zero (R10)
                o.y = fy == 0 ? 0.f : fmaf(b1f, Gv.y, -scf * Fa.y);
                o.z = fmaf(b1f, Gv.z, scf * Fb.x);
                o.w = fmaf(b1f, Gv.w, -scf * Fb.y);
                __stcg(const_cast<float4 *>(&p.ab[ps]), o);
            }
            if (tid == 0) {
                const double mean_i = ((double)*f00 + c0d * H * W) / ((double)H * (double)W);
                if (ACC) __stcg(p.acc_mean + cid, __ldcg(p.acc_mean + cid) + mean_i);
                else __stcg(p.ri_emean, b1 * __ldcg(p.ri_emean) + a0 * mean_i);
            }
        }
        __threadfence();
    };

    constexpr int RLc = cc_radix_col(H, 2) > 1 ? cc_radix_col(H, 2) : cc_radix_col(H, 1);  // radix of the fused column pass
    constexpr bool GPRE = C::LAT && NC * (H / RLc) <= NT;
    float2 gpre[GPRE ? RLc : 1];
    for (int f = cid; RT || f < p.batch; f += ncl) {
        const void *frames = p.frames;
        if (__builtin_expect(RT, false)) {
            // ---- real-time session (one displacement per camera frame, as it arrives): rank 0
            // polls the host's command word; (seq, frame pointer) go to every CTA of the cluster by st.async
            f = 0;
            setup_cluster_wait();  // the peers' command barriers exist
            if constexpr (CS > 1) {
                if (tid == 0) mbar_expect_tx(cbar, 16u);
            }
            if (rank == 0 && tid == 0) {
                const uint64_t t0 = globaltimer_ns();
                uint64_t seq, ptr = 0;
                for (;;) {
                    // one 16-byte read over PCIe: (seq, frame pointer | low 4 bits of seq); the tag in the pointer's
                    // low bits (frames are 16-byte aligned) exposes a read torn between two commands
                    ld_sys_v2u64(p.rt_cmd, seq, ptr);
                    if (seq == ~0ull) break;
                    if (seq == rt_seq + 1 && (ptr & 15ull) == (seq & 15ull)) break;
                    if (globaltimer_ns() - t0 > p.rt_timeout_ns) {  // idle for too long: end the session kernel
                        seq = ~0ull;
                        break;
                    }
                }
                ptr &= ~15ull;
#pragma unroll
                for (int r = 0; r < CS; ++r) {
                    if constexpr (CS > 1) {
                        const uint32_t rb = mapa_u32(smem_u32(cbar), (uint32_t)r);
                        st_async_b64(mapa_u32(smem_u32(&cmdslot[0]), (uint32_t)r), seq, rb);
                        st_async_b64(mapa_u32(smem_u32(&cmdslot[1]), (uint32_t)r), ptr, rb);
                    } else {
                        cmdslot[0] = seq, cmdslot[1] = ptr;
                    }
                }
            }
            if constexpr (CS > 1) {
                mbar_wait(cbar, cph);
                cph ^= 1u;
            } else {
                __syncthreads();
            }
            const uint64_t seq = cmdslot[0];
            if (seq == ~0ull) break;
            rt_seq = seq;
            frames = reinterpret_cast<const void *>(cmdslot[1]);
            if (tid == 0) issue_raw_head(frames, 0);
        }
        if (p.phase_clk && rank == 0 && tid == 0 && (RT || f != cid)) tph = clock64();  // first frame: phase 0 includes the setup
        // =============================================================== a1 + a2: ingest and row FFTs
        {
            const PIX *fbase = reinterpret_cast<const PIX *>(frames) + (size_t)f * H * W + (size_t)rank * NR * W;
            if (tid == 0 && !RT && f != cid) issue_raw_head(frames, f);  // the first frame's rows were requested during the setup
            if constexpr (!SG && CS > 1) {  // the other CTAs' rows of my columns arrive by st.async
                if (tid == 0) mbar_expect_tx(sbar, (uint32_t)((CS - 1) * NR * NC * 8));
            }
            // latency variants: every thread owns at most one butterfly of the fused column pass; its RL values of
            // conj(G)/(HW) are requested now (L2 latency hidden behind the ingest and the row FFTs)
            if constexpr (GPRE) {
                if (tid < NC * (H / RLc)) {
                    const int ql = tid % NC, g = tid / NC, q = rank * NC + ql;
                    if (q != 0) {
#pragma unroll
                        for (int k = 0; k < RLc; ++k) gpre[k] = __ldcg(&p.Gt[(size_t)(g * RLc + k) * (W / 2) + q]);
                    }
                }
            }
            RowTw<W, NTW> rtw;
            rtw.load(tw, lane);
            const float c0f = (float)p.c0;
            const bool from_regs = DIRECT && direct_first && f == cid;  // first frame of a latency variant
            for (int ck = 0; ck < C::NCHK; ++ck) {
                const int rb = ck & 1;
                if (!from_regs) bar_wait(rb);
                setup_cluster_wait();  // first frame: every CTA of the cluster is set up (remote stores follow)
                const PIX *rw = raw + (size_t)rb * C::RCH * W;
                for (int jp0 = warp * RG; jp0 < C::RCH / 2; jp0 += NWARP * RG) {
                    const int jp = jp0 + gp;
                    const PIX *ra = rw + (size_t)jp * W;
                    const PIX *rbp = rw + (size_t)(jp + C::RCH / 2) * W;
                    // decode fused into the first FFT pass: pixel x of the two rows is input x of the complex row FFT
                    warp_fft_fwd_from<W, NTW>(scr, rtw, gl, [&](int x) {
                        PIX va, vb;
                        if constexpr (DIRECT) {
                            const int i = (x - gl) / LP;  // compile-time after unrolling
                            va = from_regs ? pxa[i] : ra[x], vb = from_regs ? pxb[i] : rbp[x];
                        } else {
                            va = ra[x], vb = rbp[x];
                        }
                        if (p.sn) {  // CC-SN: I'^2 - c0 with I' = I + eps (Eq. (7)), one rounding
                            const double ta = (double)va + p.sn_eps, tb = (double)vb + p.sn_eps;
                            return make_float2((float)fma(ta, ta, -p.sn_c0), (float)fma(tb, tb, -p.sn_c0));
                        }
                        return make_float2((float)va - c0f, (float)vb - c0f);
                    });
                    // untangle the two real rows and scatter to the column owners
                    const int ya = rank * NR + ck * C::RCH + jp, yb = ya + C::RCH / 2;
                    {
                        constexpr int NK = (W / 2) / LP;  // spectrum columns per lane
                        float2 z1[NK], z2[NK];
#pragma unroll
                        for (int i = 0; i < NK; ++i) {
                            const int k = gl + i * LP;
                            z1[i] = scr[padi<W>(row_slot_of<W>(k))];
                            z2[i] = scr[padi<W>(row_slot_of<W>(k == 0 ? W / 2 : W - k))];
                        }
#pragma unroll
                        for (int i = 0; i < NK; ++i) {
                            const int k = gl + i * LP;
                            float2 A, B;
                            if (k == 0) {  // z1 = slot of frequency 0, z2 = slot of frequency W/2
                                A = make_float2(z1[i].x, z2[i].x);
                                B = make_float2(z1[i].y, z2[i].y);
                            } else {
                                A = make_float2(0.5f * (z1[i].x + z2[i].x), 0.5f * (z1[i].y - z2[i].y));
                                B = make_float2(0.5f * (z1[i].y + z2[i].y), -0.5f * (z1[i].x - z2[i].x));
                            }
                            const int dr = k / NC;
                            if constexpr (SG || CS == 1) {
                                float2 *Sd = Sof(dr);
                                Sd[(size_t)ya * NC + (k % NC)] = A;
                                Sd[(size_t)yb * NC + (k % NC)] = B;
                            } else if (dr == rank) {
                                Ssm[(size_t)ya * NC + (k % NC)] = A;
                                Ssm[(size_t)yb * NC + (k % NC)] = B;
                            } else {  // a peer's columns: the bytes complete on the peer's sbar (no fence, no cluster barrier)
                                const uint32_t rb = mapa_u32(smem_u32(sbar), (uint32_t)dr);
                                st_async_b64(mapa_u32(smem_u32(Ssm + (size_t)ya * NC + (k % NC)), (uint32_t)dr),
                                             (uint64_t)__float_as_uint(A.x) | ((uint64_t)__float_as_uint(A.y) << 32), rb);
                                st_async_b64(mapa_u32(smem_u32(Ssm + (size_t)yb * NC + (k % NC)), (uint32_t)dr),
                                             (uint64_t)__float_as_uint(B.x) | ((uint64_t)__float_as_uint(B.y) << 32), rb);
                            }
                        }
                    }
                    __syncwarp();
                }
                __syncthreads();
                if (tid == 0 && ck + 2 < C::NCHK) {
                    mbar_expect_tx(&braw[rb], C::CHB);
                    bulk_g2s(raw + (size_t)rb * C::RCH * W, fbase + (size_t)(ck + 2) * C::RCH * W, C::CHB, &braw[rb]);
                }
            }
        }
        // every F_row[y][kx] is at its column owner: my own rows by the CTA barrier above, the peers' rows when their bytes
        // have completed on sbar
        if constexpr (SG || CS == 1) {
            csync();
        } else {
            mbar_wait(sbar, sph);
            sph ^= 1u;
        }
        stamp(0, f);

        // =============================================================== a2/a3/a4: column FFT (x) Gc, column inverse
        // (SG: the CTA's spectrum block lives in L2; its columns pass through shared memory NCB at a time -- one read and
        //  one write of the block per frame instead of one per pass: the column passes at 1024 x 1024 were L2-bandwidth bound)
        constexpr int NCB = SG ? 8 : NC;  // columns per block (SG: H x 8 complex in the U region, free during this phase)
        static_assert(!SG || ((size_t)H * NCB * 8 <= (size_t)C::RAWB + C::SCRB && NC % NCB == 0), "column block fits the raw + scratch region");
        for (int cb = 0; cb < NC / NCB; ++cb) {
            constexpr int R0 = cc_radix_col(H, 0), R1 = cc_radix_col(H, 1), R2 = cc_radix_col(H, 2);
            constexpr int RL = R2 > 1 ? R2 : R1;   // radix of the last forward pass (fused with the product)
            constexpr int NPASS = R2 > 1 ? 3 : 2;
            float2 *const Sb = SG ? reinterpret_cast<float2 *>(U) : Sl;  // [H][NCB]
            // element (y, ql) of the block.  SG: a row is 64 bytes, so rows y and y + 8 (two lanes of the contiguous-slot
            // passes) would meet the same banks: odd groups of 8 rows swap the two rows of each pair
            auto sbx = [&](int y, int ql) -> int {
                int a = y * NCB + ql;
                if constexpr (SG) a ^= ((y >> 3) & 1) << 3;
                return a;
            };
            if constexpr (SG) {
#pragma unroll 4
                for (int idx = tid; idx < H * NCB / 2; idx += NT) {
                    const int y = idx / (NCB / 2), c2 = idx % (NCB / 2);
                    *reinterpret_cast<float4 *>(Sb + sbx(y, 2 * c2)) =
                        __ldcg(reinterpret_cast<const float4 *>(Sl + (size_t)y * NC + cb * NCB + 2 * c2));
                }
                __syncthreads();
            }
            // forward pass 0
            for (int it = tid; it < NCB * (H / R0); it += NT) {
                const int ql = it % NCB, g = it / NCB;
                constexpr int ST = H / R0;
                fft_bfly<R0, false, true, NTW>([&](int i) { return Sb + sbx(g + i * ST, ql); }, g * (NTW / H), tw);
            }
            __syncthreads();
            if constexpr (NPASS == 3) {  // forward pass 1 of 3
                constexpr int L = H / R0, ST = L / R1;
                for (int it = tid; it < NCB * (H / R1); it += NT) {
                    const int ql = it % NCB, g = it / NCB;
                    const int blk = g / ST, b = g % ST;
                    fft_bfly<R1, false, true, NTW>([&](int i) { return Sb + sbx(blk * L + b + i * ST, ql); },
                                                   b * (NTW / L), tw);
                }
                __syncthreads();
            }
            // last forward pass (contiguous slots), product with conj(G)/(HW), first inverse pass
            for (int it = tid; it < NCB * (H / RL); it += NT) {
                const int ql = it % NCB, g = it / NCB;
                const int q = rank * NC + cb * NCB + ql;
                // the butterfly's RL values of conj(G)/(HW) are requested first (through L2: the RI update rewrites Gt),
                // so their latency runs under the shared-memory loads and the forward DFT
                float2 gv[RL];
                if constexpr (GPRE) {
#pragma unroll
                    for (int k = 0; k < RL; ++k) gv[k] = gpre[k];  // requested at the start of the frame
                } else if (q != 0) {
#pragma unroll
                    for (int k = 0; k < RL; ++k) gv[k] = __ldcg(&p.Gt[(size_t)(g * RL + k) * (W / 2) + q]);
                }
                float2 v[RL];
#pragma unroll
                for (int i = 0; i < RL; ++i) v[i] = Sb[sbx(g * RL + i, ql)];
                dft_reg<RL, false>(v);
                constexpr int bits = ilog2c(RL);
                if (q == 0) {  // packed DC/Nyquist column: needs the -ky partner, handled below
#pragma unroll
                    for (int k = 0; k < RL; ++k) Sb[sbx(g * RL + k, ql)] = v[brev(k, bits)];
                } else {
                    float2 w[RL];
#pragma unroll
                    for (int k = 0; k < RL; ++k) {
                        const size_t gi = (size_t)(g * RL + k) * (W / 2) + q;
                        if (RI) __stcg(&Fs_of()[gi], v[brev(k, bits)]);  // the frame's spectrum feeds the RI update
                        w[k] = cmul(v[brev(k, bits)], gv[k]);
                    }
                    dft_reg<RL, true>(w);
#pragma unroll
                    for (int n = 0; n < RL; ++n) Sb[sbx(g * RL + n, ql)] = w[brev(n, bits)];
                }
            }
            __syncthreads();
            if (rank == 0 && cb == 0) {
                // two real columns (kx = 0 and kx = W/2) ride in one complex FFT: split them with the -ky
                // partner, multiply each by its conj(G) column, re-pack as PA + i PB.  The split is done
                // first so that exact zeros stay exact (a constant frame must give P = 0, not rounding noise).
                constexpr int PER = (H + NT - 1) / NT;
                float2 o[PER];
#pragma unroll
                for (int e = 0; e < PER; ++e) {
                    const int s = tid + e * NT;
                    if (s < H) {
                        const float2 z = Sb[sbx(s, 0)], zp = Sb[sbx((int)p.col_partner[s], 0)];
                        const float4 g = __ldcg(&p.ab[s]);  // (G0c.re, G0c.im, Gnc.re, Gnc.im)
                        const float2 fa = make_float2(0.5f * (z.x + zp.x), 0.5f * (z.y - zp.y));
                        const float2 fb = make_float2(0.5f * (z.y + zp.y), -0.5f * (z.x - zp.x));
                        if (RI) __stcg(&Fab_of()[s], make_float4(fa.x, fa.y, fb.x, fb.y));
                        const float2 pa = cmul(fa, make_float2(g.x, g.y)), pb = cmul(fb, make_float2(g.z, g.w));
                        o[e] = make_float2(pa.x - pb.y, pa.y + pb.x);
                        if (s == 0) *f00 = z.x;  // sum of (I - c0): DC add-back for `peak`
                    }
                }
                __syncthreads();
#pragma unroll
                for (int e = 0; e < PER; ++e) {
                    const int s = tid + e * NT;
                    if (s < H) Sb[sbx(s, 0)] = o[e];
                }
                __syncthreads();
                for (int g = tid; g < H / RL; g += NT)
                    fft_bfly<RL, true, false, NTW>([&](int i) { return Sb + sbx(g * RL + i, 0); }, 0, tw);
                __syncthreads();
            }
            if constexpr (NPASS == 3) {  // inverse of forward pass 1
                constexpr int L = H / R0, ST = L / R1;
                for (int it = tid; it < NCB * (H / R1); it += NT) {
                    const int ql = it % NCB, g = it / NCB;
                    const int blk = g / ST, b = g % ST;
                    fft_bfly<R1, true, true, NTW>([&](int i) { return Sb + sbx(blk * L + b + i * ST, ql); },
                                                  b * (NTW / L), tw);
                }
                __syncthreads();
            }
            for (int it = tid; it < NCB * (H / R0); it += NT) {
                const int ql = it % NCB, g = it / NCB;
                constexpr int ST = H / R0;
                fft_bfly<R0, true, true, NTW>([&](int i) { return Sb + sbx(g + i * ST, ql); }, g * (NTW / H), tw);
            }
            if constexpr (SG) {  // the finished block goes back to L2
                __syncthreads();
#pragma unroll 4
                for (int idx = tid; idx < H * NCB / 2; idx += NT) {
                    const int y = idx / (NCB / 2), c2 = idx % (NCB / 2);
                    __stcg(reinterpret_cast<float4 *>(Sl + (size_t)y * NC + cb * NCB + 2 * c2),
                           *reinterpret_cast<const float4 *>(Sb + sbx(y, 2 * c2)));
                }
                __syncthreads();
            }
        }
        // Q[y][kx] complete everywhere: every CTA wrote its own block, the peers read it remotely (SG: through L2, fenced)
        if constexpr (SG) csync();
        else csync_ctl();
        stamp(1, f);

        // =============================================================== a4/a5: row C2R streamed into the integer argmax
        int y0, x0;
        double cc_peak = 0.0;
        {
            RowTw<W, NTW> rtw;
            rtw.load(tw, lane);
            Best bst{-INFINITY, 0x7fffffff};
            for (int jp0 = warp * RG; jp0 < NR / 2; jp0 += NWARP * RG) {
                const int jp = jp0 + gp;
                const int ya = rank * NR + jp, yb = ya + NR / 2;
                {
                    constexpr int NK = (W / 2) / LP;  // spectrum columns per lane
                    float2 qa[NK], qb[NK];
#pragma unroll
                    for (int i = 0; i < NK; ++i) {  // all loads first: the (remote, for k / NC != rank) latencies overlap
                        const int k = gl + i * LP;
                        const float2 *Sd = Sof(k / NC);
                        qa[i] = Sd[(size_t)ya * NC + (k % NC)];
                        qb[i] = Sd[(size_t)yb * NC + (k % NC)];
                    }
#pragma unroll
                    for (int i = 0; i < NK; ++i) {
                        const int k = gl + i * LP;
                        if (k == 0) {
                            scr[padi<W>(row_slot_of<W>(0))] = make_float2(qa[i].x, qb[i].x);
                            scr[padi<W>(row_slot_of<W>(W / 2))] = make_float2(qa[i].y, qb[i].y);
                        } else {
                            scr[padi<W>(row_slot_of<W>(k))] = make_float2(qa[i].x - qb[i].y, qa[i].y + qb[i].x);
                            scr[padi<W>(row_slot_of<W>(W - k))] = make_float2(qa[i].x + qb[i].y, qb[i].x - qa[i].y);
                        }
                    }
                }
                __syncwarp();
                // the last inverse pass streams its outputs (two rows of the correlation) into the argmax
                warp_fft_inv_to<W, NTW>(scr, rtw, gl, [&](int x, float2 z) {
                    if (better(z.x, ya * W + x, bst.v, bst.i)) bst.v = z.x, bst.i = ya * W + x;
                    if (better(z.y, yb * W + x, bst.v, bst.i)) bst.v = z.y, bst.i = yb * W + x;
                });
            }
            const Best g = cluster_best(bst);
            y0 = g.i / W;
            x0 = g.i % W;
            stamp(2, f);
            if constexpr (C::TC1) {
                // the first four weight tiles of stage 1 go into their ring now (the FFT scratch they overwrite is dead; the
                // fp64 polish below uses the first bytes of U only): their latency runs under the polish
                if (tid == 0 && u > 1) {
                    constexpr int KSTEPS = (H / 2 + 1 + 7) / 8;
                    const uint32_t etile = 4u * (uint32_t)p.N1 * 32u;
                    fence_proxy_async();
                    for (int ks = 0; ks < 4 && ks < KSTEPS; ++ks) {
                        const uint32_t slot = e_issued & 3u;
                        mbar_expect_tx(&ebar[slot], etile);
                        bulk_g2s(U + 32768 + (size_t)slot * etile, p.eblob + (size_t)ks * (size_t)(etile / 4), etile, &ebar[slot]);
                        ++e_issued;
                    }
                }
            }

            // fp64 re-evaluation of the 3x3 neighbourhood of the fp32 winner
            double *terms = reinterpret_cast<double *>(U);
            double nyq[3];
#pragma unroll
            for (int b = 0; b < 3; ++b) nyq[b] = ((x0 - 1 + b) & 1) ? -1.0 : 1.0;
            const double mine = xeval9(
                [&](int a, int ql, int) {
                    const float2 v = Sl[(size_t)((y0 - 1 + a) & (H - 1)) * NC + ql];
                    return make_double2((double)v.x, (double)v.y);
                },
                [&](int b, int q) { return tw64[(q * ((x0 - 1 + b) & (W - 1))) & (W - 1)]; }, nyq, terms);
            double bv;
            int bk;  // candidate k = a*3+b sits at ((y0-1+a) mod H, (x0-1+b) mod W); equal values: the smaller pixel index
            {
                const int a = lane / 3, b = lane % 3;
                best9(mine, (((y0 - 1 + a) & (H - 1)) * W) + ((x0 - 1 + b) & (W - 1)), true, bv, bk);
            }
            y0 = (y0 - 1 + bk / 3) & (H - 1);
            x0 = (x0 - 1 + bk % 3) & (W - 1);
            cc_peak = bv;
        }
        stamp(3, f);
        const int wy = (2 * y0 >= H) ? y0 - H : y0;
        const int wx = (2 * x0 >= W) ? x0 - W : x0;

        if (__builtin_expect(u == 1, false)) {
            if (rank == 0 && tid == 0) {
                const double Em = p.ri_emean ? __ldcg(p.ri_emean) : p.Emean;
                emit(f, (float)wy, (float)wx, (float)(p.peak_sign * (cc_peak + ((double)*f00 + c0d * H * W) * Em)), wy, wx);
            }
            if (__builtin_expect(RI, false)) {
                __syncthreads();  // the reference mean was read before it is rewritten
                ri_update((long long)wy, (long long)wx);
            }
            csync();
            continue;
        }

        // =============================================================== a6/a7: upsampled DFT as two symmetric FP32 GEMMs
        // Row pairs about the integer peak become their sum and difference (in place):
        //   S[(y0+j)] <- Q(y0+j) + Q(y0-j),  S[(y0-j)] <- Q(y0+j) - Q(y0-j),  0 < j < H/2.
        // (tensor-core stage 1 forms the sums and differences while it stages its operand: S keeps the plain Q there)
        if constexpr (!C::TC1) {
            for (int idx = tid; idx < (H / 2 - 1) * NC; idx += NT) {
                const int j = 1 + idx / NC, ql = idx % NC;
                float2 *pa = Sl + (size_t)((y0 + j) & (H - 1)) * NC + ql, *pb = Sl + (size_t)((y0 - j) & (H - 1)) * NC + ql;
                const float2 a = *pa, b = *pb;
                *pa = make_float2(a.x + b.x, a.y + b.y);
                *pb = make_float2(a.x - b.x, a.y - b.y);
            }
        }
        __syncthreads();

        Best sub{-INFINITY, 0x7fffffff};
        {
            const int DS = p.DS, nd = p.nd, DSBp = p.DSBp, DSB = DS * CS;
            constexpr int TN1 = C::TN1, TM1 = C::TM1, MC1 = C::MC1, R1 = C::R1, Cn1 = C::Cn1, BK1 = C::BK1;
            constexpr int TM2 = C::TM2, TN2 = C::TN2, R2 = C::R2, Cn2 = C::Cn2, KS2 = C::KS2, G2 = C::G2, GF2 = C::GF2;
            constexpr int KS1 = C::KS1, NW1 = NWARP / KS1;  // warps per stage-1 k-slice
            const int ks1 = warp / NW1, w1 = warp % NW1;
            const int tn1 = (w1 % C::WG1C) * C::WC1 + lane % C::WC1;
            const int tm1 = (w1 / C::WG1C) * C::WR1 + lane / C::WC1;
            const int ks2 = warp / (C::WG2R * C::WG2C), w2 = warp % (C::WG2R * C::WG2C);
            const int tn2 = (w2 % C::WG2C) * C::WC2 + lane % C::WC2;
            const int tm2 = (w2 / C::WG2C) * C::WR2 + lane / C::WC2;
            float *const red = Tb + (size_t)2 * DS * LDT;  // k-split partial sums (KS1 > 1, KS2 > 1)
            for (int sb = 0; sb < p.nsb; ++sb) {
                const int db = sb * DSB;
                // stage-1 output rows reach their owner by st.async: my live offsets x 2 rows x the peers' 2 NC floats each
                if constexpr (CS > 1) {
                    if (tid == 0) {
                        const int n_live = min(max(nd - db - rank * DS, 0), DS);
                        mbar_expect_tx(trow, (uint32_t)((CS - 1) * n_live * 2 * (2 * NC) * 4));
                    }
                }
                if constexpr (C::TC1) {
                // ---------------- stage 1 on the tensor cores (tcgen05.mma kind::tf32, accumulators in tensor memory):
                //   U[d][n] = sum_j Ee[d][j] S[(y0+j)][n],  V[d][n] = sum_j Eo[d][j] S[(y0-j)][n]   (n = my 128 spectrum floats;
                //   the offsets d are the MMA's M = 128 rows = tensor-memory lanes, so a thread of the epilogue owns a row of T)
                // per 8 rows j as 128 x N x 8 MMAs, each product split into TF32 passes (x = hi + lo, the low 13 mantissa
                // bits split off exactly; lo*hi + hi*lo + hi*hi carries ~22 bits of both operands: FP32-level accuracy,
                // profiles/r2a_tc_probe.json).  An MMA instruction costs its issuing thread ~75 cycles whatever N is, so
                // the hi*hi and hi*lo passes are ONE instruction (B = [S_hi ; S_lo], N = 256, two accumulator halves
                // that the epilogue adds) and U and V are issued by two different threads.  The weight tables hold only
                // their N1 <= 128 used rows: the MMA reads 128, the rows beyond N1 produce lanes nobody reads.  The CTA's threads stage
                // the data operand (8 rows of S -> K-major core matrices, hi and lo) into a double buffer while the MMAs
                // of the previous 8 rows run; the plan-constant operand (Ee / Eo, hi / lo, already in UMMA layout)
                // arrives by TMA through a 4-slot ring.  Epilogue: tensor memory -> registers, T(c+-d) = U +- V,
                // rotation by exp(2 pi i kx x0 / W), rows to their owners.
                {
                    constexpr int KSTEPS = (H / 2 + 1 + 7) / 8;
                    const int N1 = p.N1;
                    const uint32_t etab = (uint32_t)N1 * 32u, etile = 4u * etab;   // bytes of one table / one operand tile
                    unsigned char *const abuf = U;                                   // [2][4][4096]: U_hi, U_lo, V_hi, V_lo
                    unsigned char *const ering = U + 32768;                          // [4][etile]: Ee_hi, Ee_lo, Eo_hi, Eo_lo
                    const uint32_t idescA = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(256 >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
                    const uint32_t idescB = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(128 >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
                    const float *Sf = reinterpret_cast<const float *>(Sl);
                    auto issue_etile = [&](int ks) {  // thread 0
                        const uint32_t slot = e_issued & 3u;
                        mbar_expect_tx(&ebar[slot], etile);
                        bulk_g2s(ering + (size_t)slot * etile, p.eblob + ((size_t)sb * KSTEPS + ks) * (size_t)(etile / 4), etile, &ebar[slot]);
                        ++e_issued;
                    };
                    if (tid == 0 && sb > 0) {  // (super-block 0: requested right after the integer argmax)
                        fence_proxy_async();
                        for (int ks = 0; ks < 4 && ks < KSTEPS; ++ks) issue_etile(ks);
                    }
                    // Producer / consumer: warps 0-3 stage the data operand (thread n: spectrum float n, the 8 rows of the step,
                    // sums and differences of the row pairs formed on the way: S keeps the plain Q) and arrive on afull[b];
                    // lane 0 of warp 6 (U) and of warp 7 (V) wait for it, issue the MMAs and commit to mdone[b], which frees
                    // buffer b two steps later.  No CTA barrier inside the loop.
                    if (warp < 4) {  // thread n: spectrum float n, the 8 rows of the step (two 16-byte K chunks per table)
                        const int sn = tid;
                        float qa[8], qb[8];
                        auto load_rows = [&](int ks) {
#pragma unroll
                            for (int i = 0; i < 8; ++i) {
                                const int j = ks * 8 + i;   // rows beyond H/2 meet zero weights
                                qa[i] = Sf[(size_t)((y0 + j) & (H - 1)) * (2 * NC) + sn];
                                qb[i] = Sf[(size_t)((y0 - j) & (H - 1)) * (2 * NC) + sn];
                            }
                        };
                        if constexpr (SG) load_rows(0);
                        for (int ks = 0; ks < KSTEPS; ++ks) {
                            const int b = ks & 1;
                            if constexpr (!SG) load_rows(ks);
                            float up[8], vm[8];  // Q(y0+j) + Q(y0-j), Q(y0+j) - Q(y0-j); rows j = 0 and H/2 stand alone
#pragma unroll
                            for (int i = 0; i < 8; ++i) {
                                const int j = ks * 8 + i;
                                const bool alone = j == 0 || j == H / 2;
                                up[i] = alone ? qa[i] : qa[i] + qb[i];
                                vm[i] = qa[i] - qb[i];
                            }
                            if constexpr (SG) {  // spectrum block in L2: the next step's rows are requested a step ahead
                                if (ks + 1 < KSTEPS) load_rows(ks + 1);
                            }
                            if (ks >= 2) {
                                if (lane == 0) mbar_wait(&mdone[b], mph[b] & 1u);  // one poller per warp
                                __syncwarp();
                                ++mph[b];
                                if (tid == 0 && ks + 2 < KSTEPS) issue_etile(ks + 2);
                            }
                            unsigned char *dst = abuf + (size_t)b * 16384 + (sn >> 3) * 256 + (sn & 7) * 16;
#pragma unroll
                            for (int kh = 0; kh < 2; ++kh) {
                                const float4 uh = make_float4(tf32_hi(up[4 * kh]), tf32_hi(up[4 * kh + 1]), tf32_hi(up[4 * kh + 2]), tf32_hi(up[4 * kh + 3]));
                                const float4 vh = make_float4(tf32_hi(vm[4 * kh]), tf32_hi(vm[4 * kh + 1]), tf32_hi(vm[4 * kh + 2]), tf32_hi(vm[4 * kh + 3]));
                                const float4 ul = make_float4(tf32_hi(up[4 * kh] - uh.x), tf32_hi(up[4 * kh + 1] - uh.y), tf32_hi(up[4 * kh + 2] - uh.z),
                                                              tf32_hi(up[4 * kh + 3] - uh.w));
                                const float4 vl = make_float4(tf32_hi(vm[4 * kh] - vh.x), tf32_hi(vm[4 * kh + 1] - vh.y), tf32_hi(vm[4 * kh + 2] - vh.z),
                                                              tf32_hi(vm[4 * kh + 3] - vh.w));
                                *reinterpret_cast<float4 *>(dst + kh * 128) = uh;
                                *reinterpret_cast<float4 *>(dst + kh * 128 + 4096) = ul;
                                *reinterpret_cast<float4 *>(dst + kh * 128 + 8192) = vh;
                                *reinterpret_cast<float4 *>(dst + kh * 128 + 12288) = vl;
                            }
                            fence_proxy_async();  // generic-proxy stores -> visible to the tensor core
                            asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&afull[b])) : "memory");
                        }
                    } else if (warp < 6) {
                        for (int ks = 2; ks < KSTEPS; ++ks) ++mph[ks & 1];  // keeps the completion count of every thread in step
                    } else {
                        for (int ks = 0; ks < KSTEPS; ++ks) {
                            const int b = ks & 1;
                            if (ks >= 2) ++mph[b];  // keeps the completion count of every thread in step
                            if (lane == 0) {
                                const uint32_t isV = warp == 7 ? 1u : 0u;
                                mbar_wait(&ebar[e_cons & 3u], (e_cons >> 2) & 1u);  // (landed long ago: first, off the critical path)
                                mbar_wait(&afull[b], aph[b] & 1u);
                                const uint32_t eb = smem_u32(ering + (size_t)(e_cons & 3u) * etile) + isV * 2u * etab;
                                const uint32_t ab = smem_u32(abuf + (size_t)b * 16384) + isV * 8192u;
                                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                                const uint32_t acc = ks > 0 ? 1u : 0u, d0 = tmem + isV * 256u;
                                // [D1 | D2] (+)= E_hi [S_hi ; S_lo]^T ;  D2 += E_lo S_hi^T ;  result = D1 + D2
                                umma_tf32(d0, umma_desc(eb, 128, 256), umma_desc(ab, 128, 256), idescA, acc);
                                umma_tf32(d0 + 128u, umma_desc(eb + etab, 128, 256), umma_desc(ab, 128, 256), idescB, 1u);
                                umma_commit(&mdone[b]);
                            }
                            ++aph[b];
                            ++e_cons;
                        }
                    }
                    if (warp < 6) e_cons += (uint32_t)KSTEPS;  // every thread counts the consumed tiles alike
#pragma unroll
                    for (int t = (KSTEPS >= 2 ? KSTEPS - 2 : 0); t < KSTEPS; ++t) {  // the last two steps complete
                        mbar_wait(&mdone[t & 1], mph[t & 1] & 1u);
                        ++mph[t & 1];
                    }
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    csync_ctl();  // no CTA of the cluster stages operands in its U region any more: T rows may land there
                    {   // thread = (offset d = lane of tensor memory, half of the 128 spectrum floats): a row segment of T
                        const int lb = 32 * (warp & 3), dsb = lb + lane, half = warp >> 2;
                        const bool live = dsb < DSB && db + dsb < nd;
                        const int dr = dsb / DS, row = dsb % DS;
                        float *const dstp = Tb + (size_t)row * LDT + rank * 2 * NC, *const dstm = dstp + (size_t)DS * LDT;
                        const bool remote = CS > 1 && live && dr != rank;
                        uint32_t rp = 0, rm = 0, rb = 0;  // the owner's copy of the two rows and its trow barrier
                        if constexpr (CS > 1) {
                            if (remote) rp = mapa_u32(smem_u32(dstp), (uint32_t)dr), rm = mapa_u32(smem_u32(dstm), (uint32_t)dr),
                                        rb = mapa_u32(smem_u32(trow), (uint32_t)dr);
                        }
                        const float sg = (x0 & 1) ? -1.f : 1.f;
                        const uint32_t tb = tmem + ((uint32_t)lb << 16);
#pragma unroll 1
                        for (int c0 = half * 64; c0 < half * 64 + 64; c0 += 16) {  // 16 spectrum floats per round trip
                            uint32_t r[4][2][8];
#pragma unroll
                            for (int a4 = 0; a4 < 4; ++a4)
#pragma unroll
                                for (int g = 0; g < 2; ++g) tmem_ld8(tb + (uint32_t)(a4 * 128 + c0 + 8 * g), r[a4][g]);
                            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                            float op[16], om[16];
#pragma unroll
                            for (int i = 0; i < 16; i += 2) {
                                const int g = i >> 3, k = i & 7;
                                const float ur = __uint_as_float(r[0][g][k]) + __uint_as_float(r[1][g][k]);
                                const float ui = __uint_as_float(r[0][g][k + 1]) + __uint_as_float(r[1][g][k + 1]);
                                const float vr = __uint_as_float(r[2][g][k]) + __uint_as_float(r[3][g][k]);
                                const float vi = __uint_as_float(r[2][g][k + 1]) + __uint_as_float(r[3][g][k + 1]);
                                const float2 tp = make_float2(ur + vr, ui + vi), tm = make_float2(ur - vr, ui - vi);
                                const int q = rank * NC + ((c0 + i) >> 1);
                                if (q == 0) {  // packed column: (DC, Nyquist) -- the Nyquist part carries (-1)^x0
                                    op[i] = tp.x, op[i + 1] = tp.y * sg, om[i] = tm.x, om[i + 1] = tm.y * sg;
                                } else {
                                    const float2 w = tw[((q * x0) & (W - 1)) * (NTW / W)];  // (cos, -sin)
                                    const float2 a = cmulc(tp, w), bq = cmulc(tm, w);
                                    op[i] = a.x, op[i + 1] = a.y, om[i] = bq.x, om[i + 1] = bq.y;
                                }
                            }
                            if (remote) {
#pragma unroll
                                for (int v = 0; v < 4; ++v) {
                                    st_async_v4(rp + (uint32_t)(c0 + 4 * v) * 4u, make_float4(op[4 * v], op[4 * v + 1], op[4 * v + 2], op[4 * v + 3]), rb);
                                    st_async_v4(rm + (uint32_t)(c0 + 4 * v) * 4u, make_float4(om[4 * v], om[4 * v + 1], om[4 * v + 2], om[4 * v + 3]), rb);
                                }
                            } else if (live) {
#pragma unroll
                                for (int v = 0; v < 4; ++v) {
                                    *reinterpret_cast<float4 *>(dstp + c0 + 4 * v) = make_float4(op[4 * v], op[4 * v + 1], op[4 * v + 2], op[4 * v + 3]);
                                    *reinterpret_cast<float4 *>(dstm + c0 + 4 * v) = make_float4(om[4 * v], om[4 * v + 1], om[4 * v + 2], om[4 * v + 3]);
                                }
                            }
                        }
                    }
                    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                    __syncthreads();  // my own rows of T(c+d), T(c-d) ...
                    if constexpr (CS > 1) {  // ... and the peers' (their bytes have completed on trow)
                        mbar_wait(trow, tph1);
                        tph1 ^= 1u;
                    }
                }
                } else {
                // ---------------- stage 1: rows [U(d) | V(d)] of this super-block, my 2*NC spectrum floats
                //   U(d) = sum_j Ee[d][j] S[(y0+j)],  V(d) = sum_j Eo[d][j] S[(y0-j)];  T(c+d) = U+V, T(c-d) = U-V
                for (int ch = 0; ch < p.nch1; ++ch) {
                    const int gc0 = ch * MC1 + tm1 * TM1;
                    const bool isV = gc0 >= DSBp;
                    float acc[TM1][TN1];
                    unsigned long long acc2[TM1][TN1 / 2];  // the k-loop accumulates column pairs with FFMA2
#pragma unroll
                    for (int i = 0; i < TM1; ++i)
#pragma unroll
                        for (int j = 0; j < TN1 / 2; ++j) acc2[i][j] = 0ull;
                    for (int kt = 0; kt < p.KT1; ++kt) {
                        const float *At = ring_acquire();
#pragma unroll
                        for (int kq = 0; kq < BK1 / KS1; ++kq) {
                            const int kk = kq * KS1 + ks1;
                            const int jj = kt * BK1 + kk;
                            const int ys = (isV ? y0 - jj : y0 + jj) & (H - 1);
                            float a[TM1], b[TN1];
#pragma unroll
                            for (int ci = 0; ci < cc_tm1_nchunks(TM1); ++ci) {
                                const int w = cc_tm1_width(TM1, ci), st = cc_tm1_start(TM1, ci);
                                const float *src = At + kk * MC1 + R1 * st + tm1 * w;
                                if (w == 4) {
                                    const float4 t = *reinterpret_cast<const float4 *>(src);
                                    a[st] = t.x, a[st + 1] = t.y, a[st + 2] = t.z, a[st + 3] = t.w;
                                } else if (w == 2) {
                                    const float2 t = *reinterpret_cast<const float2 *>(src);
                                    a[st] = t.x, a[st + 1] = t.y;
                                } else {
                                    a[st] = src[0];
                                }
                            }
                            const float *brow = reinterpret_cast<const float *>(Sl + (size_t)ys * NC) + tn1 * 4;
#pragma unroll
                            for (int v = 0; v < TN1 / 4; ++v) {
                                const float4 t = *reinterpret_cast<const float4 *>(brow + v * Cn1 * 4);
                                b[4 * v] = t.x, b[4 * v + 1] = t.y, b[4 * v + 2] = t.z, b[4 * v + 3] = t.w;
                            }
                            unsigned long long b2[TN1 / 2];
#pragma unroll
                            for (int j = 0; j < TN1 / 2; ++j) b2[j] = pack2(b[2 * j], b[2 * j + 1]);
#pragma unroll
                            for (int i = 0; i < TM1; ++i) {
                                const unsigned long long aa = pack2(a[i], a[i]);
#pragma unroll
                                for (int j = 0; j < TN1 / 2; ++j) acc2[i][j] = fma2(aa, b2[j], acc2[i][j]);
                            }
                        }
                        ring_release();
                    }
#pragma unroll
                    for (int i = 0; i < TM1; ++i)
#pragma unroll
                        for (int j = 0; j < TN1 / 2; ++j) unpack2(acc2[i][j], acc[i][2 * j], acc[i][2 * j + 1]);
                    if constexpr (KS1 > 1) {  // sum the k-slices into slice 0
                        const int t1 = tm1 * Cn1 + tn1;
                        if (ks1 > 0) {
                            float *r = red + (size_t)(ks1 - 1) * (TM1 * TN1) * (R1 * Cn1) + t1;
#pragma unroll
                            for (int i = 0; i < TM1; ++i)
#pragma unroll
                                for (int j = 0; j < TN1; ++j) r[(size_t)(i * TN1 + j) * (R1 * Cn1)] = acc[i][j];
                        }
                        __syncthreads();
                        if (ks1 == 0) {
                            for (int s1 = 0; s1 < KS1 - 1; ++s1) {
                                const float *r = red + (size_t)s1 * (TM1 * TN1) * (R1 * Cn1) + t1;
#pragma unroll
                                for (int i = 0; i < TM1; ++i)
#pragma unroll
                                    for (int j = 0; j < TN1; ++j) acc[i][j] += r[(size_t)(i * TN1 + j) * (R1 * Cn1)];
                            }
                        }
                        __syncthreads();
                    }
                    // epilogue: rotate by exp(2 pi i kx x0 / W), send rows to the CTA that owns offset d
                    if (ks1 == 0) {
#pragma unroll
                    for (int v = 0; v < TN1 / 4; ++v)
#pragma unroll
                        for (int pp = 0; pp < 2; ++pp) {
                            const int q = rank * NC + v * Cn1 * 2 + tn1 * 2 + pp;
                            const int j0 = 4 * v + 2 * pp;
                            if (q == 0) {
                                const float sg = (x0 & 1) ? -1.f : 1.f;
#pragma unroll
                                for (int i = 0; i < TM1; ++i) acc[i][j0 + 1] *= sg;
                            } else {
                                const float2 w = tw[((q * x0) & (W - 1)) * (NTW / W)];  // (cos, -sin)
#pragma unroll
                                for (int i = 0; i < TM1; ++i) {
                                    const float2 t = cmulc(make_float2(acc[i][j0], acc[i][j0 + 1]), w);
                                    acc[i][j0] = t.x;
                                    acc[i][j0 + 1] = t.y;
                                }
                            }
                        }
#pragma unroll
                    for (int i = 0; i < TM1; ++i) {
                        const int dsb = gc0 + i - (isV ? DSBp : 0);
                        if (dsb < DSB && db + dsb < nd) {
                            const int dr = dsb / DS, row = dsb % DS + (isV ? DS : 0);
                            float *dst = Tb + (size_t)row * LDT + rank * 2 * NC + tn1 * 4;
                            if constexpr (CS == 1) {
#pragma unroll
                                for (int v = 0; v < TN1 / 4; ++v)
                                    *reinterpret_cast<float4 *>(dst + v * Cn1 * 4) =
                                        make_float4(acc[i][4 * v], acc[i][4 * v + 1], acc[i][4 * v + 2], acc[i][4 * v + 3]);
                            } else if (dr == rank) {
#pragma unroll
                                for (int v = 0; v < TN1 / 4; ++v)
                                    *reinterpret_cast<float4 *>(dst + v * Cn1 * 4) =
                                        make_float4(acc[i][4 * v], acc[i][4 * v + 1], acc[i][4 * v + 2], acc[i][4 * v + 3]);
                            } else {  // the owner's copy of the row; the bytes complete on its trow barrier
                                const uint32_t rd = mapa_u32(smem_u32(dst), (uint32_t)dr), rb = mapa_u32(smem_u32(trow), (uint32_t)dr);
#pragma unroll
                                for (int v = 0; v < TN1 / 4; ++v)
                                    st_async_v4(rd + (uint32_t)(v * Cn1 * 4) * 4u,
                                                make_float4(acc[i][4 * v], acc[i][4 * v + 1], acc[i][4 * v + 2], acc[i][4 * v + 3]), rb);
                            }
                        }
                    }
                    }  // ks1 == 0
                }
                // U, V rows are at their owners: mine after the CTA barrier, the peers' when their bytes have completed
                __syncthreads();
                if constexpr (CS > 1) {
                    mbar_wait(trow, tph1);
                    tph1 ^= 1u;
                }
                // rows dl and DS+dl become T(c+d) = U+V and T(c-d) = U-V
                for (int idx = tid; idx < DS * (W / 4); idx += NT) {
                    const int dl = idx / (W / 4), c4 = idx % (W / 4);
                    float4 *pu = reinterpret_cast<float4 *>(Tb + (size_t)dl * LDT) + c4;
                    float4 *pv = reinterpret_cast<float4 *>(Tb + (size_t)(DS + dl) * LDT) + c4;
                    const float4 a = *pu, b = *pv;
                    *pu = make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w);
                    *pv = make_float4(a.x - b.x, a.y - b.y, a.z - b.z, a.w - b.w);
                }
                __syncthreads();
                }  // FP32 stage 1
                stamp(4, f);

                // ---------------- stage 2: E(m,e) = sum_q T_re w cos, O(m,e) = sum_q T_im w sin;
                //   C(m, c+e) = E - O,  C(m, c-e) = E + O, streamed into the argmax
                const int d0 = db + rank * DS;  // offset d of my T row 0
                for (int rc2 = 0; rc2 < p.nrc2; ++rc2) {
                    const int rbase = rc2 * R2 * TM2 + tm2 * TM2;
                    const float *Arow[TM2];
#pragma unroll
                    for (int i = 0; i < TM2; ++i) Arow[i] = Tb + (size_t)min(rbase + i, 2 * DS - 1) * LDT;
                    for (int nc2 = 0; nc2 < p.nnc2; ++nc2) {
                        float aE[TM2][TN2], aO[TM2][TN2];
                        unsigned long long aE2[TM2][2], aO2[TM2][2];  // columns 0..3 as pairs (FFMA2); column 4 scalar
#pragma unroll
                        for (int i = 0; i < TM2; ++i) {
                            aE2[i][0] = aE2[i][1] = aO2[i][0] = aO2[i][1] = 0ull;
                            if constexpr (TN2 > 4) aE[i][4] = 0.f, aO[i][4] = 0.f;
                        }
                        constexpr int KT2 = W / (4 * G2);
                        for (int kt = 0; kt < KT2; ++kt) {
                            const float *Bt = ring_acquire();
#pragma unroll
                            for (int gi = 0; gi < G2 / KS2; ++gi) {
                                const int g = gi * KS2 + ks2;
                                const int k0 = (kt * G2 + g) * 4;
                                const float *grp = Bt + g * GF2 + tn2 * 4;
                                float4 a4[TM2];
#pragma unroll
                                for (int i = 0; i < TM2; ++i) a4[i] = *reinterpret_cast<const float4 *>(Arow[i] + k0);
                                float4 x4 = make_float4(0.f, 0.f, 0.f, 0.f);
                                if constexpr (C::X2 == 1) x4 = *reinterpret_cast<const float4 *>(grp + 16 * Cn2);
#pragma unroll
                                for (int kk = 0; kk < 4; ++kk) {
                                    const float4 b4 = *reinterpret_cast<const float4 *>(grp + kk * Cn2 * 4);
                                    float b[TN2];
                                    b[0] = b4.x, b[1] = b4.y, b[2] = b4.z, b[3] = b4.w;
                                    if constexpr (C::X2 == 1) b[4] = kk == 0 ? x4.x : kk == 1 ? x4.y : kk == 2 ? x4.z : x4.w;
                                    const unsigned long long b01 = pack2(b[0], b[1]), b23 = pack2(b[2], b[3]);
#pragma unroll
                                    for (int i = 0; i < TM2; ++i) {
                                        const float av = kk == 0 ? a4[i].x : kk == 1 ? a4[i].y : kk == 2 ? a4[i].z : a4[i].w;
                                        const unsigned long long aa = pack2(av, av);
                                        if ((kk & 1) == 0) {
                                            aE2[i][0] = fma2(aa, b01, aE2[i][0]), aE2[i][1] = fma2(aa, b23, aE2[i][1]);
                                            if constexpr (TN2 > 4) aE[i][4] = fmaf(av, b[4], aE[i][4]);
                                        } else {
                                            aO2[i][0] = fma2(aa, b01, aO2[i][0]), aO2[i][1] = fma2(aa, b23, aO2[i][1]);
                                            if constexpr (TN2 > 4) aO[i][4] = fmaf(av, b[4], aO[i][4]);
                                        }
                                    }
                                }
                            }
                            ring_release();
                        }
#pragma unroll
                        for (int i = 0; i < TM2; ++i) {
                            unpack2(aE2[i][0], aE[i][0], aE[i][1]), unpack2(aE2[i][1], aE[i][2], aE[i][3]);
                            unpack2(aO2[i][0], aO[i][0], aO[i][1]), unpack2(aO2[i][1], aO[i][2], aO[i][3]);
                        }
                        if constexpr (KS2 > 1) {  // sum the k-slices into slice 0
                            const int t2 = tm2 * Cn2 + tn2;
                            if (ks2 > 0) {
                                float *r = red + (size_t)(ks2 - 1) * (2 * TM2 * TN2) * (R2 * Cn2) + t2;
#pragma unroll
                                for (int i = 0; i < TM2; ++i)
#pragma unroll
                                    for (int j = 0; j < TN2; ++j) {
                                        r[(size_t)(2 * (i * TN2 + j)) * (R2 * Cn2)] = aE[i][j];
                                        r[(size_t)(2 * (i * TN2 + j) + 1) * (R2 * Cn2)] = aO[i][j];
                                    }
                            }
                            __syncthreads();
                            if (ks2 == 0) {
                                for (int s2 = 0; s2 < KS2 - 1; ++s2) {
                                    const float *r = red + (size_t)s2 * (2 * TM2 * TN2) * (R2 * Cn2) + t2;
#pragma unroll
                                    for (int i = 0; i < TM2; ++i)
#pragma unroll
                                        for (int j = 0; j < TN2; ++j) {
                                            aE[i][j] += r[(size_t)(2 * (i * TN2 + j)) * (R2 * Cn2)];
                                            aO[i][j] += r[(size_t)(2 * (i * TN2 + j) + 1) * (R2 * Cn2)];
                                        }
                                }
                            }
                            __syncthreads();
                        }
                        if (ks2 == 0) {
                            const int ebase = nc2 * C::NCOL2;
                            float ny[TN2];
                            int ee[TN2];
#pragma unroll
                            for (int j = 0; j < TN2; ++j) {
                                ee[j] = ebase + (j < 4 ? tn2 * 4 + j : 4 * Cn2 + tn2);
                                ny[j] = __ldg(&p.nyqc[ee[j]]);
                            }
                            // C(m, c+e) = E - O and C(m, c-e) = E + O overwrite the accumulators (-inf outside the
                            // grid); the chunk's maximum comes from an independent max tree, its smallest index from a
                            // min tree over the equal entries -- no serial compare-select chain per output
                            constexpr float NEG = -INFINITY;
                            int mrow[TM2];
                            float vmax = NEG;
#pragma unroll
                            for (int i = 0; i < TM2; ++i) {
                                const int r = rbase + i;
                                const bool lower = r >= DS;          // row holds T(c-d)
                                const int d = d0 + (lower ? r - DS : r);
                                const int m = lower ? cM - d : cM + d;
                                const bool rok = r < 2 * DS && d < nd && m >= 0 && m < M && !(lower && d == 0);
                                mrow[i] = rok ? m * M + cM : -1;
                                const float tny = Arow[i][1];         // Nyquist column of this T row
#pragma unroll
                                for (int j = 0; j < TN2; ++j) {
                                    const int e = ee[j];
                                    const float E = fmaf(tny, ny[j], aE[i][j]), O = aO[i][j];
                                    const bool ok = rok && e < nd;
                                    aE[i][j] = (ok && cM + e < M) ? E - O : NEG;   // column c + e
                                    aO[i][j] = (ok && e > 0) ? E + O : NEG;        // column c - e
                                }
                                float rm = NEG;
#pragma unroll
                                for (int j = 0; j < TN2; ++j) rm = fmaxf(rm, fmaxf(aE[i][j], aO[i][j]));
                                vmax = fmaxf(vmax, rm);
                            }
                            if (vmax > sub.v || (vmax == sub.v && vmax > NEG)) {
                                int imin = 0x7fffffff;
#pragma unroll
                                for (int i = 0; i < TM2; ++i)
#pragma unroll
                                    for (int j = 0; j < TN2; ++j) {
                                        if (aO[i][j] == vmax) imin = min(imin, mrow[i] - ee[j]);
                                        if (aE[i][j] == vmax) imin = min(imin, mrow[i] + ee[j]);
                                    }
                                if (better(vmax, imin, sub.v, sub.i)) sub.v = vmax, sub.i = imin;
                            }
                        }
                    }
                }
                stamp(5, f);
                if (sb + 1 < p.nsb) csync_ctl();  // T is overwritten by the next super-block
            }
        }
        int ms, ns;
        {
            const Best g = cluster_best(sub);
            ms = g.i / M;
            ns = g.i % M;
        }
        stamp(6, f);

        // ---------------- fp64 3x3 hill-climb on the 1/u grid, from the fp32 Q
        double up_peak = 0.0;
        {
            constexpr int NSL = (NT / NC) > 0 ? (NT / NC) : 1;  // j-slices per column
            double *dtab = reinterpret_cast<double *>(U);                      // [3][H]
            double2 *part = reinterpret_cast<double2 *>(dtab + 3 * H);         // [3][NSL][NC]
            double *terms = reinterpret_cast<double *>(part + 3 * NSL * NC);   // [9][NC]
            if (pol_pending) {  // first frame: the resident polish tables (TMA copies issued during the setup) have landed
                mbar_wait(pbar, 0u);
                pol_pending = false;
            }
            static_assert(NSL * NC == NT, "one (column, slice) element per thread in the fp64 polish");
            // the three row sums  sum_j D[m][j] Q[(y0+j)][q]  of rows ms-1, ms, ms+1: a move along n keeps all of them, a
            // move along m keeps two -- only what entered the window is evaluated again (need: bit a = row a)
            double2 s0 = make_double2(0.0, 0.0), s1 = s0, s2 = s0;
            int need = 7;
            for (int iter = 0; iter < 8; ++iter) {
                // weights of the physical rows (y0+j) mod H, which hold Q(y0), Q(y0+H/2), the sums
                // Q(y0+j)+Q(y0-j) (0 < j < H/2) and the differences Q(y0+j')-Q(y0-j') (j = H-j'):
                // rows ms-1..ms+1 of the plan's fp64 table Dpol[M][H] (out-of-grid rows: their values are never used)
                const double *dr0 = dtab, *dr1 = dtab + H, *dr2 = dtab + 2 * H;
                if (POLS) {
                    dr0 = DpolS + (size_t)min(max(ms - 1, 0), M - 1) * H;
                    dr1 = DpolS + (size_t)min(max(ms, 0), M - 1) * H;
                    dr2 = DpolS + (size_t)min(max(ms + 1, 0), M - 1) * H;
                } else {
#pragma unroll
                    for (int it = 0; it < (3 * H + NT - 1) / NT; ++it) {  // unrolled: all loads of a thread go out together
                        const int e = tid + it * NT;
                        if (e < 3 * H) {
                            const int a = e / H, j = e % H;
                            const int mm = ms - 1 + a;
                            dtab[e] = (mm >= 0 && mm < M) ? __ldg(&(C::TC1 ? p.DpolPlain : p.Dpol)[(size_t)mm * H + j]) : 0.0;
                        }
                    }
                    __syncthreads();
                }
                {   // (NSL * NC == NT: one (column, slice) element per thread, whose three row sums live across the iterations)
                    const int ql = tid % NC, sl = tid / NC;
                    if (need == 7) {
                        for (int j = sl; j < H; j += NSL) {
                            const float2 v = Sl[(size_t)((y0 + j) & (H - 1)) * NC + ql];
                            const double vx = (double)v.x, vy = (double)v.y;
                            const double d0 = dr0[j], d1 = dr1[j], d2 = dr2[j];
                            s0.x = fma(d0, vx, s0.x), s0.y = fma(d0, vy, s0.y);
                            s1.x = fma(d1, vx, s1.x), s1.y = fma(d1, vy, s1.y);
                            s2.x = fma(d2, vx, s2.x), s2.y = fma(d2, vy, s2.y);
                        }
                    } else if (need != 0) {  // after a move along m: only the row that entered the window (same order of additions)
                        const double *const dn = need == 1 ? dr0 : dr2;
                        double2 sn = make_double2(0.0, 0.0);
                        for (int j = sl; j < H; j += NSL) {
                            const float2 v = Sl[(size_t)((y0 + j) & (H - 1)) * NC + ql];
                            const double d = dn[j];
                            sn.x = fma(d, (double)v.x, sn.x), sn.y = fma(d, (double)v.y, sn.y);
                        }
                        if (need == 1) s0 = sn;
                        else s2 = sn;
                    }
                    part[(0 * NSL + sl) * NC + ql] = s0;
                    part[(1 * NSL + sl) * NC + ql] = s1;
                    part[(2 * NSL + sl) * NC + ql] = s2;
                }
                double nyq[3];
                const double sgx = (x0 & 1) ? -1.0 : 1.0;
#pragma unroll
                for (int b = 0; b < 3; ++b) {
                    const int nn = min(max(ns - 1 + b, 0), M - 1);  // out-of-grid neighbours are skipped below
                    nyq[b] = sgx * (POLS ? nyqS[nn] : __ldg(&p.nyq64[nn]));
                }
                __syncthreads();
                const double mine = xeval9(
                    [&](int a, int ql, int sub) {  // sum of the j-slices, 8 lanes per (a, ql)
                        double sx = 0.0, sy = 0.0;
                        for (int sl = sub; sl < NSL; sl += 8) {
                            const double2 t = part[(a * NSL + sl) * NC + ql];
                            sx += t.x, sy += t.y;
                        }
#pragma unroll
                        for (int o = 1; o < 8; o <<= 1) {
                            sx += __shfl_xor_sync(0xffffffffu, sx, o);
                            sy += __shfl_xor_sync(0xffffffffu, sy, o);
                        }
                        return make_double2(sx, sy);
                    },
                    [&](int b, int q) {
                        // exp(2 pi i q (x0 u + n - c) / (u W)) = exp(2 pi i q x0 / W) * exp(2 pi i q (n - c) / (u W))
                        const int nn = min(max(ns - 1 + b, 0), M - 1);
                        const double2 w0 = tw64[(q * x0) & (W - 1)];
                        const double2 w1 = POLS ? XpolS[(size_t)nn * NC + (q - rank * NC)] : __ldg(&p.Xpol[(size_t)nn * (W / 2) + q]);
                        return make_double2(w0.x * w1.x - w0.y * w1.y, w0.x * w1.y + w0.y * w1.x);
                    },
                    nyq, terms);
                double bv;
                int bk;  // candidate k = a*3+b is grid point (ms-1+a, ns-1+b); points outside the M x M grid do not compete
                {
                    const int mm = ms - 1 + lane / 3, nn = ns - 1 + lane % 3;
                    best9(mine, mm * M + nn, mm >= 0 && mm < M && nn >= 0 && nn < M, bv, bk);
                }
                const int ba = bk / 3, bb = bk % 3;
                up_peak = bv;
                if (ba == 1 && bb == 1) break;
                ms += ba - 1;
                ns += bb - 1;
                if (ba == 0) s2 = s1, s1 = s0, need = 1;
                else if (ba == 2) s0 = s1, s1 = s2, need = 4;
                else need = 0;
                __syncthreads();
            }
        }
        stamp(7, f);
        if (rank == 0 && tid == 0) {
            const double Em = p.ri_emean ? __ldcg(p.ri_emean) : p.Emean;
            emit(f, (float)((double)wy + (double)(ms - cM) / (double)u), (float)((double)wx + (double)(ns - cM) / (double)u),
                 (float)(p.peak_sign * (up_peak + ((double)*f00 + c0d * H * W) * Em)), wy, wx);
        }
        // this cluster's last frame of a plain launch goes straight to the exit (single-frame calls run this code from a
        // cold instruction cache: every taken branch to code not yet fetched costs ~250 cycles)
        if (__builtin_expect(!RT && !RI && f + ncl >= p.batch, true)) break;
        if (__builtin_expect(RI, false)) {
            __syncthreads();  // the reference mean was read before it is rewritten
            ri_update((long long)wy * u + (ms - cM), (long long)wx * u + (ns - cM));
        }
        __syncthreads();  // U (polish scratch) is reused by the next frame's raw ring
    }
    if (RT && total_tiles > 0) {  // the ring ran ahead: let the outstanding operand copies land before the CTA leaves
        for (int i = 0; i < NSTG; ++i) {
            mbar_wait(&bfull[c_slot], c_par);
            if (++c_slot == NSTG) c_slot = 0, c_par ^= 1u;
        }
    }
    csync_ctl();  // no CTA of the cluster exits while peers may still address its shared memory
    if constexpr (C::TC1) {
        if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
    }
    if (RT && rank == 0 && tid == 0) {
        *reinterpret_cast<volatile int *>(p.rt_alive) = 0;  // the session kernel is gone (quit or idle timeout)
        __threadfence_system();
    }
}

// ------------------------------------------------------------------ host-side launcher glue
template <class C>
struct Launcher {
    static size_t fixed_smem() { return C::FIXED_BYTES; }
    static int raw_scratch_bytes() { return C::RAWB + C::SCRB; }
    static cudaError_t prepare(int smem_bytes)
    {
        cudaError_t e = cudaFuncSetAttribute(cc_fused_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
        if (e != cudaSuccess) return e;
        if (C::CS > 8) e = cudaFuncSetAttribute(cc_fused_kernel<C>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        return e;
    }
    static void fill(cudaLaunchConfig_t &cfg, cudaLaunchAttribute *attr, int n_clusters, int smem_bytes, cudaStream_t st)
    {
        cfg = cudaLaunchConfig_t{};
        cfg.gridDim = dim3((unsigned)(n_clusters * C::CS), 1, 1);
        cfg.blockDim = dim3(C::NT, 1, 1);
        cfg.dynamicSmemBytes = (size_t)smem_bytes;
        cfg.stream = st;
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = C::CS;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
    }
    static cudaError_t max_clusters(int smem_bytes, int *n)
    {
        cudaLaunchConfig_t cfg;
        cudaLaunchAttribute attr[1];
        fill(cfg, attr, 1, smem_bytes, 0);
        return cudaOccupancyMaxActiveClusters(n, cc_fused_kernel<C>, &cfg);
    }
    static cudaError_t launch(const CcParams &p, int n_clusters, int smem_bytes, cudaStream_t st)
    {
        cudaLaunchConfig_t cfg;
        cudaLaunchAttribute attr[1];
        fill(cfg, attr, n_clusters, smem_bytes, st);
        return cudaLaunchKernelEx(&cfg, cc_fused_kernel<C>, p);
    }
    static CcVariant variant()
    {
        CcVariant v{};
        v.H = C::H, v.W = C::W, v.CS = C::CS, v.NT = C::NT, v.dtype = sizeof(typename C::PIX) == 1 ? 0 : 1;
        v.TM1 = C::TM1, v.TN1 = C::TN1, v.TM2 = C::TM2, v.TN2 = C::TN2;
        v.R1 = C::R1, v.Cn1 = C::Cn1, v.R2 = C::R2, v.Cn2 = C::Cn2, v.KS2 = C::KS2, v.BK1 = C::BK1, v.G2 = C::G2;
        v.KS1 = C::KS1;
        v.s_global = C::SG ? 1 : 0;
        v.NSTG = C::NSTG;
        v.lat = C::LAT ? 1 : 0;
        v.tc1 = C::TC1 ? 1 : 0;
        v.fixed_smem = &fixed_smem;
        v.raw_scratch_bytes = &raw_scratch_bytes;
        v.prepare = &prepare;
        v.max_clusters = &max_clusters;
        v.launch = &launch;
        return v;
    }
};

}  // namespace ccf

// cc_tc_probe.cu -- measured tensor-core experiment for step a6 (the upsampled DFT as matrix products, PAPER.md:L90,
// L163): one 128 x 128 x K product D = A B per CTA on the 5th-generation tensor cores (tcgen05.mma kind::tf32,
// accumulator in tensor memory), either as a single TF32 pass or as the three-pass split
//     A B ~= A_hi B_hi + A_lo B_hi + A_hi B_lo,   x_hi = x with the low 13 mantissa bits cleared, x_lo = x - x_hi (exact),
// which carries ~22 bits of each operand.  It is NOT on the decision path of cc_track: it
// measures what the two GEMM stages of the fused kernel would cost on the tensor cores and how far such a product is
// from the FP32 / float64 result, so that the trade can be judged with numbers.
//
// Shapes follow stage 1 of the 256 x 256 variant: M = 128 rows of the even/odd Dirichlet operand (80 used), N = 128
// spectrum floats of one CTA, K = the rows of Q (a multiple of 64 here).  Operands are staged in shared memory in the
// canonical no-swizzle UMMA layouts (both operands K-major: 8-row x 16-byte core matrices) by the CTA's threads, which
// is also where the hi/lo split of the data operand would happen inside the fused kernel.  (The MN-major form of the
// data operand, which would match the fused kernel's row-major spectrum block, produced all-zero products with
// kind::tf32 in a stand-alone check on this B200 / driver 580, so the data operand is transposed while staging.)
// Product code: shares nothing with oracle/.
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "../../include/cc_bench.h"

namespace {

constexpr int TM = 128, TN = 128, KT = 64, NTHR = 256;
constexpr uint32_t A_LBO = 128, A_SBO = (KT / 4) * 128;   // K-major: 16-byte K chunks adjacent, 8-row groups 2 KB apart
constexpr uint32_t B_LBO = 128, B_SBO = (KT / 4) * 128;   // B (N x K) K-major as well: kind::tf32 returned zeros for MN-major
                                                          // operands on this part (instruction-descriptor bits 15 / 16 set)
constexpr uint32_t TILE_BYTES = TM * KT * 4;              // 32 KB (A and B tiles have the same size)

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo)
{
    // start address, leading / stride byte offsets (all >> 4), descriptor version 1 (sm_100), no swizzle, base offset 0
    return (uint64_t)((saddr >> 4) & 0x3fffu) | ((uint64_t)((lbo >> 4) & 0x3fffu) << 16) | ((uint64_t)((sbo >> 4) & 0x3fffu) << 32) |
           (1ull << 46);
}
__device__ __forceinline__ void umma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}\n" ::"r"(d_tmem),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *b, uint32_t parity)
{
    uint32_t ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(ok)
                     : "r"(smem_u32(b)), "r"(parity)
                     : "memory");
    } while (!ok);
}
__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xffffe000u); }

// passes: 1 = single TF32 product, 3 = the three-pass split.  cyc[0] = cycles spent staging (load + split + layout),
// cyc[1] = cycles from the first tcgen05.mma to the completion of the last, per product, averaged over `iters`.
__global__ void __launch_bounds__(NTHR, 1) cc_tc_probe_kernel(const float *A, const float *B, int K, int passes, int iters, int repeat,
                                                            float *D, unsigned long long *cyc)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    float *Ahi = reinterpret_cast<float *>(smem), *Alo = Ahi + TM * KT, *Bhi = Alo + TM * KT, *Blo = Bhi + KT * TN;
    __shared__ uint64_t bar;
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;" ::"r"(smem_u32(&tmem_base_s)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&bar)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = tmem_base_s;
    // instruction descriptor: D = F32, A = B = TF32, both K-major, N = 128, M = 128
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(TN >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);
    uint32_t par = 0;
    long long c_stage = 0, c_mma = 0;
    const int ntile = K / KT;
    for (int it = 0; it < iters; ++it) {
        for (int t = 0; t < ntile; ++t) {
            const long long t0 = clock64();
            // stage tile t: A[m][t*KT + k] -> K-major core matrices, B[t*KT + k][n] -> MN-major core matrices, hi / lo parts
            for (int i = tid; i < TM * KT / 4; i += NTHR) {
                const int m = i / (KT / 4), k4 = i % (KT / 4);
                const float4 v = *reinterpret_cast<const float4 *>(A + (size_t)m * K + t * KT + k4 * 4);
                const float4 h = make_float4(tf32_hi(v.x), tf32_hi(v.y), tf32_hi(v.z), tf32_hi(v.w));
                const uint32_t off = (m / 8) * A_SBO + k4 * A_LBO + (m % 8) * 16;
                *reinterpret_cast<float4 *>(reinterpret_cast<unsigned char *>(Ahi) + off) = h;
                *reinterpret_cast<float4 *>(reinterpret_cast<unsigned char *>(Alo) + off) =
                    make_float4(tf32_hi(v.x - h.x), tf32_hi(v.y - h.y), tf32_hi(v.z - h.z), tf32_hi(v.w - h.w));
            }
            for (int i = tid; i < KT * TN / 4; i += NTHR) {
                const int k = i / (TN / 4), n4 = i % (TN / 4);
                const float4 v = *reinterpret_cast<const float4 *>(B + (size_t)(t * KT + k) * TN + n4 * 4);
                const float4 h = make_float4(tf32_hi(v.x), tf32_hi(v.y), tf32_hi(v.z), tf32_hi(v.w));
                const float hv[4] = {h.x, h.y, h.z, h.w};
                const float lv[4] = {tf32_hi(v.x - h.x), tf32_hi(v.y - h.y), tf32_hi(v.z - h.z), tf32_hi(v.w - h.w)};
#pragma unroll
                for (int j = 0; j < 4; ++j) {  // element (n, k) of the N x K operand
                    const int n = n4 * 4 + j;
                    const uint32_t off = (n / 8) * B_SBO + (k / 4) * B_LBO + (n % 8) * 16 + (k % 4) * 4;
                    *reinterpret_cast<float *>(reinterpret_cast<unsigned char *>(Bhi) + off) = hv[j];
                    *reinterpret_cast<float *>(reinterpret_cast<unsigned char *>(Blo) + off) = lv[j];
                }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy writes -> visible to the tensor core
            __syncthreads();
            const long long t1 = clock64();
            if (tid == 0) {
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t ah = smem_u32(Ahi), al = smem_u32(Alo), bh = smem_u32(Bhi), bl = smem_u32(Blo);
                for (int rep = 0; rep < repeat; ++rep)  // repeat > 1: the same tile again (D = repeat A B), for the issue rate
#pragma unroll
                for (int ks = 0; ks < KT / 8; ++ks) {  // UMMA K = 8 for TF32: two 16-byte K chunks of each operand
                    const uint32_t ao = ks * 2 * A_LBO, bo = ks * 2 * B_LBO;
                    if (passes == 3) {  // the small terms first
                        umma_tf32(tmem, umma_desc(al + ao, A_LBO, A_SBO), umma_desc(bh + bo, B_LBO, B_SBO), idesc, (t | ks | rep) != 0);
                        umma_tf32(tmem, umma_desc(ah + ao, A_LBO, A_SBO), umma_desc(bl + bo, B_LBO, B_SBO), idesc, 1u);
                        umma_tf32(tmem, umma_desc(ah + ao, A_LBO, A_SBO), umma_desc(bh + bo, B_LBO, B_SBO), idesc, 1u);
                    } else {
                        umma_tf32(tmem, umma_desc(ah + ao, A_LBO, A_SBO), umma_desc(bh + bo, B_LBO, B_SBO), idesc, (t | ks | rep) != 0);
                    }
                }
                // completion of every MMA issued so far arrives on the mbarrier (implies tcgen05.fence::before_thread_sync)
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&bar)) : "memory");
            }
            mbar_wait(&bar, par);  // the tile buffers may be overwritten, the accumulator is up to date
            par ^= 1u;
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const long long t2 = clock64();
            c_stage += t1 - t0, c_mma += t2 - t1;
        }
    }
    // epilogue: tensor memory -> registers -> global.  Warp w reads lanes 32 (w % 4) .. +32, columns 64 (w / 4) .. +64.
    {
        const int row = (warp % 4) * 32 + lane;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int col0 = (warp / 4) * 64 + h * 32;
            uint32_t r[32];
            const uint32_t taddr = tmem + ((uint32_t)((warp % 4) * 32) << 16) + (uint32_t)col0;
            asm volatile(
                "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, "
                "%18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
                  "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
                  "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]),
                  "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                : "r"(taddr)
                : "memory");
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (blockIdx.x == 0) {
#pragma unroll
                for (int j = 0; j < 32; ++j) D[(size_t)row * TN + col0 + j] = __uint_as_float(r[j]);
            }
        }
    }
    if (tid == 0 && blockIdx.x == 0) {
        cyc[0] = (unsigned long long)(c_stage / ((long long)iters)), cyc[1] = (unsigned long long)(c_mma / ((long long)iters));
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" ::"r"(tmem) : "memory");
}

}  // namespace

extern "C" cc_status cc_tc_gemm_probe(const float *A, const float *B, int K, int passes, int iters, int repeat, float *D,
                                      double *stage_cycles, double *mma_cycles)
{
    if (!A || !B || !D || K <= 0 || K % KT != 0 || (passes != 1 && passes != 3) || iters < 1 || repeat < 1) return CC_ERR_INVALID_ARG;
    int dev = 0, major = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return CC_ERR_ARCH;
    cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (major != 10) return CC_ERR_ARCH;
    float *dA = nullptr, *dB = nullptr, *dD = nullptr;
    unsigned long long *dc = nullptr;
    cudaError_t e = cudaMalloc((void **)&dA, (size_t)TM * K * 4);
    if (e == cudaSuccess) e = cudaMalloc((void **)&dB, (size_t)K * TN * 4);
    if (e == cudaSuccess) e = cudaMalloc((void **)&dD, (size_t)TM * TN * 4);
    if (e == cudaSuccess) e = cudaMalloc((void **)&dc, 16);
    if (e == cudaSuccess) e = cudaMemcpy(dA, A, (size_t)TM * K * 4, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(dB, B, (size_t)K * TN * 4, cudaMemcpyHostToDevice);
    const int smem = 4 * (int)TILE_BYTES + 1024;
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cc_tc_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e == cudaSuccess) {
        cc_tc_probe_kernel<<<sms, NTHR, smem>>>(dA, dB, K, passes, iters, repeat, dD, dc);  // every SM busy, as inside the fused kernel
        e = cudaDeviceSynchronize();
    }
    unsigned long long hc[2] = {0, 0};
    if (e == cudaSuccess) e = cudaMemcpy(D, dD, (size_t)TM * TN * 4, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(hc, dc, 16, cudaMemcpyDeviceToHost);
    cudaFree(dA), cudaFree(dB), cudaFree(dD), cudaFree(dc);
    if (e != cudaSuccess) return CC_ERR_CUDA;
    if (stage_cycles) *stage_cycles = (double)hc[0];
    if (mma_cycles) *mma_cycles = (double)hc[1];
    return CC_OK;
}

/*
 * cc_bench.h -- measurement aids of libcc_b200.so (same library as include/cc.h, separate header: none of these
 * is part of the tracking interface).  Used by bench.py and the GPU tests.
 */
#ifndef CC_BENCH_H
#define CC_BENCH_H

#include "cc.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * cc_track_latency_probe -- measurement aid for the real-time (batch-1)
 * mode of the paper (one displacement per camera frame):
 * n sequential calls of cc_track(batch = 1) on consecutive frames, each
 * followed by cudaStreamSynchronize, with the host monotonic clock read
 * around every call + synchronise pair.
 *   frames   DEVICE pointer, n frames (as for cc_track)
 *   dx,dy    DEVICE pointers, n float32 each (call i writes element i)
 *   peak     DEVICE pointer, n float32, or NULL
 *   lat_us   HOST pointer, receives n latencies in microseconds
 * Synchronises the stream.
 */
cc_status cc_track_latency_probe(const cc_plan *plan, const void *frames, int n,
                                 float *dx, float *dy, float *peak, double *lat_us, void *stream);

/*
 * cc_rt_latency_probe -- measurement aid: n sequential cc_rt_track calls on
 * consecutive frames with the host monotonic clock around each call.
 *   frames   n frames, DEVICE or pinned mapped HOST pointer
 *   dx,dy,peak  HOST pointers, n float32 each (peak may be NULL)
 *   lat_us   HOST pointer, n latencies in microseconds
 */
cc_status cc_rt_latency_probe(cc_rt *rt, const void *frames, int n, float *dx, float *dy, float *peak,
                              double *lat_us);

/*
 * cc_fp32_peak_probe -- measurement aid for bench.py's roofline: runs a
 * dependent-free FFMA loop on every SM and returns the achieved FP32 rate.
 *   tflops   HOST pointer, receives TFLOP/s (2 flop per FFMA)
 */
cc_status cc_fp32_peak_probe(double *tflops, void *stream);

/*
 * cc_fp32_tile_probe -- second measurement aid: an 8x8 register-tile loop of scalar FFMA with all three operands
 * in registers (the instruction mix of a classic register-tiled FP32 GEMM inner loop, no memory traffic).  It stays
 * well below the lane rate that cc_fp32_peak_probe's constant-operand loop reaches; the library's own GEMM loops
 * therefore use the packed fma.rn.f32x2 form.
 *   tflops   HOST pointer, receives TFLOP/s (2 flop per FFMA)
 */
cc_status cc_fp32_tile_probe(double *tflops, void *stream);

/*
 * cc_tc_gemm_probe -- measured tensor-core experiment for step a6 (the upsampled DFT as matrix products,
 * PAPER.md:L90; "the most computationally intensive component", L163).  Every SM computes the 128 x 128 x K product
 * D = A B with tcgen05.mma kind::tf32 (accumulator in tensor memory): passes = 1 a single TF32 product, passes = 3
 * the split A_hi B_hi + A_lo B_hi + A_hi B_lo that carries ~22 bits of each operand.  Not used by cc_track: the
 * decision path stays FP32 + float64; this call provides the numbers behind that choice.
 *   A        HOST pointer, 128 x K float32, row-major (the plan-constant operand, e.g. Dirichlet weights)
 *   B        HOST pointer, K x 128 float32, row-major (the data operand, e.g. rows of Q)
 *   K        multiple of 64
 *   repeat   >= 1: every staged K tile is multiplied `repeat` times (D = repeat * A B): the slope of mma_cycles
 *            against repeat is the issue-to-completion rate of the MMAs without the staging round trip
 *   D        HOST pointer, receives 128 x 128 float32, row-major
 *   stage_cycles, mma_cycles   HOST pointers (may be NULL): SM cycles per product spent staging the operands in
 *            shared memory (load, hi/lo split, UMMA core-matrix layout) and from the first tcgen05.mma to the
 *            completion of the last, averaged over `iters` repetitions with all SMs busy
 * Synchronises the device.  CC_ERR_INVALID_ARG / CC_ERR_ARCH / CC_ERR_CUDA.
 */
cc_status cc_tc_gemm_probe(const float *A, const float *B, int K, int passes, int iters, int repeat, float *D,
                           double *stage_cycles, double *mma_cycles);

#ifdef __cplusplus
}
#endif
#endif /* CC_BENCH_H */

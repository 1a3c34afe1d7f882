// cc_variant_list.h -- the compiled kernel variants (X-macro).
// CCV(name, H, W, CS, PIX, NT, TM1, TN1, TM2, TN2, SG, BK1, G2, R2, KS2, NSTG, PFD, KS1, TC)
//   CS  : CTAs per frame (thread-block cluster size)
//   TM1 x TN1 : per-thread tile of the stage-1 GEMM ([U|V] rows x spectrum floats)
//   TM2 x TN2 : per-thread tile of the stage-2 GEMM (T rows x offsets e; two accumulators E, O each)
//   SG  : spectrum block in global memory (L2) instead of shared memory
//   BK1 : stage-1 k-rows per staged tile;  G2 : stage-2 groups of 4 k-rows per staged tile
//   R2  : thread rows of stage 2;  KS2 : k-split of stage 2 (thread grid R2 x NT/(R2*KS2) x KS2)
//   NSTG, PFD : operand-ring depth (tiles, <= 8; all slots are kept in flight); PFD > 4 marks a small-batch (latency)
//               variant: a whole frame's tiles fit the ring, fp64 twiddles live in shared memory
//   KS1 : k-split of stage 1 (thread grid NT/(Cn1*KS1) x Cn1 x KS1); > 1 only where M is too small to fill the CTA
//   TC  : 1 = stage 1 of the upsampled DFT on the tensor cores (tcgen05.mma kind::tf32, three-pass hi/lo split, accumulators
//         in tensor memory; needs 2 * W/2/CS == 128 spectrum floats per CTA), 0 = FP32 register-tiled loop
// build.py compiles cc_variant.cu once per line.
CCV(f64_u16,        64,   64, 1, uint16_t, 256,  5, 8,  5, 5, false, 11, 16, 32,  1,  3,  2,  1, 0)
CCV(f64_u8,         64,   64, 1, uint8_t,  256,  5, 8,  5, 5, false, 11, 16, 32,  1,  3,  2,  1, 0)
CCV(f128_u8,       128,  128, 1, uint8_t,  256,  2, 8,  4, 4, false, 16,  8,  8,  8,  6,  4,  1, 0)
CCV(f128_u16,      128,  128, 1, uint16_t, 256,  2, 8,  4, 4, false, 16,  8,  8,  8,  6,  4,  1, 0)
CCV(f128_u8_c8,    128,  128, 8, uint8_t,  256,  2, 4,  1, 4, false, 68, 32,  8,  8,  8,  6,  4, 0)
CCV(f128_u16_c8,   128,  128, 8, uint16_t, 256,  2, 4,  1, 4, false, 68, 32,  8,  8,  8,  6,  4, 0)
CCV(f256_u16,      256,  256, 2, uint16_t, 256, 10, 8,  5, 5, false, 12,  4, 16,  1,  2,  2,  1, 1)
CCV(f256_u8,       256,  256, 2, uint8_t,  256, 10, 8,  5, 5, false, 12,  4, 16,  1,  2,  2,  1, 1)
CCV(f512_u16,      512,  512, 8, uint16_t, 256,  5, 4,  2, 5, false, 16,  8,  8,  4,  3,  2,  1, 0)
CCV(f512_u8,       512,  512, 8, uint8_t,  256,  5, 4,  2, 5, false, 16,  8,  8,  4,  3,  2,  1, 0)
CCV(f1024_u16,    1024, 1024, 8, uint16_t, 256, 10, 8,  5, 5, true,  16, 16,  4,  4,  3,  2,  1, 1)
CCV(f1024_u8,     1024, 1024, 8, uint8_t,  256, 10, 8,  5, 5, true,  16, 16,  4,  4,  3,  2,  1, 1)
// non-square camera formats of the paper's Table I; H = rows, W = columns
CCV(f128x256_u16,  128,  256, 1, uint16_t, 256, 10, 8,  5, 5, false, 12,  4, 16,  1,  2,  2,  1, 0)
CCV(f256x128_u16,  256,  128, 1, uint16_t, 256, 10, 8,  5, 5, false, 12,  4, 16,  1,  2,  2,  1, 0)
CCV(f256x512_u16,  256,  512, 4, uint16_t, 256, 10, 8,  5, 5, false, 12,  4, 16,  1,  2,  2,  1, 0)
CCV(f512x256_u16,  512,  256, 4, uint16_t, 256, 10, 4,  5, 5, false, 12,  4, 16,  1,  2,  2,  1, 0)
CCV(f128x1024_u16,  128, 1024, 8, uint16_t, 256, 10, 8,  5, 5, false, 12,  4, 16,  1,  2,  2,  1, 0)
CCV(f1024x128_u16, 1024,  128, 4, uint16_t, 256,  5, 4,  5, 5, false, 12,  4, 16,  1,  2,  2,  1, 0)
// 512x512 single-frame (latency) variant: one frame over a 16-CTA cluster (non-portable cluster size)
CCV(f512_u16_c16,  512,  512, 16, uint16_t, 256,  8, 4,  1, 5, false, 32, 16,  8,  4,  3,  2,  2, 0)
CCV(f512_u8_c16,   512,  512, 16, uint8_t,  256,  8, 4,  1, 5, false, 32, 16,  8,  4,  3,  2,  2, 0)
// 256x256 single-frame (latency) variants: one frame over a 16-CTA cluster (8 CTAs: 61 us per call at u = 128, 16: 46 us)
CCV(f256_u16_c16,  256,  256, 16, uint16_t, 256,  5, 4,  5, 5, false, 32, 16,  4,  4,  3,  2,  1, 0)
CCV(f256_u8_c16,   256,  256, 16, uint8_t,  256,  5, 4,  5, 5, false, 32, 16,  4,  4,  3,  2,  1, 0)
// non-square single-frame (latency) variants: one frame over a 16-CTA cluster (the paper's Table I is measured one
// image per call)
CCV(f256x512_u16_c16,  256,  512, 16, uint16_t, 256,  5, 4,  5, 5, false, 32, 16,  4,  4,  3,  2,  1, 0)
CCV(f512x256_u16_c16,  512,  256, 16, uint16_t, 256,  5, 4,  5, 5, false, 32, 16,  4,  4,  3,  2,  1, 0)
CCV(f128x1024_u16_c16, 128, 1024, 16, uint16_t, 256,  5, 4,  5, 5, false, 32, 16,  4,  4,  3,  2,  1, 0)
CCV(f128x256_u16_c16,  128,  256, 16, uint16_t, 256,  5, 4,  5, 5, false, 32, 16,  4,  4,  3,  2,  1, 0)
CCV(f256x128_u16_c16,  256,  128, 16, uint16_t, 256,  5, 4,  5, 5, false,  8, 16,  4,  4,  3,  2,  1, 0)
CCV(f1024x128_u16_c16, 1024, 128, 16, uint16_t, 256,  5, 4,  5, 5, false,  8, 16,  4,  4,  3,  2,  1, 0)
// 1024x1024 single-frame (latency) variant: one frame over a 16-CTA cluster
CCV(f1024_u16_c16, 1024, 1024, 16, uint16_t, 256, 10, 8,  5, 5, true,  16, 16,  4,  4,  3,  2,  1, 0)
CCV(f1024_u8_c16,  1024, 1024, 16, uint8_t,  256, 10, 8,  5, 5, true,  16, 16,  4,  4,  3,  2,  1, 0)

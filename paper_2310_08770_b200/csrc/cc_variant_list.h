// cc_variant_list.h -- the compiled kernel variants (X-macro).
// CCV(name, H, W, CS, PIX, NT, TM1, TN1, TM2, TN2, SG)
//   CS  : CTAs per frame (thread-block cluster size)
//   TM1 x TN1 : per-thread tile of the stage-1 GEMM (T = D * Q)
//   TM2 x TN2 : per-thread tile of the stage-2 GEMM (C = T * AxT)
//   SG  : spectrum block in global memory (L2) instead of shared memory
// build.py compiles cc_variant.cu once per line.
CCV(f64_u16,       64,   64, 1, uint16_t, 256,  5, 8, 10, 10, false)
CCV(f64_u8,        64,   64, 1, uint8_t,  256,  5, 8, 10, 10, false)
CCV(f128_u8,      128,  128, 1, uint8_t,  256,  2, 8,  2,  2, false)
CCV(f128_u16,     128,  128, 1, uint16_t, 256,  2, 8,  2,  2, false)
CCV(f128_u8_c8,   128,  128, 8, uint8_t,  256,  1, 4,  1,  1, false)
CCV(f128_u16_c8,  128,  128, 8, uint16_t, 256,  1, 4,  1,  1, false)
CCV(f256_u16,     256,  256, 2, uint16_t, 256, 10, 8,  5, 10, false)
CCV(f256_u8,      256,  256, 2, uint8_t,  256, 10, 8,  5, 10, false)
CCV(f512_u16,     512,  512, 8, uint16_t, 256,  5, 4,  1,  3, false)
CCV(f512_u8,      512,  512, 8, uint8_t,  256,  5, 4,  1,  3, false)
CCV(f1024_u16,   1024, 1024, 8, uint16_t, 256, 10, 8,  2, 10, true)
CCV(f1024_u8,    1024, 1024, 8, uint8_t,  256, 10, 8,  2, 10, true)

// cc_refupdate.h -- host interface of the CC-SN reference-image updates (cc_refupdate.cu); used by cc_api.cu only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

struct CcSnState;  // fp64 state G = F[E] of a CC-SN plan with a moving reference image (R19)

// the plan tables the fused kernel reads, rewritten after every update
struct CcSnTables {
    float2 *Gt;               // [H][W/2] conj(F[-1/(E+eps)]) / (HW), column-slot order
    float4 *ab;               // [H] packed DC / Nyquist columns
    double *emean;            // mean of the weight image
    const int16_t *col_freq;  // [H] signed row frequency of column-FFT slot p
};

cudaError_t cc_sn_state_create(CcSnState **out, int H, int W, int u, int dtype, double eps, const float *reference_host);
void cc_sn_state_destroy(CcSnState *s);
cudaError_t cc_sn_refresh_weight(CcSnState *s, const CcSnTables &t, cudaStream_t st);
cudaError_t cc_sn_update_eq9(CcSnState *s, const void *frame, const float *dy, const float *dx, double a0, const CcSnTables &t,
                             cudaStream_t st);
cudaError_t cc_sn_accumulate(CcSnState *s, const void *frames, int batch, const float *dy, const float *dx, cudaStream_t st);
cudaError_t cc_sn_finish_pass(CcSnState *s, long long count, const CcSnTables &t, cudaStream_t st);
cudaError_t cc_sn_read_state(CcSnState *s, double *out_re_im, int *status);

// cc_refupdate.cu -- reference-image updates of CC-SN plans (PAPER.md:L92 applied to Eqs. (8), (9); R19).
//
// Not on the per-frame hot path of the fixed-reference tracker: these kernels run between frames (Eq. (9)) or after
// a batch (Eq. (8)) and keep the plan's state -- the spectrum G = F[E] of the average raw image -- in fp64, so that
// the weight spectrum F[-1/(E + eps)] handed to the fused kernel is rounded to fp32 exactly once, like the one
// cc_plan_create builds on the host.  Plain radix-2 FFTs, one CTA per line.  Product code: shares nothing with oracle/.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <algorithm>
#include <vector>

#include "cc_refupdate.h"

namespace {

constexpr int FT = 256;  // threads per line FFT

// In-place complex FFT of `n` points (power of two <= 1024) on every line of a batch of H x W arrays.
// line l: array l / lines_per_array, line l % lines_per_array inside it; element i at base + i * stride_e.
// tw[j] = (cos, sin)(2 pi j / n); forward uses exp(-i theta), inverse exp(+i theta); no scaling.
__global__ void __launch_bounds__(FT) k_fft_lines(double2 *data, int n, long long stride_e, long long stride_l, int lines_per_array,
                                                  long long array_stride, int inverse, const double2 *tw)
{
    __shared__ double2 s[1024];
    const int l = blockIdx.x;
    double2 *base = data + (long long)(l / lines_per_array) * array_stride + (long long)(l % lines_per_array) * stride_l;
    int bits = 0;
    while ((1 << bits) < n) ++bits;
    for (int i = threadIdx.x; i < n; i += FT) s[__brev((unsigned)i) >> (32 - bits)] = base[(long long)i * stride_e];
    __syncthreads();
    for (int len = 2; len <= n; len <<= 1) {
        const int half = len >> 1, step = n / len;
        for (int t = threadIdx.x; t < n / 2; t += FT) {
            const int blk = t / half, k = t % half;
            const int i = blk * len + k, j = i + half;
            double2 w = tw[k * step];
            if (!inverse) w.y = -w.y;
            const double2 a = s[i], b = s[j];
            const double2 y = make_double2(b.x * w.x - b.y * w.y, b.x * w.y + b.y * w.x);
            s[i] = make_double2(a.x + y.x, a.y + y.y);
            s[j] = make_double2(a.x - y.x, a.y - y.y);
        }
        __syncthreads();
    }
    for (int i = threadIdx.x; i < n; i += FT) base[(long long)i * stride_e] = s[i];
}

template <typename PIX>
__global__ void k_pixels_to_complex(const PIX *frames, long long n, double2 *out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = make_double2((double)frames[i], 0.0);
}

// exp(+2 pi i f n / (u N)) for the signed frequency of bin k (cos(pi n / u) on the Nyquist bin: DESIGN.md R18)
__device__ __forceinline__ double2 shift_phase(int k, int N, long long n, int u)
{
    if (2 * k == N) {
        long long r = n % (2LL * u);
        if (r < 0) r += 2LL * u;
        return make_double2(cospi((double)r / (double)u), 0.0);
    }
    const long long f = 2 * k < N ? k : k - N, den = (long long)u * N;
    long long num = (f * n) % den;
    if (num < 0) num += den;
    double sn, cs;
    sincospi(2.0 * (double)num / (double)den, &sn, &cs);
    return make_double2(cs, sn);
}

// Eq. (9): G <- a0 F w(d) + (1 - a0) G, d = (dy, dx)[idx] read on the device (multiples of 1/u)
__global__ void k_blend(double2 *G, const double2 *F, int H, int W, int u, const float *dy, const float *dx, double a0)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= H * W) return;
    const int ky = i / W, kx = i % W;
    const long long ny = llrint((double)dy[0] * u), nx = llrint((double)dx[0] * u);
    const double2 wy = shift_phase(ky, H, ny, u), wx = shift_phase(kx, W, nx, u);
    const double2 w = make_double2(wy.x * wx.x - wy.y * wx.y, wy.x * wx.y + wy.y * wx.x);
    const double2 f = F[i], g = G[i];
    const double ar = f.x * w.x - f.y * w.y, ai = f.x * w.y + f.y * w.x;
    const double b1 = 1.0 - a0;
    G[i] = make_double2(a0 * ar + b1 * g.x, a0 * ai + b1 * g.y);
}

// Eq. (8): acc += sum over the nb frames of a chunk of F_b w(d_b), in frame order (deterministic)
__global__ void k_accumulate(double2 *acc, const double2 *F, int nb, int H, int W, int u, const float *dy, const float *dx)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= H * W) return;
    const int ky = i / W, kx = i % W;
    double2 a = acc[i];
    for (int b = 0; b < nb; ++b) {
        const long long ny = llrint((double)dy[b] * u), nx = llrint((double)dx[b] * u);
        const double2 wy = shift_phase(ky, H, ny, u), wx = shift_phase(kx, W, nx, u);
        const double2 w = make_double2(wy.x * wx.x - wy.y * wx.y, wy.x * wx.y + wy.y * wx.x);
        const double2 f = F[(long long)b * H * W + i];
        a.x += f.x * w.x - f.y * w.y;
        a.y += f.x * w.y + f.y * w.x;
    }
    acc[i] = a;
}

__global__ void k_scale_copy(double2 *dst, const double2 *src, int n, double scale)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = make_double2(src[i].x * scale, src[i].y * scale);
}

// T holds the unnormalised inverse transform of G: E = Re T / (HW); T <- -1 / (E + eps) (weight image of Eq. (7), R15)
__global__ void k_weight(double2 *T, int n, double inv_hw, double eps, int *status)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double ep = T[i].x * inv_hw + eps;
    if (!(ep > 0.0)) atomicExch(status, 1);  // reported by the next synchronising call (cc_plan_get_reference_spectrum)
    T[i] = make_double2(-1.0 / ep, 0.0);
}

// the fused kernel's tables from Gw = F[-1/(E + eps)]: conj(Gw)/(HW) by column-FFT slot, packed DC/Nyquist columns,
// mean of the weight image (DC add-back of `peak`); rounded to fp32 once
__global__ void k_pack_plan(const double2 *Gw, int H, int W, const int16_t *col_freq, float2 *Gt, float4 *ab, double *emean)
{
    const int Wh = W / 2;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const double inv = 1.0 / ((double)H * (double)W);
    if (i < H * Wh) {
        const int p = i / Wh, q = i % Wh;
        const int fy = col_freq[p], ky = fy < 0 ? fy + H : fy;
        if (q == 0) {
            Gt[i] = make_float2(0.f, 0.f);
            const double2 g0 = Gw[(long long)ky * W], gn = Gw[(long long)ky * W + Wh];
            ab[p] = make_float4(ky == 0 ? 0.f : (float)(g0.x * inv), ky == 0 ? 0.f : (float)(-g0.y * inv), (float)(gn.x * inv),
                                (float)(-gn.y * inv));
        } else {
            const double2 g = Gw[(long long)ky * W + q];
            Gt[i] = make_float2((float)(g.x * inv), (float)(-g.y * inv));
        }
    }
    if (i == 0) *emean = Gw[0].x * inv;
}

cudaError_t fft2(double2 *data, int nb, int H, int W, bool inverse, const double2 *twW, const double2 *twH, cudaStream_t st)
{
    const long long arr = (long long)H * W;
    k_fft_lines<<<nb * H, FT, 0, st>>>(data, W, 1, W, H, arr, inverse ? 1 : 0, twW);  // rows
    k_fft_lines<<<nb * W, FT, 0, st>>>(data, H, W, 1, W, arr, inverse ? 1 : 0, twH);  // columns
    return cudaGetLastError();
}

std::vector<double2> unit_roots_ld(int n)
{
    std::vector<double2> t(n);
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int j = 0; j < n; ++j) t[j] = make_double2((double)cosl(2.0L * pi * j / n), (double)sinl(2.0L * pi * j / n));
    return t;
}

}  // namespace

struct CcSnState {
    int H = 0, W = 0, u = 0, dtype = 0;
    double eps = 0.0;
    double2 *G = nullptr, *T = nullptr, *acc = nullptr, *twW = nullptr, *twH = nullptr;
    double2 *chunk = nullptr;
    int chunk_frames = 0;
    int *status = nullptr;
};

void cc_sn_state_destroy(CcSnState *s)
{
    if (!s) return;
    cudaFree(s->G), cudaFree(s->T), cudaFree(s->acc), cudaFree(s->twW), cudaFree(s->twH), cudaFree(s->chunk), cudaFree(s->status);
    delete s;
}

cudaError_t cc_sn_state_create(CcSnState **out, int H, int W, int u, int dtype, double eps, const float *reference_host)
{
    CcSnState *s = new CcSnState();
    s->H = H, s->W = W, s->u = u, s->dtype = dtype, s->eps = eps;
    const size_t n = (size_t)H * W;
    cudaError_t e = cudaMalloc((void **)&s->G, n * sizeof(double2));
    if (e == cudaSuccess) e = cudaMalloc((void **)&s->T, n * sizeof(double2));
    if (e == cudaSuccess) e = cudaMalloc((void **)&s->acc, n * sizeof(double2));
    if (e == cudaSuccess) e = cudaMemset(s->acc, 0, n * sizeof(double2));
    if (e == cudaSuccess) e = cudaMalloc((void **)&s->twW, W * sizeof(double2));
    if (e == cudaSuccess) e = cudaMalloc((void **)&s->twH, H * sizeof(double2));
    if (e == cudaSuccess) e = cudaMalloc((void **)&s->status, sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(s->status, 0, sizeof(int));
    if (e == cudaSuccess) {
        const auto tw = unit_roots_ld(W), th = unit_roots_ld(H);
        e = cudaMemcpy(s->twW, tw.data(), W * sizeof(double2), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(s->twH, th.data(), H * sizeof(double2), cudaMemcpyHostToDevice);
    }
    if (e == cudaSuccess) {  // G = F[E] of the caller's reference image
        std::vector<double2> E(n);
        for (size_t i = 0; i < n; ++i) E[i] = make_double2((double)reference_host[i], 0.0);
        e = cudaMemcpy(s->G, E.data(), n * sizeof(double2), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = fft2(s->G, 1, H, W, false, s->twW, s->twH, 0);
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
    }
    if (e != cudaSuccess) {
        cc_sn_state_destroy(s);
        return e;
    }
    *out = s;
    return cudaSuccess;
}

// G -> weight spectrum -> the fused kernel's tables
cudaError_t cc_sn_refresh_weight(CcSnState *s, const CcSnTables &t, cudaStream_t st)
{
    const int n = s->H * s->W, B = 256;
    k_scale_copy<<<(n + B - 1) / B, B, 0, st>>>(s->T, s->G, n, 1.0);
    cudaError_t e = fft2(s->T, 1, s->H, s->W, true, s->twW, s->twH, st);
    if (e != cudaSuccess) return e;
    k_weight<<<(n + B - 1) / B, B, 0, st>>>(s->T, n, 1.0 / ((double)s->H * (double)s->W), s->eps, s->status);
    e = fft2(s->T, 1, s->H, s->W, false, s->twW, s->twH, st);
    if (e != cudaSuccess) return e;
    const int m = s->H * (s->W / 2);
    k_pack_plan<<<(m + B - 1) / B, B, 0, st>>>(s->T, s->H, s->W, t.col_freq, t.Gt, t.ab, t.emean);
    return cudaGetLastError();
}

// Eq. (9) for one frame whose displacement the fused kernel has just written to dy[0], dx[0] (device)
cudaError_t cc_sn_update_eq9(CcSnState *s, const void *frame, const float *dy, const float *dx, double a0, const CcSnTables &t,
                             cudaStream_t st)
{
    const int n = s->H * s->W, B = 256;
    if (s->dtype == 0) k_pixels_to_complex<<<(n + B - 1) / B, B, 0, st>>>((const uint8_t *)frame, (long long)n, s->T);
    else k_pixels_to_complex<<<(n + B - 1) / B, B, 0, st>>>((const uint16_t *)frame, (long long)n, s->T);
    cudaError_t e = fft2(s->T, 1, s->H, s->W, false, s->twW, s->twH, st);
    if (e != cudaSuccess) return e;
    k_blend<<<(n + B - 1) / B, B, 0, st>>>(s->G, s->T, s->H, s->W, s->u, dy, dx, a0);
    return cc_sn_refresh_weight(s, t, st);
}

// Eq. (8): add the aligned raw spectra of `batch` frames (displacements on the device) to the accumulator
cudaError_t cc_sn_accumulate(CcSnState *s, const void *frames, int batch, const float *dy, const float *dx, cudaStream_t st)
{
    const long long n = (long long)s->H * s->W;
    const int want = (int)std::max<long long>(1, std::min<long long>(batch, (256LL << 20) / (n * (long long)sizeof(double2))));
    if (want > s->chunk_frames) {  // first use (or a larger batch): may synchronise
        cudaFree(s->chunk);
        s->chunk = nullptr, s->chunk_frames = 0;
        cudaError_t e = cudaMalloc((void **)&s->chunk, (size_t)want * n * sizeof(double2));
        if (e != cudaSuccess) return e;
        s->chunk_frames = want;
    }
    const int B = 256, px = s->dtype == 0 ? 1 : 2;
    for (int f0 = 0; f0 < batch; f0 += s->chunk_frames) {
        const int nb = std::min(s->chunk_frames, batch - f0);
        const long long tot = (long long)nb * n;
        const unsigned char *src = (const unsigned char *)frames + (size_t)f0 * n * px;
        if (s->dtype == 0) k_pixels_to_complex<<<(unsigned)((tot + B - 1) / B), B, 0, st>>>((const uint8_t *)src, tot, s->chunk);
        else k_pixels_to_complex<<<(unsigned)((tot + B - 1) / B), B, 0, st>>>((const uint16_t *)src, tot, s->chunk);
        cudaError_t e = fft2(s->chunk, nb, s->H, s->W, false, s->twW, s->twH, st);
        if (e != cudaSuccess) return e;
        k_accumulate<<<(unsigned)((n + B - 1) / B), B, 0, st>>>(s->acc, s->chunk, nb, s->H, s->W, s->u, dy + f0, dx + f0);
    }
    return cudaGetLastError();
}

// end of a pass of Eq. (8): G = acc / count, accumulator cleared, weight refreshed
cudaError_t cc_sn_finish_pass(CcSnState *s, long long count, const CcSnTables &t, cudaStream_t st)
{
    const int n = s->H * s->W, B = 256;
    k_scale_copy<<<(n + B - 1) / B, B, 0, st>>>(s->G, s->acc, n, 1.0 / (double)count);
    cudaError_t e = cudaMemsetAsync(s->acc, 0, (size_t)n * sizeof(double2), st);
    if (e != cudaSuccess) return e;
    return cc_sn_refresh_weight(s, t, st);
}

// host copy of the state G (H x W complex128, natural order) and of the sticky status flag; synchronises
cudaError_t cc_sn_read_state(CcSnState *s, double *out_re_im, int *status)
{
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess && out_re_im) e = cudaMemcpy(out_re_im, s->G, (size_t)s->H * s->W * sizeof(double2), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && status) e = cudaMemcpy(status, s->status, sizeof(int), cudaMemcpyDeviceToHost);
    return e;
}

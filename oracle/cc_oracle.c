/*
 * cc_oracle.c -- CPU ORACLE (TEST INFRASTRUCTURE, NOT A PRODUCT PATH).
 * See cc_oracle.h for the conventions and citations.  Plain C, double
 * precision, naive DFTs (no FFT), no blocking / fusion / reordering beyond
 * what the definitions state.  OpenMP is used only across frames (cco_track)
 * and across independent output rows of a single upsampled grid.
 */
#include "cc_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* cos/sin(2*pi*j/N), j = 0..N-1 */
static int unit_table(int N, double **c_out, double **s_out)
{
    double *c = (double *)malloc(sizeof(double) * (size_t)N);
    double *s = (double *)malloc(sizeof(double) * (size_t)N);
    if (!c || !s) { free(c); free(s); return -1; }
    for (int j = 0; j < N; ++j) {
        double a = 2.0 * M_PI * (double)j / (double)N;
        c[j] = cos(a);
        s[j] = sin(a);
    }
    *c_out = c; *s_out = s;
    return 0;
}

/* One pass of a naive DFT along one axis of a complex H x W array.
 * axis = 1: along x (rows), axis = 0: along y (columns).
 * sign = -1 forward, +1 inverse (no scaling here). */
static int dft_axis(const double *in_re, const double *in_im, int H, int W,
                    int axis, int sign, double *out_re, double *out_im)
{
    int N = axis ? W : H;
    double *c, *s;
    if (unit_table(N, &c, &s)) return -1;
    if (axis == 1) {
        for (int y = 0; y < H; ++y) {
            const double *xr = in_re + (size_t)y * W;
            const double *xi = in_im ? in_im + (size_t)y * W : NULL;
            for (int k = 0; k < W; ++k) {
                double ar = 0.0, ai = 0.0;
                int idx = 0;                       /* (k*n) mod N */
                for (int n = 0; n < W; ++n) {
                    double wr = c[idx], wi = sign * s[idx];
                    double vr = xr[n], vi = xi ? xi[n] : 0.0;
                    ar += vr * wr - vi * wi;
                    ai += vr * wi + vi * wr;
                    idx += k; if (idx >= N) idx -= N;
                }
                out_re[(size_t)y * W + k] = ar;
                out_im[(size_t)y * W + k] = ai;
            }
        }
    } else {
        for (int k = 0; k < H; ++k) {
            for (int x = 0; x < W; ++x) {
                double ar = 0.0, ai = 0.0;
                int idx = 0;
                for (int n = 0; n < H; ++n) {
                    double wr = c[idx], wi = sign * s[idx];
                    double vr = in_re[(size_t)n * W + x];
                    double vi = in_im ? in_im[(size_t)n * W + x] : 0.0;
                    ar += vr * wr - vi * wi;
                    ai += vr * wi + vi * wr;
                    idx += k; if (idx >= N) idx -= N;
                }
                out_re[(size_t)k * W + x] = ar;
                out_im[(size_t)k * W + x] = ai;
            }
        }
    }
    free(c); free(s);
    return 0;
}

int cco_dft2_real(const double *img, int H, int W, double *F_re, double *F_im)
{
    size_t n = (size_t)H * W;
    double *t_re = (double *)malloc(sizeof(double) * n);
    double *t_im = (double *)malloc(sizeof(double) * n);
    if (!t_re || !t_im) { free(t_re); free(t_im); return -1; }
    int rc = dft_axis(img, NULL, H, W, 1, -1, t_re, t_im);      /* rows    */
    if (!rc) rc = dft_axis(t_re, t_im, H, W, 0, -1, F_re, F_im); /* columns */
    free(t_re); free(t_im);
    return rc;
}

int cco_dft2_literal(const double *img, int H, int W, double *F_re, double *F_im)
{
    for (int ky = 0; ky < H; ++ky)
        for (int kx = 0; kx < W; ++kx) {
            double ar = 0.0, ai = 0.0;
            for (int y = 0; y < H; ++y)
                for (int x = 0; x < W; ++x) {
                    double a = -2.0 * M_PI * ((double)((long)ky * y % H) / H +
                                              (double)((long)kx * x % W) / W);
                    ar += img[(size_t)y * W + x] * cos(a);
                    ai += img[(size_t)y * W + x] * sin(a);
                }
            F_re[(size_t)ky * W + kx] = ar;
            F_im[(size_t)ky * W + kx] = ai;
        }
    return 0;
}

int cco_idft2(const double *P_re, const double *P_im, int H, int W,
              double *out_re, double *out_im)
{
    size_t n = (size_t)H * W;
    double *t_re = (double *)malloc(sizeof(double) * n);
    double *t_im = (double *)malloc(sizeof(double) * n);
    if (!t_re || !t_im) { free(t_re); free(t_im); return -1; }
    int rc = dft_axis(P_re, P_im, H, W, 0, +1, t_re, t_im);       /* columns */
    if (!rc) rc = dft_axis(t_re, t_im, H, W, 1, +1, out_re, out_im); /* rows */
    double inv = 1.0 / ((double)H * (double)W);
    for (size_t i = 0; i < n; ++i) { out_re[i] *= inv; out_im[i] *= inv; }
    free(t_re); free(t_im);
    return rc;
}

int cco_cc_direct(const double *I, const double *E, int H, int W, double *cc)
{
    for (int sy = 0; sy < H; ++sy)
        for (int sx = 0; sx < W; ++sx) {
            double acc = 0.0;
            for (int y = 0; y < H; ++y)
                for (int x = 0; x < W; ++x)
                    acc += I[(size_t)((y + sy) % H) * W + (x + sx) % W] *
                           E[(size_t)y * W + x];
            cc[(size_t)sy * W + sx] = acc;
        }
    return 0;
}

/* O3: P = F (x) conj(G) */
static void conj_product(const double *F_re, const double *F_im,
                         const double *G_re, const double *G_im, size_t n,
                         double *P_re, double *P_im)
{
    for (size_t i = 0; i < n; ++i) {
        P_re[i] = F_re[i] * G_re[i] + F_im[i] * G_im[i];
        P_im[i] = F_im[i] * G_re[i] - F_re[i] * G_im[i];
    }
}

int cco_cc_dft(const double *I, const double *E, int H, int W,
               double *cc, double *P_re, double *P_im)
{
    size_t n = (size_t)H * W;
    double *buf = (double *)malloc(sizeof(double) * n * 5);
    if (!buf) return -1;
    double *F_re = buf, *F_im = buf + n, *G_re = buf + 2 * n, *G_im = buf + 3 * n;
    double *c_im = buf + 4 * n;
    int rc = cco_dft2_real(I, H, W, F_re, F_im);
    if (!rc) rc = cco_dft2_real(E, H, W, G_re, G_im);
    if (!rc) {
        conj_product(F_re, F_im, G_re, G_im, n, P_re, P_im);
        rc = cco_idft2(P_re, P_im, H, W, cc, c_im);
    }
    free(buf);
    return rc;
}

long cco_argmax(const double *a, long n)
{
    long best = 0;
    for (long i = 1; i < n; ++i)
        if (a[i] > a[best]) best = i;      /* strict: smallest index on ties */
    return best;
}

int cco_grid_size(int u) { return (3 * u + 1) / 2; }   /* ceil(1.5 u) */

/* Interpolation row A[k] = exp(2*pi*i*f_N(k)*q/(u*N)), k = 0..N-1, for the
 * lag s = q/u (q integer): signed frequencies f_N(k) = k for k < N/2,
 * k - N above; for even N the Nyquist bin is split half/half between +N/2
 * and -N/2, i.e. A[N/2] = cos(pi*s).  Phases are reduced exactly: the
 * numerator f*q is an integer, taken mod (u*N) before cos/sin. */
static void interp_row(int N, int u, long q, double *a_re, double *a_im)
{
    long long den = (long long)u * N;
    for (int k = 0; k < N; ++k) {
        long long f = (2 * k < N) ? k : (long long)k - N;
        int nyq = (N % 2 == 0 && 2 * k == N);
        if (nyq) f = N / 2;
        long long num = (f * (long long)q) % den;
        if (num < 0) num += den;
        double ang = 2.0 * M_PI * (double)num / (double)den;
        a_re[k] = cos(ang);
        a_im[k] = nyq ? 0.0 : sin(ang);
    }
}

int cco_upsampled(const double *P_re, const double *P_im, int H, int W, int u,
                  int y0, int x0, double *C,
                  int *best_m, int *best_n, double *top1, double *top2)
{
    int M = cco_grid_size(u), c = M / 2;
    size_t mw = (size_t)M * W, mh = (size_t)M * H;
    double *Ay_re = (double *)malloc(sizeof(double) * mh);
    double *Ay_im = (double *)malloc(sizeof(double) * mh);
    double *Ax_re = (double *)malloc(sizeof(double) * mw);
    double *Ax_im = (double *)malloc(sizeof(double) * mw);
    double *T_re = (double *)malloc(sizeof(double) * mw);
    double *T_im = (double *)malloc(sizeof(double) * mw);
    double *r_t1 = (double *)malloc(sizeof(double) * M);
    double *r_t2 = (double *)malloc(sizeof(double) * M);
    int *r_n = (int *)malloc(sizeof(int) * M);
    if (!Ay_re || !Ay_im || !Ax_re || !Ax_im || !T_re || !T_im || !r_t1 || !r_t2 || !r_n) {
        free(Ay_re); free(Ay_im); free(Ax_re); free(Ax_im); free(T_re); free(T_im);
        free(r_t1); free(r_t2); free(r_n);
        return -1;
    }
    for (int m = 0; m < M; ++m) {
        interp_row(H, u, (long)y0 * u + (m - c), Ay_re + (size_t)m * H, Ay_im + (size_t)m * H);
        interp_row(W, u, (long)x0 * u + (m - c), Ax_re + (size_t)m * W, Ax_im + (size_t)m * W);
    }
    double inv = 1.0 / ((double)H * (double)W);
    /* T = A_y * P   (M x H times H x W) */
    #pragma omp parallel for schedule(static)
    for (int m = 0; m < M; ++m) {
        const double *ar = Ay_re + (size_t)m * H, *ai = Ay_im + (size_t)m * H;
        for (int kx = 0; kx < W; ++kx) {
            double sr = 0.0, si = 0.0;
            for (int ky = 0; ky < H; ++ky) {
                double pr = P_re[(size_t)ky * W + kx], pi = P_im[(size_t)ky * W + kx];
                sr += ar[ky] * pr - ai[ky] * pi;
                si += ar[ky] * pi + ai[ky] * pr;
            }
            T_re[(size_t)m * W + kx] = sr;
            T_im[(size_t)m * W + kx] = si;
        }
    }
    /* C = Re(T * A_x^T) / (H W)   (M x W times W x M), argmax per row */
    #pragma omp parallel for schedule(static)
    for (int m = 0; m < M; ++m) {
        const double *tr = T_re + (size_t)m * W, *ti = T_im + (size_t)m * W;
        double t1 = -INFINITY, t2 = -INFINITY; int bn = 0;
        for (int n = 0; n < M; ++n) {
            const double *ar = Ax_re + (size_t)n * W, *ai = Ax_im + (size_t)n * W;
            double sr = 0.0;
            for (int kx = 0; kx < W; ++kx) sr += tr[kx] * ar[kx] - ti[kx] * ai[kx];
            sr *= inv;
            if (C) C[(size_t)m * M + n] = sr;
            if (sr > t1) { t2 = t1; t1 = sr; bn = n; }
            else if (sr > t2) t2 = sr;
        }
        r_t1[m] = t1; r_t2[m] = t2; r_n[m] = bn;
    }
    double t1 = -INFINITY, t2 = -INFINITY; int bm = 0, bn = 0;
    for (int m = 0; m < M; ++m) {                 /* row-major order: strict > */
        if (r_t1[m] > t1) {
            if (t1 > t2) t2 = t1;
            if (r_t2[m] > t2) t2 = r_t2[m];
            t1 = r_t1[m]; bm = m; bn = r_n[m];
        } else {
            if (r_t1[m] > t2) t2 = r_t1[m];
        }
    }
    if (best_m) *best_m = bm;
    if (best_n) *best_n = bn;
    if (top1) *top1 = t1;
    if (top2) *top2 = t2;
    free(Ay_re); free(Ay_im); free(Ax_re); free(Ax_im); free(T_re); free(T_im);
    free(r_t1); free(r_t2); free(r_n);
    return 0;
}

int cco_upsampled_literal(const double *P_re, const double *P_im, int H, int W,
                          int u, int y0, int x0, double *C)
{
    int M = cco_grid_size(u), c = M / 2;
    double *ay_re = (double *)malloc(sizeof(double) * H), *ay_im = (double *)malloc(sizeof(double) * H);
    double *ax_re = (double *)malloc(sizeof(double) * W), *ax_im = (double *)malloc(sizeof(double) * W);
    if (!ay_re || !ay_im || !ax_re || !ax_im) { free(ay_re); free(ay_im); free(ax_re); free(ax_im); return -1; }
    double inv = 1.0 / ((double)H * (double)W);
    for (int m = 0; m < M; ++m)
        for (int n = 0; n < M; ++n) {
            interp_row(H, u, (long)y0 * u + (m - c), ay_re, ay_im);
            interp_row(W, u, (long)x0 * u + (n - c), ax_re, ax_im);
            double acc = 0.0;
            for (int ky = 0; ky < H; ++ky)
                for (int kx = 0; kx < W; ++kx) {
                    /* Re( P * Ay * Ax ) */
                    double wr = ay_re[ky] * ax_re[kx] - ay_im[ky] * ax_im[kx];
                    double wi = ay_re[ky] * ax_im[kx] + ay_im[ky] * ax_re[kx];
                    acc += P_re[(size_t)ky * W + kx] * wr - P_im[(size_t)ky * W + kx] * wi;
                }
            C[(size_t)m * M + n] = acc * inv;
        }
    free(ay_re); free(ay_im); free(ax_re); free(ax_im);
    return 0;
}

double cco_interp_at(const double *P_re, const double *P_im, int H, int W,
                     double sy, double sx)
{
    double acc = 0.0;
    for (int ky = 0; ky < H; ++ky) {
        double fy = (2 * ky < H) ? ky : (double)ky - H;
        int nyq_y = (H % 2 == 0 && 2 * ky == H);
        double ayr = cos(2.0 * M_PI * fy * sy / H);
        double ayi = nyq_y ? 0.0 : sin(2.0 * M_PI * fy * sy / H);
        for (int kx = 0; kx < W; ++kx) {
            double fx = (2 * kx < W) ? kx : (double)kx - W;
            int nyq_x = (W % 2 == 0 && 2 * kx == W);
            double axr = cos(2.0 * M_PI * fx * sx / W);
            double axi = nyq_x ? 0.0 : sin(2.0 * M_PI * fx * sx / W);
            double wr = ayr * axr - ayi * axi, wi = ayr * axi + ayi * axr;
            acc += P_re[(size_t)ky * W + kx] * wr - P_im[(size_t)ky * W + kx] * wi;
        }
    }
    return acc / ((double)H * (double)W);
}

/* two largest values of a[0..n): top1 at the smallest index attaining the
 * max, top2 the largest value at any other index */
static void top_two(const double *a, long n, long *i1, double *t1, double *t2)
{
    long b = cco_argmax(a, n);
    double s = -INFINITY;
    for (long i = 0; i < n; ++i)
        if (i != b && a[i] > s) s = a[i];
    *i1 = b; *t1 = a[b]; *t2 = s;
}

int cco_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* The whole path for CC-U (sn == 0; Eq. (4)) and CC-SN (sn != 0;
 * Eqs. (5)-(7)).  CC-SN: chi^2 of Eq. (6) is MINIMISED, and
 * the only term that depends on the displacement is
 *     S(s) = sum_r [I'(r+s)]^2 / E'(r),   I' = I + eps,  E' = E + eps
 * (Eq. (7); E estimates the average image, so the offset added to the images
 * is added to it too -- DESIGN.md R16).  The displacement is the position of
 * the minimum of S (the sentence before Eq. (7) says "maximum"; Eq. (6) and
 * Cauchy-Schwarz say minimum -- DESIGN.md R15).  argmin S = argmax (-S), so
 * the weighted image pair (I'^2, -1/E') goes through exactly the steps of
 * CC-U ("replacing I -> I'^2 and E -> 1/E") and `peak` is
 * reported as the minimised sum S. */
static int track_impl(const void *frames, int dtype, int batch, int H, int W, int u,
                      const float *reference, int sn, double eps, cco_result *out, int threads)
{
    if (!frames || !reference || !out || batch < 0 || H <= 0 || W <= 0 || u < 1 ||
        (dtype != 0 && dtype != 1))
        return -2;
    size_t n = (size_t)H * W;
    /* O1/O2 for the reference: E = (double) reference_f32, G = DFT2(E) */
    double *E = (double *)malloc(sizeof(double) * n * 3);
    if (!E) return -1;
    double *G_re = E + n, *G_im = E + 2 * n;
    for (size_t i = 0; i < n; ++i) E[i] = (double)reference[i];
    if (sn)
        for (size_t i = 0; i < n; ++i) E[i] = -1.0 / (E[i] + eps);   /* -(1/E'), Eq. (7) */
    if (cco_dft2_real(E, H, W, G_re, G_im)) { free(E); return -1; }

    int fail = 0;
#ifdef _OPENMP
    int nt = threads > 0 ? threads : omp_get_max_threads();
#else
    int nt = 1; (void)threads;
#endif
    #pragma omp parallel for schedule(dynamic) num_threads(nt)
    for (int b = 0; b < batch; ++b) {
        double *buf = (double *)malloc(sizeof(double) * n * 7);
        if (!buf) {
            #pragma omp atomic write
            fail = 1;
            continue;
        }
        double *I = buf, *F_re = buf + n, *F_im = buf + 2 * n, *P_re = buf + 3 * n,
               *P_im = buf + 4 * n, *cc = buf + 5 * n, *cc_im = buf + 6 * n;
        /* O1: pixels to double */
        if (dtype == 0) {
            const unsigned char *p = (const unsigned char *)frames + (size_t)b * n;
            for (size_t i = 0; i < n; ++i) I[i] = (double)p[i];
        } else {
            const unsigned short *p = (const unsigned short *)frames + (size_t)b * n;
            for (size_t i = 0; i < n; ++i) I[i] = (double)p[i];
        }
        if (sn)                                                       /* I'^2, Eq. (7) */
            for (size_t i = 0; i < n; ++i) I[i] = (I[i] + eps) * (I[i] + eps);
        int rc = cco_dft2_real(I, H, W, F_re, F_im);                 /* O2 */
        conj_product(F_re, F_im, G_re, G_im, n, P_re, P_im);          /* O3 */
        if (!rc) rc = cco_idft2(P_re, P_im, H, W, cc, cc_im);         /* O4 */
        cco_result r;
        memset(&r, 0, sizeof r);
        long idx;                                                     /* O5 */
        top_two(cc, (long)n, &idx, &r.cc_top1, &r.cc_top2);
        int y0 = (int)(idx / W), x0 = (int)(idx % W);
        r.wy = (2 * y0 >= H) ? y0 - H : y0;
        r.wx = (2 * x0 >= W) ? x0 - W : x0;
        if (u == 1) {
            r.dy = r.wy; r.dx = r.wx; r.peak = r.cc_top1;
            r.up_top1 = r.cc_top1; r.up_top2 = r.cc_top2;
        } else {
            int M = cco_grid_size(u), c = M / 2;                      /* O6 */
            if (!rc) rc = cco_upsampled(P_re, P_im, H, W, u, y0, x0, NULL,
                                        &r.m, &r.n, &r.up_top1, &r.up_top2);
            r.dy = (double)r.wy + (double)(r.m - c) / (double)u;      /* O7 */
            r.dx = (double)r.wx + (double)(r.n - c) / (double)u;
            r.peak = r.up_top1;
        }
        if (sn) {   /* report S = -(-S): the minimised sum and its runner-up */
            r.peak = -r.peak;
            r.cc_top1 = -r.cc_top1; r.cc_top2 = -r.cc_top2;
            r.up_top1 = -r.up_top1; r.up_top2 = -r.up_top2;
        }
        out[b] = r;
        if (rc) {
            #pragma omp atomic write
            fail = 1;
        }
        free(buf);
    }
    free(E);
    return fail ? -1 : 0;
}

int cco_track(const void *frames, int dtype, int batch, int H, int W, int u,
              const float *reference, cco_result *out, int threads)
{
    return track_impl(frames, dtype, batch, H, W, u, reference, 0, 0.0, out, threads);
}

int cco_track_sn(const void *frames, int dtype, int batch, int H, int W, int u,
                 const float *reference, double eps, cco_result *out, int threads)
{
    if (!(eps >= 0.0)) return -2;
    return track_impl(frames, dtype, batch, H, W, u, reference, 1, eps, out, threads);
}

/* Drift correction of the detected motion.
 * Plain (max_step <= 0), Eq. (10):      R_n = a0 r_n + b1 R_{n-1},  b1 = 1 - a0
 * Rate-limited (max_step = alpha/u), Eqs. (11)-(12):
 *     dR_n = a0 r_n + (b1 - 1) R_{n-1}
 *     R_n  = R_{n-1} + max_step * dR_n/|dR_n|   if |dR_n| > max_step,   else R_{n-1} + dR_n
 * Output r'_n = r_n - R_n.  R_{-1} = (0, 0) (so R_0 = a0 r_0 in the plain case, as the paper states);
 * state[2] = (Rx, Ry) carries R across calls. */
int cco_drift_correct(const float *dx, const float *dy, int n, double a0, double max_step,
                      double state[2], double *out_dx, double *out_dy)
{
    if (!dx || !dy || !state || !out_dx || !out_dy || n < 0 || !(a0 >= 0.0 && a0 <= 1.0)) return -2;
    const double b1 = 1.0 - a0;
    double Rx = state[0], Ry = state[1];
    for (int i = 0; i < n; ++i) {
        const double rx = (double)dx[i], ry = (double)dy[i];
        if (max_step > 0.0) {
            const double ex = a0 * rx + (b1 - 1.0) * Rx;      /* Eq. (11) */
            const double ey = a0 * ry + (b1 - 1.0) * Ry;
            const double norm = sqrt(ex * ex + ey * ey);
            if (norm > max_step) {                           /* Eq. (12), first case */
                Rx = Rx + max_step * (ex / norm);
                Ry = Ry + max_step * (ey / norm);
            } else {
                Rx = Rx + ex;
                Ry = Ry + ey;
            }
        } else {
            Rx = a0 * rx + b1 * Rx;                          /* Eq. (10) */
            Ry = a0 * ry + b1 * Ry;
        }
        out_dx[i] = rx - Rx;
        out_dy[i] = ry - Ry;
    }
    state[0] = Rx; state[1] = Ry;
    return 0;
}

/* ---- shared steps of the analyses with a moving reference image (Secs. III.A, III.B) ----
 *
 * measure_against_spectrum: steps O1-O7 for ONE frame against a reference given by its spectrum G = F[E]
 * (the paper holds the RI in Fourier space, Eqs. (8), (9)).  I: the frame's pixels as
 * doubles.  F (out): F[I].  work: 4*H*W doubles. */
static int measure_against_spectrum(const double *I, const double *G_re, const double *G_im, int H, int W, int u,
                                    double *F_re, double *F_im, double *work, cco_result *out)
{
    const size_t n = (size_t)H * W;
    double *P_re = work, *P_im = work + n, *cc = work + 2 * n, *cc_im = work + 3 * n;
    int rc = cco_dft2_real(I, H, W, F_re, F_im);                     /* O2 */
    conj_product(F_re, F_im, G_re, G_im, n, P_re, P_im);              /* O3 */
    if (!rc) rc = cco_idft2(P_re, P_im, H, W, cc, cc_im);             /* O4 */
    cco_result r;
    memset(&r, 0, sizeof r);
    long idx;                                                         /* O5 */
    top_two(cc, (long)n, &idx, &r.cc_top1, &r.cc_top2);
    int y0 = (int)(idx / W), x0 = (int)(idx % W);
    r.wy = (2 * y0 >= H) ? y0 - H : y0;
    r.wx = (2 * x0 >= W) ? x0 - W : x0;
    if (u == 1) {
        r.dy = r.wy; r.dx = r.wx; r.peak = r.cc_top1;
        r.up_top1 = r.cc_top1; r.up_top2 = r.cc_top2;
    } else {
        int M = cco_grid_size(u), c = M / 2;                          /* O6 */
        if (!rc) rc = cco_upsampled(P_re, P_im, H, W, u, y0, x0, NULL, &r.m, &r.n, &r.up_top1, &r.up_top2);
        r.dy = (double)r.wy + (double)(r.m - c) / (double)u;          /* O7 */
        r.dx = (double)r.wx + (double)(r.n - c) / (double)u;
        r.peak = r.up_top1;
    }
    *out = r;
    return rc;
}

/* align_spectrum: the spectrum of "I(r - r0)", the new image translated by its detected displacement so that it
 * lines up with the RI (Eq. (1); used in Eqs. (8), (9)).  With this build's sign (frame(r) ~
 * reference(r - d), R1) the aligned image is J(r) = I(r + d):
 *     F[J](k) = F[I](k) exp(+2 pi i (fy dy / H + fx dx / W)),   fy, fx the signed frequencies;
 * d is fractional, and on the Nyquist bins (even H, W) the real minimal-bandwidth interpolant multiplies by
 * cos(pi d) instead (R18). */
static void align_spectrum(const double *F_re, const double *F_im, int H, int W, double dy, double dx,
                           double *A_re, double *A_im)
{
    for (int ky = 0; ky < H; ++ky) {
        double wyr, wyi;
        if (H % 2 == 0 && 2 * ky == H) { wyr = cos(M_PI * dy); wyi = 0.0; }
        else {
            double fy = (2 * ky < H) ? ky : (double)ky - H;
            wyr = cos(2.0 * M_PI * fy * dy / H); wyi = sin(2.0 * M_PI * fy * dy / H);
        }
        for (int kx = 0; kx < W; ++kx) {
            double wxr, wxi;
            if (W % 2 == 0 && 2 * kx == W) { wxr = cos(M_PI * dx); wxi = 0.0; }
            else {
                double fx = (2 * kx < W) ? kx : (double)kx - W;
                wxr = cos(2.0 * M_PI * fx * dx / W); wxi = sin(2.0 * M_PI * fx * dx / W);
            }
            const double wr = wyr * wxr - wyi * wxi, wi = wyr * wxi + wyi * wxr;
            const size_t k = (size_t)ky * W + kx;
            A_re[k] = F_re[k] * wr - F_im[k] * wi;
            A_im[k] = F_re[k] * wi + F_im[k] * wr;
        }
    }
}

static void pixels_to_double(const void *frames, int dtype, size_t n, int b, double *I)
{
    if (dtype == 0) {
        const unsigned char *p = (const unsigned char *)frames + (size_t)b * n;
        for (size_t i = 0; i < n; ++i) I[i] = (double)p[i];
    } else {
        const unsigned short *p = (const unsigned short *)frames + (size_t)b * n;
        for (size_t i = 0; i < n; ++i) I[i] = (double)p[i];
    }
}

/* One step of Eq. (9) from a GIVEN reference spectrum: the frame is measured against G (O1-O7),
 * then Gn = a0 F[I aligned] + (1 - a0) G.  a0 = 1 returns the aligned spectrum itself -- one summand of Eq. (8)
 * (PAPER.md:L98); a0 = 0 leaves G unchanged.  CC-U.  Gn may be NULL. */
int cco_step_from_spectrum(const void *frame, int dtype, int H, int W, int u, const double *G_re, const double *G_im,
                           double a0, cco_result *out, double *Gn_re, double *Gn_im)
{
    if (!frame || !G_re || !G_im || !out || H <= 0 || W <= 0 || u < 1 || (dtype != 0 && dtype != 1) || !(a0 >= 0.0 && a0 <= 1.0))
        return -2;
    const size_t n = (size_t)H * W;
    double *buf = (double *)malloc(sizeof(double) * n * 9);
    if (!buf) return -1;
    double *I = buf, *F_re = buf + n, *F_im = buf + 2 * n, *A_re = buf + 3 * n, *A_im = buf + 4 * n, *work = buf + 5 * n;
    pixels_to_double(frame, dtype, n, 0, I);
    int rc = measure_against_spectrum(I, G_re, G_im, H, W, u, F_re, F_im, work, out);
    if (!rc && Gn_re && Gn_im) {
        align_spectrum(F_re, F_im, H, W, out->dy, out->dx, A_re, A_im);
        const double b1 = 1.0 - a0;
        for (size_t k = 0; k < n; ++k) {
            Gn_re[k] = a0 * A_re[k] + b1 * G_re[k];
            Gn_im[k] = a0 * A_im[k] + b1 * G_im[k];
        }
    }
    free(buf);
    return rc ? -1 : 0;
}

/* Real-time analysis with a running reference image, Eq. (9):
 *     F[E_i] = a0 F[I_i(r - r0)] + b1 F[E_{i-1}],   b1 = 1 - a0
 * (alignment: align_spectrum above).  Frames are processed strictly in order: frame i is measured against
 * E_{i-1} (the RI given by the caller is E_{-1}), then E_i is formed.  CC-U only.
 * G_re/G_im (H*W each, may be NULL) receive the spectrum of the last RI. */
int cco_track_rt(const void *frames, int dtype, int batch, int H, int W, int u,
                 const float *reference, double a0, cco_result *out, double *G_out_re, double *G_out_im)
{
    if (!frames || !reference || !out || batch < 0 || H <= 0 || W <= 0 || u < 1 || (dtype != 0 && dtype != 1) ||
        !(a0 >= 0.0 && a0 <= 1.0))
        return -2;
    const size_t n = (size_t)H * W;
    const double b1 = 1.0 - a0;
    double *buf = (double *)malloc(sizeof(double) * n * 12);
    if (!buf) return -1;
    double *E = buf, *G_re = buf + n, *G_im = buf + 2 * n, *I = buf + 3 * n, *F_re = buf + 4 * n, *F_im = buf + 5 * n,
           *A_re = buf + 6 * n, *A_im = buf + 7 * n, *work = buf + 8 * n;
    for (size_t i = 0; i < n; ++i) E[i] = (double)reference[i];
    int rc = cco_dft2_real(E, H, W, G_re, G_im);
    for (int b = 0; b < batch && !rc; ++b) {
        pixels_to_double(frames, dtype, n, b, I);
        rc = measure_against_spectrum(I, G_re, G_im, H, W, u, F_re, F_im, work, &out[b]);
        align_spectrum(F_re, F_im, H, W, out[b].dy, out[b].dx, A_re, A_im);
        for (size_t k = 0; k < n; ++k) {                 /* Eq. (9) */
            G_re[k] = a0 * A_re[k] + b1 * G_re[k];
            G_im[k] = a0 * A_im[k] + b1 * G_im[k];
        }
    }
    if (!rc && G_out_re && G_out_im) {
        memcpy(G_out_re, G_re, sizeof(double) * n);
        memcpy(G_out_im, G_im, sizeof(double) * n);
    }
    free(buf);
    return rc ? -1 : 0;
}

/* Offline analysis, Eq. (8): for each complete pass through the images,
 *     F[E_n] = (1/N) sum_i F[I_i(r - r0_i)],
 * every displacement r0_i of the pass being measured against the constant RI E_{n-1} (alignment: align_spectrum
 * above).  n_iter passes are made, starting from the caller's reference (the paper starts from E_0 = I_0: pass the
 * first frame).  `out` receives the displacements measured in the LAST pass (against E_{n_iter-1}), G_out the
 * spectrum of E_{n_iter}.  CC-U.  Sequential. */
int cco_iterate_reference(const void *frames, int dtype, int batch, int H, int W, int u, const float *reference,
                          int n_iter, cco_result *out, double *G_out_re, double *G_out_im)
{
    if (!frames || !reference || !out || batch <= 0 || H <= 0 || W <= 0 || u < 1 || (dtype != 0 && dtype != 1) || n_iter < 1)
        return -2;
    const size_t n = (size_t)H * W;
    double *buf = (double *)malloc(sizeof(double) * n * 14);
    if (!buf) return -1;
    double *E = buf, *G_re = buf + n, *G_im = buf + 2 * n, *I = buf + 3 * n, *F_re = buf + 4 * n, *F_im = buf + 5 * n,
           *A_re = buf + 6 * n, *A_im = buf + 7 * n, *S_re = buf + 8 * n, *S_im = buf + 9 * n, *work = buf + 10 * n;
    for (size_t i = 0; i < n; ++i) E[i] = (double)reference[i];
    int rc = cco_dft2_real(E, H, W, G_re, G_im);
    for (int it = 0; it < n_iter && !rc; ++it) {
        for (size_t i = 0; i < n; ++i) S_re[i] = S_im[i] = 0.0;
        for (int b = 0; b < batch && !rc; ++b) {
            pixels_to_double(frames, dtype, n, b, I);
            rc = measure_against_spectrum(I, G_re, G_im, H, W, u, F_re, F_im, work, &out[b]);
            align_spectrum(F_re, F_im, H, W, out[b].dy, out[b].dx, A_re, A_im);
            for (size_t k = 0; k < n; ++k) { S_re[k] += A_re[k]; S_im[k] += A_im[k]; }
        }
        for (size_t i = 0; i < n; ++i) { G_re[i] = S_re[i] / batch; G_im[i] = S_im[i] / batch; }   /* Eq. (8) */
    }
    if (!rc && G_out_re && G_out_im) {
        memcpy(G_out_re, G_re, sizeof(double) * n);
        memcpy(G_out_im, G_im, sizeof(double) * n);
    }
    free(buf);
    return rc ? -1 : 0;
}

/* ---- CC-SN with a moving reference image (R19) -------------------------------------------------------
 * the discussion of Secs. III.A/III.B "can be easily adapted for the CC-SN method by replacing
 * I_i -> I_i'^2 and E_n -> 1/E_n".  Substituted literally into Eqs. (8)/(9) this would average I'^2 into "1/E",
 * which is neither the reciprocal of an image average nor dimensionally consistent with Eq. (7).  Reading taken:
 * the replacement applies to the CORRELATION (Eq. (7) instead of Eq. (4)), while the RI keeps the meaning Eq. (5)
 * gives it -- the estimate of the average image ("see Sec. III for how this [the offset] affects the RI",
 * the RI is built from the offset images I' = I + eps).  So the state is F[E'], updated by Eqs. (8)/(9)
 * from the ALIGNED OFFSET IMAGES I_i', and every frame is measured by Eq. (7) with the weight 1/E' of the current
 * state.  Because the alignment leaves the DC bin untouched and a0 + b1 = 1 (and a mean has weights summing to 1),
 * E'_i = E_i + eps exactly, E_i being the same filter on the raw images: the state is held as G = F[E] and
 * the offset is added when the weight is formed. */

/* Gw = F[-1/(E + eps)] from the state G = F[E]  (E = Re F^-1[G]); fails (-3) unless E + eps > 0 everywhere.
 * work: 3*H*W doubles. */
static int sn_weight_spectrum(const double *G_re, const double *G_im, int H, int W, double eps,
                              double *Gw_re, double *Gw_im, double *work)
{
    const size_t n = (size_t)H * W;
    double *e_re = work, *e_im = work + n, *w = work + 2 * n;
    if (cco_idft2(G_re, G_im, H, W, e_re, e_im)) return -1;
    for (size_t i = 0; i < n; ++i) {
        const double ep = e_re[i] + eps;
        if (!(ep > 0.0)) return -3;
        w[i] = -1.0 / ep;                                   /* -(1/E'), Eq. (7); minimum of S = maximum of -S (R15) */
    }
    return cco_dft2_real(w, H, W, Gw_re, Gw_im);
}

/* One frame by Eq. (7) against the state G = F[E]; F (out) = F[I] of the RAW frame (what Eqs. (8)/(9) align).
 * work: 9*H*W doubles. */
static int measure_sn_against_state(const double *I, const double *G_re, const double *G_im, int H, int W, int u, double eps,
                                    double *F_re, double *F_im, double *work, cco_result *out)
{
    const size_t n = (size_t)H * W;
    double *Gw_re = work, *Gw_im = work + n, *I2 = work + 2 * n, *F2_re = work + 3 * n, *F2_im = work + 4 * n, *w2 = work + 5 * n;
    int rc = sn_weight_spectrum(G_re, G_im, H, W, eps, Gw_re, Gw_im, w2);
    if (rc) return rc;
    for (size_t i = 0; i < n; ++i) I2[i] = (I[i] + eps) * (I[i] + eps);        /* I'^2, Eq. (7) */
    rc = measure_against_spectrum(I2, Gw_re, Gw_im, H, W, u, F2_re, F2_im, w2, out);
    out->peak = -out->peak;                                  /* report S, as cco_track_sn does */
    out->cc_top1 = -out->cc_top1; out->cc_top2 = -out->cc_top2;
    out->up_top1 = -out->up_top1; out->up_top2 = -out->up_top2;
    if (!rc) rc = cco_dft2_real(I, H, W, F_re, F_im);
    return rc;
}

int cco_step_from_spectrum_sn(const void *frame, int dtype, int H, int W, int u, const double *G_re, const double *G_im,
                              double eps, double a0, cco_result *out, double *Gn_re, double *Gn_im)
{
    if (!frame || !G_re || !G_im || !out || H <= 0 || W <= 0 || u < 1 || (dtype != 0 && dtype != 1) || !(a0 >= 0.0 && a0 <= 1.0) ||
        !(eps >= 0.0))
        return -2;
    const size_t n = (size_t)H * W;
    double *buf = (double *)malloc(sizeof(double) * n * 14);
    if (!buf) return -1;
    double *I = buf, *F_re = buf + n, *F_im = buf + 2 * n, *A_re = buf + 3 * n, *A_im = buf + 4 * n, *work = buf + 5 * n;
    pixels_to_double(frame, dtype, n, 0, I);
    int rc = measure_sn_against_state(I, G_re, G_im, H, W, u, eps, F_re, F_im, work, out);
    if (!rc && Gn_re && Gn_im) {
        align_spectrum(F_re, F_im, H, W, out->dy, out->dx, A_re, A_im);
        const double b1 = 1.0 - a0;
        for (size_t k = 0; k < n; ++k) {
            Gn_re[k] = a0 * A_re[k] + b1 * G_re[k];
            Gn_im[k] = a0 * A_im[k] + b1 * G_im[k];
        }
    }
    free(buf);
    return rc == -3 ? -3 : (rc ? -1 : 0);
}

int cco_track_rt_sn(const void *frames, int dtype, int batch, int H, int W, int u, const float *reference, double eps,
                    double a0, cco_result *out, double *G_out_re, double *G_out_im)
{
    if (!frames || !reference || !out || batch < 0 || H <= 0 || W <= 0 || u < 1 || (dtype != 0 && dtype != 1) ||
        !(a0 >= 0.0 && a0 <= 1.0) || !(eps >= 0.0))
        return -2;
    const size_t n = (size_t)H * W;
    const double b1 = 1.0 - a0;
    double *buf = (double *)malloc(sizeof(double) * n * 17);
    if (!buf) return -1;
    double *E = buf, *G_re = buf + n, *G_im = buf + 2 * n, *I = buf + 3 * n, *F_re = buf + 4 * n, *F_im = buf + 5 * n,
           *A_re = buf + 6 * n, *A_im = buf + 7 * n, *work = buf + 8 * n;
    for (size_t i = 0; i < n; ++i) E[i] = (double)reference[i];
    int rc = cco_dft2_real(E, H, W, G_re, G_im);
    for (int b = 0; b < batch && !rc; ++b) {
        pixels_to_double(frames, dtype, n, b, I);
        rc = measure_sn_against_state(I, G_re, G_im, H, W, u, eps, F_re, F_im, work, &out[b]);
        if (rc) break;
        align_spectrum(F_re, F_im, H, W, out[b].dy, out[b].dx, A_re, A_im);
        for (size_t k = 0; k < n; ++k) {                 /* Eq. (9) on the raw images; E' = E + eps (see above) */
            G_re[k] = a0 * A_re[k] + b1 * G_re[k];
            G_im[k] = a0 * A_im[k] + b1 * G_im[k];
        }
    }
    if (!rc && G_out_re && G_out_im) {
        memcpy(G_out_re, G_re, sizeof(double) * n);
        memcpy(G_out_im, G_im, sizeof(double) * n);
    }
    free(buf);
    return rc == -3 ? -3 : (rc ? -1 : 0);
}

int cco_iterate_reference_sn(const void *frames, int dtype, int batch, int H, int W, int u, const float *reference,
                             double eps, int n_iter, cco_result *out, double *G_out_re, double *G_out_im)
{
    if (!frames || !reference || !out || batch <= 0 || H <= 0 || W <= 0 || u < 1 || (dtype != 0 && dtype != 1) || n_iter < 1 ||
        !(eps >= 0.0))
        return -2;
    const size_t n = (size_t)H * W;
    double *buf = (double *)malloc(sizeof(double) * n * 19);
    if (!buf) return -1;
    double *E = buf, *G_re = buf + n, *G_im = buf + 2 * n, *I = buf + 3 * n, *F_re = buf + 4 * n, *F_im = buf + 5 * n,
           *A_re = buf + 6 * n, *A_im = buf + 7 * n, *S_re = buf + 8 * n, *S_im = buf + 9 * n, *work = buf + 10 * n;
    for (size_t i = 0; i < n; ++i) E[i] = (double)reference[i];
    int rc = cco_dft2_real(E, H, W, G_re, G_im);
    for (int it = 0; it < n_iter && !rc; ++it) {
        for (size_t i = 0; i < n; ++i) S_re[i] = S_im[i] = 0.0;
        for (int b = 0; b < batch && !rc; ++b) {
            pixels_to_double(frames, dtype, n, b, I);
            rc = measure_sn_against_state(I, G_re, G_im, H, W, u, eps, F_re, F_im, work, &out[b]);
            if (rc) break;
            align_spectrum(F_re, F_im, H, W, out[b].dy, out[b].dx, A_re, A_im);
            for (size_t k = 0; k < n; ++k) { S_re[k] += A_re[k]; S_im[k] += A_im[k]; }
        }
        if (rc) break;
        for (size_t i = 0; i < n; ++i) { G_re[i] = S_re[i] / batch; G_im[i] = S_im[i] / batch; }   /* Eq. (8) */
    }
    if (!rc && G_out_re && G_out_im) {
        memcpy(G_out_re, G_re, sizeof(double) * n);
        memcpy(G_out_im, G_im, sizeof(double) * n);
    }
    free(buf);
    return rc == -3 ? -3 : (rc ? -1 : 0);
}

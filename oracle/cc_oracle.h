/*
 * cc_oracle.h -- CPU ORACLE (TEST INFRASTRUCTURE, NOT A PRODUCT PATH).
 *
 * Plain, slow, double-precision restatement of the per-frame displacement
 * estimator of Werneck et al. (arxiv 2310.08770): cross-correlation through
 * the Fourier domain (Eq. (4)), integer peak and upsampled
 * sub-pixel peak (Sec. III).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code, header, table or
 * constant with the CUDA library under paper_2310_08770_b200/csrc.
 *
 * Conventions (DESIGN.md "Readings of the paper" R1-R9):
 *   images are row-major [y][x]; DFT sign exp(-2*pi*i*k*n/N) forward;
 *   cc(s) = sum_r I(r+s) E(r) = IDFT2[ DFT2[I] * conj(DFT2[E]) ](s)   (Eq. 4)
 *   displacement d = the lag s that maximises cc (frame(r) ~ reference(r-d));
 *   ties: smallest row-major index; wrap p >= N/2 -> p-N;
 *   upsampled grid: M = ceil(1.5*u) points per axis, spacing 1/u, offsets
 *   (m - floor(M/2))/u around the integer peak; Nyquist bins (even N) are
 *   split half/half between +N/2 and -N/2 (the real, minimal-bandwidth
 *   trigonometric interpolant).
 *
 * Parity pins: every function below is pinned by tests/test_oracle_pins.py
 * (P0-P11, SN1-5, D1-3, RI1-3, IT1-3, ST1, SR1-6); nothing here is
 * "parity unpinned".
 */
#ifndef CC_ORACLE_H
#define CC_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

/* O2: separable naive 2D DFT of a real H x W image (row pass then column
 * pass, twiddles from a cos/sin table indexed by (k*n) mod N).  Full complex
 * H x W output, no Hermitian shortcuts.  `F[.]` in Eq. (4). */
int cco_dft2_real(const double *img, int H, int W, double *F_re, double *F_im);

/* O2 (tiny frames): the literal O(H^2 W^2) double sum of the 2D DFT. */
int cco_dft2_literal(const double *img, int H, int W, double *F_re, double *F_im);

/* O4: separable naive inverse 2D DFT with the 1/(HW) factor; complex in,
 * complex out (the imaginary part of a correlation of real images is
 * rounding noise and is returned so tests can check that).  PAPER.md:L68. */
int cco_idft2(const double *P_re, const double *P_im, int H, int W,
              double *out_re, double *out_im);

/* Left-hand side of Eq. (4), by brute force:
 * cc[s] = sum_r I[(r+s) mod (H,W)] * E[r]      -- O(H^2 W^2). */
int cco_cc_direct(const double *I, const double *E, int H, int W, double *cc);

/* Right-hand side of Eq. (4): P = F[I] (x) conj(F[E]) (O3), cc = Re IDFT2[P]
 * (O4).  P_re/P_im (H*W each) receive the element-wise product. */
int cco_cc_dft(const double *I, const double *E, int H, int W,
               double *cc, double *P_re, double *P_im);

/* O5/O7: smallest linear index attaining the maximum of a[0..n). */
long cco_argmax(const double *a, long n);

/* Number of upsampled samples per axis: M = ceil(1.5*u)
 * ("1.5u points"; u = 256 -> 384). */
int cco_grid_size(int u);

/* O6: upsampled cross-correlation on the M x M grid around integer peak
 * (y0, x0), evaluated as A_y * P * A_x^T ("interpolated into the upsampled
 * region, followed by an inverse discrete Fourier transform").
 * C may be NULL (then only the argmax outputs are produced).
 * best_m/best_n: smallest row-major index attaining the maximum; top1 its
 * value; top2 the largest value at any other grid index. */
int cco_upsampled(const double *P_re, const double *P_im, int H, int W, int u,
                  int y0, int x0, double *C,
                  int *best_m, int *best_n, double *top1, double *top2);

/* O6 unfactored: the O(M^2 H W) double sum, for tiny inputs (pin P9). */
int cco_upsampled_literal(const double *P_re, const double *P_im, int H, int W,
                          int u, int y0, int x0, double *C);

/* One upsampled value at an arbitrary real lag (sy, sx): the band-limited
 * interpolant of cc evaluated from P by its defining sum.  Used by pins. */
double cco_interp_at(const double *P_re, const double *P_im, int H, int W,
                     double sy, double sx);

/* Result of the whole path for one frame. */
typedef struct {
    double dy, dx;      /* displacement in pixels (O7)                        */
    double peak;        /* upsampled correlation value at the maximum         */
    int    wy, wx;      /* wrapped integer peak (O5)                          */
    int    m, n;        /* grid indices of the sub-pixel maximum              */
    double cc_top1, cc_top2;   /* two largest values of the integer CC       */
    double up_top1, up_top2;   /* two largest values of the upsampled CC     */
} cco_result;

/* The whole path O1-O7 for `batch` frames against one reference.
 * dtype: 0 = uint8 pixels, 1 = uint16 pixels.  reference: float32 H*W
 * (the same 32-bit values the GPU plan receives).  u == 1 -> integer peak
 * only.  OpenMP across frames only (threads <= 0 -> library default).
 * Returns 0 on success. */
int cco_track(const void *frames, int dtype, int batch, int H, int W, int u,
              const float *reference, cco_result *out, int threads);

/* The same path for the shot-noise-weighted method CC-SN (PAPER.md:L72-84,
 * Eqs. (5)-(7); L92 "replacing I -> I'^2 and E -> 1/E"): the displacement is
 * the position of the MINIMUM of S(s) = sum_r (I(r+s)+eps)^2 / (E(r)+eps)
 * (R15, R16), first on the integer lags, then on the upsampled
 * grid; `peak`, cc_top1/2 and up_top1/2 are values of S (top1 = minimum,
 * top2 = smallest value at any other index).  eps >= 0; E + eps must be > 0. */
int cco_track_sn(const void *frames, int dtype, int batch, int H, int W, int u,
                 const float *reference, double eps, cco_result *out, int threads);

/* Drift correction: r'_n = r_n - R_n with the low-pass offset R_n of Eq. (10)
 * (max_step <= 0) or its rate-limited form, Eqs. (11)-(12), with max_step = alpha/u.  b1 = 1 - a0,
 * R_{-1} = 0; state[2] = (Rx, Ry) in/out.  Garbling: Eq. (12) prints "d\hat{R}_n" for the unit vector
 * dR_n/|dR_n| (R14).  Returns 0 on success. */
int cco_drift_correct(const float *dx, const float *dy, int n, double a0, double max_step,
                      double state[2], double *out_dx, double *out_dy);

/* Real-time analysis, Eq. (9): frames in order, frame i measured against the running RI
 * E_{i-1} (reference = E_{-1}), then F[E_i] = a0 F[I_i aligned] + (1 - a0) F[E_{i-1}], the aligned image being
 * I_i(r + d_i) by the Fourier shift theorem (cos(pi d) on the Nyquist bins; R18).  CC-U.  G_out_re/im
 * (H*W each, may be NULL): spectrum of the last RI.  Sequential (no OpenMP). */
int cco_track_rt(const void *frames, int dtype, int batch, int H, int W, int u,
                 const float *reference, double a0, cco_result *out, double *G_out_re, double *G_out_im);

/* Offline analysis, Eq. (8): n_iter complete passes; in each, every frame is measured against the
 * constant RI of the previous pass and the new RI is the mean of the aligned images, F[E_n] = (1/N) sum_i
 * F[I_i(r + d_i)] (alignment as in cco_track_rt).  out: displacements of the last pass; G_out: spectrum of E_{n_iter}. */
int cco_iterate_reference(const void *frames, int dtype, int batch, int H, int W, int u, const float *reference,
                          int n_iter, cco_result *out, double *G_out_re, double *G_out_im);

/* One step of Eq. (9) from a GIVEN reference spectrum G = F[E] (H*W complex, full spectrum): O1-O7 of `frame`
 * against G, then Gn = a0 F[frame aligned] + (1 - a0) G.  a0 = 1: Gn is the aligned spectrum itself, one summand of
 * Eq. (8).  Lets a test drive the oracle from the state another implementation holds (input only).  CC-U.
 * Shares its two steps (measure against a spectrum; align by the Fourier shift theorem) with cco_track_rt and
 * cco_iterate_reference, so the pins of either function pin all three. */
int cco_step_from_spectrum(const void *frame, int dtype, int H, int W, int u, const double *G_re, const double *G_im,
                           double a0, cco_result *out, double *Gn_re, double *Gn_im);

/* CC-SN with a moving reference image (PAPER.md:L92 applied to Eqs. (8), (9); R19): the state is the
 * spectrum G = F[E] of the average RAW image; every frame is measured by Eq. (7) with the weight 1/(E + eps) formed
 * from the current state (E = Re F^-1[G]; returns -3 unless E + eps > 0 everywhere), then the state is updated with
 * the frame aligned by its displacement, exactly as in the CC-U functions (E' = E + eps holds identically).
 * Results report S (the minimised sum) like cco_track_sn.
 *   cco_track_rt_sn            Eq. (9), frames in order (as cco_track_rt)
 *   cco_iterate_reference_sn   Eq. (8), n_iter passes (as cco_iterate_reference)
 *   cco_step_from_spectrum_sn  one step from a given state (as cco_step_from_spectrum) */
int cco_track_rt_sn(const void *frames, int dtype, int batch, int H, int W, int u, const float *reference, double eps,
                    double a0, cco_result *out, double *G_out_re, double *G_out_im);
int cco_iterate_reference_sn(const void *frames, int dtype, int batch, int H, int W, int u, const float *reference,
                             double eps, int n_iter, cco_result *out, double *G_out_re, double *G_out_im);
int cco_step_from_spectrum_sn(const void *frame, int dtype, int H, int W, int u, const double *G_re, const double *G_im,
                              double eps, double a0, cco_result *out, double *Gn_re, double *Gn_im);

int cco_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif

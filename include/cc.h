/*
 * cc.h -- C-ABI boundary of the B200-native cross-correlation tracker.
 *
 * The library computes, for every camera frame, the displacement of a single
 * particle against a fixed reference image (RI) by the method of Werneck et
 * al., arxiv 2310.08770:
 *
 *   cc(s) = sum_r I(r+s) E(r) = F^-1[ F[I] (x) conj(F[E]) ](s)
 *                                    -- PAPER.md:L66-70, Eq. (4), Sec. II (CC-U)
 *   integer peak  = argmax_s cc(s)   -- PAPER.md:L90, Sec. III, sentence 1
 *   sub-pixel peak = argmax over a 1.5-pixel window around the integer peak,
 *                    sampled at ceil(1.5*u) points per axis (spacing 1/u), of
 *                    the element-wise product "interpolated into the upsampled
 *                    region, followed by an inverse discrete Fourier transform"
 *                                    -- PAPER.md:L90, Sec. III, sentences 2-5
 *
 * Every step runs in hand-written CUDA kernels for sm_100a (one fused kernel
 * per frame shape).  There is no CPU fallback: on a device
 * that is not compute capability 10.x every entry point returns CC_ERR_ARCH.
 *
 * Conventions:
 *   - images are row-major [y][x]; +x = increasing column, +y = increasing row;
 *   - the displacement d = (dy, dx) is the lag that maximises cc, i.e.
 *     frame(r) ~ reference(r - d); it is a multiple of 1/upsample;
 *   - the integer peak is wrapped to [-N/2, N/2) per axis; ties are resolved
 *     towards the smallest row-major index;
 *   - `peak` is the (upsampled) correlation sum at the maximum, in
 *     pixel-value^2 units (sum_r I(r+d) E(r)).
 *
 * Threading: a plan is immutable after creation (unless the reference update
 * of Eq. (9) is switched on, see cc_plan_enable_reference_update).  cc_track()
 * on one plan may be enqueued on several streams concurrently only when
 * cc_plan_info() reports scratch_bytes == 0; otherwise serialise the calls.
 * cc_track_host() uses plan-owned staging buffers and must be serialised per
 * plan.  A real-time session (cc_rt_*) owns its scratch and may run beside
 * cc_track on the same plan.  Measurement aids: include/cc_bench.h.
 */
#ifndef CC_H
#define CC_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cc_plan cc_plan; /* opaque; owned by the library */

typedef enum { CC_U8 = 0, CC_U16 = 1 } cc_dtype; /* pixel type of the frames */

typedef enum {
    CC_OK = 0,
    CC_ERR_INVALID_ARG = 1, /* NULL pointer, batch < 0, H/W <= 0, upsample < 1, misaligned frames */
    CC_ERR_UNSUPPORTED = 2, /* frame shape outside the built kernel variants                        */
    CC_ERR_NOMEM = 3,       /* host or device allocation failed                                    */
    CC_ERR_CUDA = 4,        /* a CUDA runtime call failed; text in cc_last_error()                 */
    CC_ERR_ARCH = 5         /* no CUDA device of compute capability 10.x                           */
} cc_status;

/* Static description of the kernel variant(s) a plan selected. */
typedef struct {
    int H, W, upsample, dtype;
    int grid_M;               /* M = ceil(1.5*upsample) upsampled samples per axis */
    int cluster_size;         /* CTAs per frame, throughput variant                               */
    int threads;              /* threads per CTA                                                   */
    int smem_bytes;           /* dynamic shared memory per CTA                                     */
    int max_clusters;         /* co-resident clusters = frames in flight                           */
    int lat_cluster_size;     /* CTAs per frame of the small-batch (latency) variant, 0 if none    */
    int lat_max_clusters;
    long long scratch_bytes;  /* plan-owned device scratch used by cc_track (0: stream-concurrent)  */
    long long table_bytes;    /* plan-owned constant tables (reference spectrum, upsampling tables) */
    int super_blocks;         /* passes of the upsampled DFT over the offsets d (T buffer capacity), throughput variant */
    int offsets_per_cta;      /* offsets d per CTA per pass                                                             */
    int tensor_core_stage1;   /* 1 if stage 1 of the upsampled DFT runs on the tensor cores (tcgen05.mma kind::tf32,   */
                              /* three-pass hi/lo split) in the throughput variant, 0 if on the FP32 pipes              */
} cc_plan_info_t;

/*
 * cc_plan_create -- PAPER.md:L98/L108 ("F[E_0] = F[I_0]": the RI is held as its
 * spectrum) plus the plan-time tables of the upsampled DFT.
 *   out        receives the plan (host pointer); untouched on error
 *   H, W       frame rows / columns; supported: powers of two, 64..1024 each
 *   dtype      pixel type of the frames later passed to cc_track
 *   upsample   u >= 1; u == 1 means "integer peak only"
 *   reference  H*W float32, row-major, HOST or DEVICE pointer; copied, the
 *              caller may free it on return
 * May synchronise the device.  Returns CC_OK or an error code.
 */
cc_status cc_plan_create(cc_plan **out, int H, int W, cc_dtype dtype, int upsample,
                         const float *reference);

/*
 * cc_plan_create_weighted -- cc_plan_create with the choice of the paper's
 * weighting:
 *   CC_METHOD_U   uniform weights, Eq. (4): maximum of sum_r I(r+d) E(r)
 *   CC_METHOD_SN  shot-noise weights, Eqs. (5)-(7): with I' = I + epsilon and
 *                 E' = E + epsilon, the MINIMUM of S(d) = sum_r I'(r+d)^2 / E'(r)
 *                 (chi^2 of Eq. (6) is minimised; R15, R16).  `peak`
 *                 then returns S at the minimum.  Needs E + epsilon > 0 in
 *                 every pixel (else CC_ERR_INVALID_ARG).  The paper's
 *                 recommendation is epsilon = 200 x the noise gain (L161).
 * Everything else as cc_plan_create; cc_track etc. work on either plan.
 */
typedef enum { CC_METHOD_U = 0, CC_METHOD_SN = 1 } cc_method;
cc_status cc_plan_create_weighted(cc_plan **out, int H, int W, cc_dtype dtype, int upsample,
                                  const float *reference, cc_method method, float epsilon);

/*
 * cc_track -- the hot path (Eq. (4)):
 * ingest -> real 2D FFT -> (x) conj(F[E]) -> inverse FFT -> integer argmax ->
 * upsampled DFT -> sub-pixel argmax, fused so that each frame is read from HBM
 * once and 12 bytes are written back.
 *   frames   DEVICE pointer, batch*H*W pixels of the plan's dtype, contiguous,
 *            16-byte aligned; owned by the caller, read only
 *   batch    number of frames (0 -> CC_OK, nothing enqueued)
 *   dx,dy    DEVICE pointers, batch float32 each: displacement in pixels
 *   peak     DEVICE pointer, batch float32, or NULL
 *   stream   cudaStream_t (as void*), NULL = default stream
 * Only enqueues work on `stream`; never synchronises, never allocates.
 */
cc_status cc_track(const cc_plan *plan, const void *frames, int batch,
                   float *dx, float *dy, float *peak, void *stream);

/*
 * cc_track_static -- cc_track for callers that cannot tolerate a device allocation anywhere near the call (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same computation, same results, same
 * arguments as cc_track (Eq. (4)), but:
 *   - the global spectrum scratch of the shapes that need one (1024 x 1024: the half spectrum of a frame, H*W/2
 *     complex64 = 4 MiB per frame in flight, does not fit a cluster's shared memory) is NOT the plan's cudaMalloc'ed
 *     buffer but a file-scope `static __device__` array of CC_STATIC_SCRATCH_BYTES inside the library; every GPU that
 *     loads the library holds that array until the process exits;
 *   - the launch is a plain kernel launch (no graph object); the call performs no cudaMalloc / cudaFree and calls no
 *     allocating library routine.  The first call on a device resolves the array's device address
 *     (cudaGetSymbolAddress, once per device, with that device current): make that call outside a stream capture.
 * Limits: the call launches min(batch, resident clusters) clusters like cc_track and is rejected with
 * CC_ERR_UNSUPPORTED (cc_last_error names the largest batch) when their spectrum blocks exceed the array -- at
 * 1024 x 1024 batch <= 2; shapes whose spectrum stays in shared memory (all others) need no scratch and take any
 * batch.  Plans with the reference update of Eq. (9) switched on are rejected (CC_ERR_UNSUPPORTED): use cc_track.
 * Sharing: ALL calls on a device, from every plan and stream, use the same array.  Nothing in it has to start at zero
 * (the kernel writes each element of a spectrum block before it reads it), so calls need no clearing between them,
 * but two calls that OVERLAP on the GPU (different streams, or a cc_track_static racing another process thread's)
 * overwrite each other's spectra: serialise them (same stream, or an event).  cc_track is not affected.
 * Arguments, ownership and error behaviour otherwise as cc_track.
 */
#define CC_STATIC_SCRATCH_BYTES (8u << 20)
cc_status cc_track_static(const cc_plan *plan, const void *frames, int batch,
                          float *dx, float *dy, float *peak, void *stream);

/*
 * cc_track_debug -- cc_track that additionally returns the wrapped integer
 * peak of step a5 (PAPER.md:L90 sentence 1).
 *   iy, ix   DEVICE pointers, batch int32 each, or NULL
 * (The optional per-phase timing argument of the interface sketch in SURVEY.md 8(b), `phase_ns`, lives in
 * cc_track_profile below, as SM-clock cycles per phase.)
 */
cc_status cc_track_debug(const cc_plan *plan, const void *frames, int batch,
                         float *dx, float *dy, float *peak, int *iy, int *ix, void *stream);

/*
 * cc_track_profile -- cc_track that additionally records, per frame, the SM
 * clock cycles spent in each phase of the fused kernel (the per-frame latency
 * breakdown).  Phases: 0 ingest + row FFT, 1 column FFT (x) conj(F[E]) +
 * column inverse, 2 row inverse FFT + integer argmax, 3 fp64 integer polish,
 * 4 upsampled-DFT stage 1, 5 stage 2, 6 sub-pixel argmax reduction, 7 fp64
 * sub-pixel polish.
 *   phase_cycles   DEVICE pointer, batch * CC_NUM_PHASES uint64
 */
#define CC_NUM_PHASES 8
cc_status cc_track_profile(const cc_plan *plan, const void *frames, int batch,
                           float *dx, float *dy, float *peak,
                           unsigned long long *phase_cycles, void *stream);

/*
 * cc_plan_set_host_chunk -- frames per host->device chunk of cc_track_host (0: the default, about 64 MB of
 * frames and at least one wave of clusters).  Chunks alternate between two plan-owned streams so that the copy
 * of one overlaps the kernel of the other.
 */
cc_status cc_plan_set_host_chunk(cc_plan *plan, int frames_per_chunk);

/*
 * cc_track_host -- the same path for HOST buffers (pageable or pinned): frames
 * are copied host->device in chunks overlapped with compute, results are
 * copied back, and the call returns after everything has completed.
 *   frames            HOST pointer, batch*H*W pixels
 *   dx, dy, peak      HOST pointers, batch float32 each (peak may be NULL)
 * Uses plan-owned streams and staging buffers (grown on first use; shapes whose spectrum block lives in global
 * scratch get a second scratch for the second stream).  On an error both streams are drained before the call
 * returns: nothing is in flight on the caller's buffers afterwards.
 */
cc_status cc_track_host(cc_plan *plan, const void *frames, int batch,
                        float *dx, float *dy, float *peak);

/*
 * Real-time session -- the paper's real-time mode (PAPER.md:L102-104, L216:
 * every camera frame is analysed as it arrives and the displacement is fed
 * back): one persistent cluster kernel stays resident and serves single
 * frames handed to it through a mailbox in mapped host memory, so a frame
 * costs neither a kernel launch nor a stream synchronisation.  Same kernel
 * code, same results as cc_track(batch = 1).
 *
 * cc_rt_open      starts the session kernel on a stream owned by the session.
 *   idle_timeout_ms  the kernel exits by itself after this long without a
 *                    frame (<= 0: 1000 ms); the next cc_rt_submit restarts it.
 *                    While the kernel is resident, device-wide synchronisation
 *                    (cudaDeviceSynchronize, cudaFree, ...) blocks until it
 *                    exits: use stream or event synchronisation instead.
 * cc_rt_submit    hands over one frame: DEVICE pointer, or HOST pointer to
 *                 pinned mapped memory (the kernel then reads the pixels over
 *                 PCIe itself); H*W pixels, 16-byte aligned; must stay valid
 *                 until cc_rt_wait returns.  One frame in flight at a time.
 * cc_rt_wait      spins (host) until the result of the submitted frame has
 *                 arrived; dx, dy, peak are HOST pointers (peak may be NULL).
 * cc_rt_track     submit + wait.
 * cc_rt_close     ends the kernel, frees the session.  NULL is a no-op.  Close
 *                 every session before cc_plan_destroy.
 * Errors: CC_ERR_INVALID_ARG (NULL/misaligned/no frame submitted),
 * CC_ERR_CUDA (launch failure, or no answer from the kernel).
 */
typedef struct cc_rt cc_rt;
cc_status cc_rt_open(cc_plan *plan, int idle_timeout_ms, cc_rt **out);
cc_status cc_rt_submit(cc_rt *rt, const void *frame);
cc_status cc_rt_wait(cc_rt *rt, float *dx, float *dy, float *peak);
cc_status cc_rt_track(cc_rt *rt, const void *frame, float *dx, float *dy, float *peak);
cc_status cc_rt_close(cc_rt *rt);

/*
 * cc_plan_enable_reference_update -- the paper's real-time analysis (Eq. (9)): after every
 * frame the plan's reference image is replaced by  F[E_i] = a0 F[I_i aligned] + (1 - a0) F[E_{i-1}],  the aligned
 * image being the frame translated by its detected displacement (Fourier shift theorem; cos(pi d) on the Nyquist
 * bins -- DESIGN.md R18).  a0 = 1 - exp(-T/tau) in (0, 1]; a0 == 0 switches the update off again.
 * Frames are then processed strictly in order: frame i of a cc_track batch is measured against the reference left
 * by frame i-1, and consecutive cc_track / cc_rt_track calls continue the sequence.  cc_track thereby MODIFIES the
 * plan: calls on one plan must be serialised (same stream).  May synchronise the device.
 *   CC-U plans   the update runs inside the fused kernel (one cluster, the largest-cluster variant of the shape).
 *   CC-SN plans  (R19) the state is F[E] of the average RAW image, kept in float64; after
 *                every frame separate kernels apply Eq. (9) to it and rebuild the weight spectrum F[-1/(E + eps)]
 *                that the fused kernel correlates with (one launch of the fused kernel per frame).  cc_rt_* cannot
 *                serve such a plan (CC_ERR_UNSUPPORTED).  If E + eps ever becomes <= 0 in some pixel, the next
 *                cc_plan_get_reference_spectrum call reports CC_ERR_INVALID_ARG.
 *
 * cc_plan_get_reference_spectrum -- debugging / checkpoint aid: the spectrum F[E] of the plan's current reference
 * image (for CC-SN plans: of E itself, not of the weight 1/(E + eps)).
 *   out   HOST pointer, H * (W/2 + 1) complex float32 (re, im interleaved), row ky, column kx = 0..W/2,
 *         natural frequency order, unnormalised (sum over pixels).  Synchronises the device.
 * cc_plan_get_reference_spectrum_f64 -- the same as complex float64 (CC-SN plans hold their state in float64;
 * CC-U plans return their float32 state widened).
 */
cc_status cc_plan_enable_reference_update(cc_plan *plan, double a0);
cc_status cc_plan_get_reference_spectrum(const cc_plan *plan, float *out);
cc_status cc_plan_get_reference_spectrum_f64(const cc_plan *plan, double *out);

/*
 * Offline analysis -- PAPER.md:L94-100, Eq. (8): the reference image of pass n is the mean of all images of the
 * data set, each aligned by its displacement against the reference of pass n-1:
 *     F[E_n] = (1/N) sum_i F[I_i aligned]        (alignment as in cc_plan_enable_reference_update).
 * cc_track_accumulate   cc_track over a batch (all clusters in parallel: "embarrassingly parallel", L100) that also
 *                       adds every frame's aligned spectrum to plan-owned per-cluster accumulators.  May be called
 *                       several times per pass (chunks of a data set).  Plans without the Eq. (9) update.  CC-SN
 *                       plans (R19) sum the aligned RAW spectra in float64 with separate kernels after
 *                       the tracking launch.  Allocates on first use; arguments as cc_track.
 * cc_plan_update_reference_from_accumulator
 *                       ends a pass: reduces the accumulators in a fixed order (deterministic), replaces the plan's
 *                       reference by the mean over all frames accumulated since the last call and clears them.
 *                       Enqueues on `stream` (use the stream of the cc_track_accumulate calls).
 *                       CC_ERR_INVALID_ARG if nothing was accumulated.
 */
cc_status cc_track_accumulate(cc_plan *plan, const void *frames, int batch, float *dx, float *dy, float *peak, void *stream);
cc_status cc_plan_update_reference_from_accumulator(cc_plan *plan, void *stream);

/*
 * cc_drift_correct -- PAPER.md:L110-127: removes the slowly drifting equilibrium position from a sequence of
 * displacements, r'_n = r_n - R_n, with the low-pass offset of Eq. (10), R_n = a0 r_n + b1 R_{n-1}
 * (b1 = 1 - a0; R_{-1} = 0, so R_0 = a0 r_0), or, when max_step > 0, its rate-limited form of Eqs. (11)-(12):
 * the offset moves by at most max_step = alpha/u per sample (the paper suggests alpha = 0.5).  A sequential
 * recurrence, evaluated in double precision by one warp on the device.
 *   dx, dy     DEVICE pointers, n float32 each (e.g. the outputs of cc_track)
 *   a0         1 - exp(-T/tau), in [0, 1]
 *   max_step   alpha / upsample, or <= 0 for the plain filter
 *   state      DEVICE pointer, 2 float64 (Rx, Ry), read and updated: zero it before the first call; consecutive
 *              calls then continue the same filter
 *   dxc, dyc   DEVICE pointers, n float32 each: the corrected displacements (may alias dx, dy)
 * Only enqueues work on `stream`.  n == 0 -> CC_OK.
 */
cc_status cc_drift_correct(const float *dx, const float *dy, int n, double a0, double max_step,
                           double *state, float *dxc, float *dyc, void *stream);

/* Frees every device/host allocation of the plan.  NULL is a no-op. */
cc_status cc_plan_destroy(cc_plan *plan);

/* Fills *info; returns CC_ERR_INVALID_ARG on NULL. */
cc_status cc_plan_info(const cc_plan *plan, cc_plan_info_t *info);

const char *cc_status_string(cc_status s);
const char *cc_last_error(void); /* thread-local detail of the last failure */

#ifdef __cplusplus
}
#endif
#endif /* CC_H */

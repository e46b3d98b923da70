/* tc.h -- C ABI of the tomoCAM hot path on one B200 (sm_100a).
 *
 * Paper: arXiv 2304.12934 (tomoCAM).  "P:L<n>" = line n of /root/reference/PAPER.md.
 * The three calls follow the paper's problem statement: the Radon transform R (eq. (2))
 * and its adjoint R* (eq. (11)) computed slice by slice with a NUFFT
 * (eqs. (6)-(8)), inside the MBIR gradient iteration (eqs. (9)-(10)) with
 * the qGGMRF prior (eqs. (12)-(13)).
 *
 * Layouts (all float32, C-contiguous; no complex numbers cross the boundary):
 *   volume   [slice][row i <-> y][col j <-> x],  x_j = j - n/2, y_i = i - n/2   (n x n per slice)
 *   sinogram [slice][angle a][bin u]            (sinogram order), t_u = u - center
 * Pointers: every data pointer may be DEVICE memory or HOST memory (pinned or pageable); the
 *   library looks the pointer up (cudaPointerGetAttributes).  Host pointers take the slab-streaming
 *   path: slabs of slices go through device staging buffers on side streams, overlapped
 *   with compute, and the call returns when the output is complete.  Pageable host arrays are page-locked
 *   (cudaHostRegister) for the duration of the call so that their copies overlap; if that fails the call
 *   still completes, without overlap.  Device-pointer calls are ordered on `cuda_stream` (a cudaStream_t,
 *   NULL = default stream) and return asynchronously.
 * Concurrency: a plan owns one set of scratch buffers, one side stream and its events: use it from one thread
 *   and ONE stream at a time (two device-pointer calls on different streams would race on the scratch).
 * Ownership: the caller owns every data buffer; the plan owns all scratch; nothing allocated by the
 *   library is ever returned.  A plan is not thread-safe.
 * Errors: every call returns a tc_status; nothing throws or aborts across the ABI; outputs are
 *   unspecified after an error; tc_last_error() gives thread-local text for the last failure.
 */
#ifndef TC_H
#define TC_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef enum { TC_OK = 0, TC_EINVAL = 1, TC_ENOMEM = 2, TC_ECUDA = 3, TC_EUNSUPPORTED = 4 } tc_status;

/* Acquisition geometry.  n: image side (even); n_det: detector bins (even); angles: HOST pointer to
 * n_angles float32 radians (copied at plan creation; any finite values); center: rotation-axis
 * position in bins (< 0 means n_det/2); oversamp must be 2.0; kb_width = 4, 6 or 8 taps per axis of the Kaiser-Bessel
 * window (w ~ log10(1/eps): about 3e-4, 3e-6 and 4e-8 against the direct DFT in exact arithmetic).  Sizes (else TC_EUNSUPPORTED): n must be a multiple of 32; n and n_det (even) must
 * factor into 2, 3, 5, 7 and 17 with at most five FFT passes (one per 16, per remaining power of two and per odd factor), e.g.
 * 2048, 2560 = 2^9 5, and the 2448 = 2^4 3^2 17 detector bins of the paper's Table 1 on an n = 2560 image; at most 6800. */
typedef struct {
    int n, n_det, n_angles;
    const float *angles;
    float center;
    float oversamp;
    int kb_width;
} tc_geom;

/* qGGMRF prior h = (|D|/sigma)^2 / (c + (|D|/sigma)^(2-p)), eq. (13); paper's values
 * p = 1.2, sigma = 1/0.7, c = 1e-4; 1 <= p <= 2.  p = 1 is the smoothed total variation:
 * h = u^2 / (c + u) = u - c + c^2 / (c + u), i.e. |D|/sigma up to a constant for |D| >> c sigma, still twice differentiable at 0.
 * lambda multiplies the prior (extension, default 1).
 * L is the step constant of the fixed 1/L step; 0 means: estimated by the library (power iteration
 * on A^T A plus the curvature bound of the prior, reading G15).  nonneg != 0 adds the constraint f >= 0 (P:L24:
 * "the choice of the constraint is not limited by the algorithm design"): the candidate is projected, z = max(y - g/L, 0).
 * grad_restart != 0 adds the gradient restart test: an accepted candidate with <g, z - x> > 0 resets the momentum.
 * neighbours: the neighbour set of eq. (12): 26 (1-hop, the paper's; 0 means 26), 10 (the 8 in-plane neighbours and
 * the 2 along z: the set P:L149 quotes for SVMBIR) or 6 (faces); weights 1/distance, normalised to sum 1 over the set.
 * mm_step != 0 replaces the fixed step 1/L by the majorise-minimise step length along -g ("other optimizers"; G23):
 * alpha = <g, g> / (||A g||^2 + lambda sum_pairs w h'(D)/D (g_m - g_n)^2), D = y_m - y_n; in-core problems only (TC_EUNSUPPORTED
 * when the problem has to be streamed). */
typedef struct { float p, sigma, c, lambda, L; int nonneg, grad_restart, neighbours, mm_step; } tc_prior;

/* One record per MBIR iteration: F = objective of the kept iterate, data / prior = the two terms of
 * the CANDIDATE, margin = (F_prev - F_cand)/F_prev, dot = <g, z - x> (0 unless grad_restart), beta = momentum used,
 * accepted = 1/0, restarted = 1 if the gradient test reset the momentum, alpha = step length used (1/L unless mm_step),
 * ms = wall-clock milliseconds of this iteration (every iteration ends with a stream synchronisation for the accept test, so
 * this is the GPU time of the iteration plus its launch overhead; bench.py's MBIR figure is the median of these). */
typedef struct { double F, data, prior, margin, dot; float beta; int accepted, restarted; float alpha; float ms; } tc_iter_log;

typedef struct tc_plan tc_plan;

/* Builds window coefficients, deapodisation vector, FFT twiddles, sorted angle tables.  Scratch is
 * allocated lazily by the first call that needs it.  max_slab_slices (0 = automatic) caps the number
 * of slices processed per slab. */
tc_status tc_plan_create(const tc_geom *geom, int max_slab_slices, tc_plan **out);
tc_status tc_plan_destroy(tc_plan *plan);

/* sinogram[n_slices][n_angles][n_det] = A volume[n_slices][n][n]  (forward, type-2 NUFFT route). */
tc_status tc_radon(tc_plan *plan, const float *volume, int n_slices, float *sinogram, void *cuda_stream);

/* volume[n_slices][n][n] = A^T sinogram[n_slices][n_angles][n_det]  (exact transpose of tc_radon). */
tc_status tc_backproject(tc_plan *plan, const float *sinogram, int n_slices, float *volume, void *cuda_stream);

/* Filtered back-projection, eq. (4) P:L64 (f = R* F^-1 |k| F p; filters P:L68): tc_backproject with every radial mode m weighted
 * by (pi / n_angles) * r(m) * win(m), r = |m| / n_det (1 / (4 n_det) at m = 0, the mean of |k| over the DC bin), win = 1 for
 * TC_FILTER_RAMP, 0.5 (1 + cos(2 pi m / n_det)) for TC_FILTER_HANN, and the Shepp-Logan and Butterworth windows below (the filters
 * P:L68 names), so that tc_fbp(tc_radon(f)) ~ f for angles uniform in [0, pi).
 * Same pointers, layouts, slab streaming and stream semantics as tc_backproject.  TC_EINVAL for an unknown filter. */
#define TC_FILTER_RAMP 0          /* Ram-Lak */
#define TC_FILTER_HANN 1
#define TC_FILTER_SHEPP_LOGAN 2   /* ramp x sin(pi m / n_det) / (pi m / n_det) */
#define TC_FILTER_BUTTERWORTH 3   /* ramp / (1 + (|m| / (n_det / 4))^4): order 2, cut-off at half the Nyquist frequency */
tc_status tc_fbp(tc_plan *plan, const float *sinogram, int n_slices, int filter, float *volume, void *cuda_stream);

/* Pre-pass for measured data ("b = -log(I / I0)", P:L129 sinogram order): Beer-Lambert transform and the reorder from
 * projection order, proj[n_angles][n_slices][n_det] as a detector delivers it, to sinogram[n_slices][n_angles][n_det]:
 *   sinogram[s][a][u] = -log(max((proj[a][s][u] - dark[s][u]) / (flat[s][u] - dark[s][u]), floor)),
 * flat (I0) and dark are [n_slices][n_det], nullable (1 and 0).  floor > 0 guards dead or saturated pixels.  All device or all
 * host pointers; device calls are ordered on cuda_stream. */
tc_status tc_preprocess(const float *proj, const float *flat, const float *dark, int n_angles, int n_slices, int n_det,
                        float floor, float *sinogram, void *cuda_stream);

/* `iters` iterations of the monotone accelerated gradient method with restart on
 * F(f) = 1/2 ||A f - b||^2 + lambda H(f) from f = 0.  volume: out.  log: HOST pointer, nullable,
 * `iters` records.  Synchronous (returns when `volume` is complete).
 * Device pointers: in core (4 volumes + 5 sinograms + FFT scratch of at most 128 slices in device memory; TC_ENOMEM if that
 * does not fit).  Host pointers: in core if it fits, else streamed slab by slab (S1) with `volume` itself as one of
 * the two host-resident volumes of the iteration and one more pinned by the library (n_slices n^2 floats). */
tc_status tc_mbir(tc_plan *plan, const float *sinogram, int n_slices, const tc_prior *prior, int iters,
                  float *volume, tc_iter_log *log, void *cuda_stream);

/* z-sharded MBIR (the paper's level-1 partition: one contiguous range of slices per GPU).  Forward and adjoint are
 * slice-wise, so the ranks only meet in the prior (one halo slice of the candidate towards each z-neighbour per iteration)
 * and in the three scalars of the accept test.  The library does the arithmetic; the caller supplies the transport:
 *   exchange(ctx): deliver this rank's send_down to the lower rank's recv_up and send_up to the upper rank's recv_down (n*n floats
 *                  each).  The send buffers are complete when it is called; the recv buffers must be complete when it returns.
 *   allreduce(ctx, vals, n): in-place sum over all ranks of n doubles in HOST memory (same result on every rank).
 * Both return 0 on success.  send_ / recv_ buffers are DEVICE memory owned by the caller; a rank at the bottom (top) of the volume
 * passes NULL for the down (up) pair.  tc_mbir_sharded(sinogram, volume: DEVICE, this rank's n_slices) is tc_mbir on the rank's
 * range; prior->L must be given (> 0, the same everywhere) and every rank must make the same calls.  The iterate sequence equals
 * the unsharded one up to the float64 summation order of the objective. */
typedef struct {
    void *ctx;
    int (*exchange)(void *ctx);
    int (*allreduce)(void *ctx, double *vals, int n);
    float *send_down, *send_up, *recv_down, *recv_up;
} tc_comm;
tc_status tc_mbir_sharded(tc_plan *plan, const float *sinogram, int n_slices, const tc_prior *prior, int iters, float *volume,
                          tc_iter_log *log, const tc_comm *comm, void *cuda_stream);

/* lambda_hat = ||A^T A v|| / ||v|| after `iters` power iterations on one slice from v = ones. */
tc_status tc_power_iteration(tc_plan *plan, int iters, double *lambda_hat);

/* Prior alone (test hook for the M2/M4 stencil kernels): grad (nullable) = grad H(volume),
 * *value (HOST, nullable) = H(volume); device or host pointers for volume/grad. */
tc_status tc_prior_eval(const float *volume, int n_slices, int n, const tc_prior *prior, float *grad, double *value);

/* tc_radon without any allocation, for callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses
 * that forbid it): the FFT scratch is a 16 MiB static device array of the library (held by every GPU that loads it, until exit)
 * instead of the plan's lazily allocated buffers.  DEVICE pointers only, ordered on cuda_stream; limits: n <= 256 and
 * n_angles * n_det <= 131072 (TC_EUNSUPPORTED beyond, with the sizes in tc_last_error); any n_slices (groups of 8, one after the
 * other).  Same result as tc_radon.  All calls on a device share the array, which keeps the last call's contents: calls that
 * overlap on the GPU (two streams, plans or host threads) race.  The array's address is looked up at tc_plan_create. */
tc_status tc_radon_static(tc_plan *plan, const float *volume, int n_slices, float *sinogram, void *cuda_stream);

/* Stage hooks for the per-stage unit tests: ONE complex plane through ONE stage of the NUFFT, HOST arrays in natural order
 * (complex = interleaved float pairs).  fine_grid: F1 + F2 of eq. (8) read backwards: slices re, im (im nullable) ->
 * Ghat[k_y][k_x], G x G, G = 2 n, FFT order, of the plane re + i im (deapodised, zero-padded, 2-D FFT); gather: F3, eq. (7) reversed
 * (P:L83): Ghat -> c[a][m mod n_det] (before the centre phase; the Nyquist mode stays 0); spread: B2, eq. (7): c -> Ghat.
 * Cells of Ghat farther than n + kb_width - 1 from the origin are never touched by the method and come back as 0. */
tc_status tc_stage_fine_grid(tc_plan *plan, const float *re, const float *im, float *grid_out);
tc_status tc_stage_gather(tc_plan *plan, const float *grid_in, float *cpol_out);
tc_status tc_stage_spread(tc_plan *plan, const float *cpol_in, float *grid_out);

/* One-shot form with exactly the problem statement's shape = create plan, tc_radon, destroy. */
tc_status tc_radon1(const float *volume, int n_slices, int n, const float *angles, int n_angles, int n_det,
                    float center, float *sinogram);

/* Page-locked host memory for callers without a CUDA runtime of their own (host-resident volumes of the streamed path):
 * *ptr = `bytes` of pinned memory (not rounded up); release with tc_host_free.  TC_ENOMEM if it cannot be had. */
tc_status tc_host_alloc(size_t bytes, void **ptr);
tc_status tc_host_free(void *ptr);

/* Kernel launches issued by this library on the calling thread since the last reset (for bench.py). */
long long tc_launch_count(int reset);

/* Scheduler statistics of the last host-pointer call: seconds of H2D, compute, D2H (CUDA-event spans summed over the slabs; each
 * stream is serial, so each is <= wall_s) and wall time of the streamed loop; overlap in [0, 1] =
 * (h2d + compute + d2h - wall) / (h2d + compute + d2h - max(h2d, compute, d2h)): the fraction of the two shorter resources' work
 * hidden behind the others (1: wall = the busiest resource alone; 0: no overlap).  setup_s: before the loop (page-locking,
 * buffers, ||b||^2), handover_s: after it (copy into `volume` when x ended up in the library's buffer); both outside wall_s. */
typedef struct { double h2d_s, compute_s, d2h_s, wall_s, overlap; long long h2d_bytes, d2h_bytes; int n_slabs; double setup_s, handover_s; } tc_sched_stats;
tc_status tc_last_sched_stats(tc_plan *plan, tc_sched_stats *out);

/* Per-kernel timing with CUDA events recorded on the launching stream around every NUFFT stage launch
 * (stages: 0 fwd_rows, 1 fwd_cols, 2 fwd_gather, 3 adj_radial, 4 adj_spread, 5 adj_cols, 6 adj_rows, 7 fwd_radial).
 * tc_profile switches recording on/off; tc_profile_read waits for the recorded events, returns summed
 * milliseconds and launch counts per stage (arrays of TC_N_STAGES, HOST) and clears the records. */
#define TC_N_STAGES 8
tc_status tc_profile(tc_plan *plan, int enable);
tc_status tc_profile_read(tc_plan *plan, double *ms, long long *launches);

const char *tc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif

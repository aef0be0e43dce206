/*
 * gbk.h -- C ABI of libgbk: batched residual / chi^2 evaluation of GBKFIT-style
 * kinematic models of disc galaxies on NVIDIA B200 (sm_100a).
 *
 * The operation is the paper's "intensity cube modelling strategy"
 * (Bekiaris et al., arXiv:1510.01815; citations are /root/reference/PAPER.md
 * lines): one fitting iteration = evaluate the model cube (PAPER.md:63,
 * 197-210), convolve it with the PSF and LSF,
 * down-sample, extract velocity and dispersion maps as the
 * first and second moments, and form the error-weighted
 * residual and chi^2 against the observed maps (eq. 11).
 * Every optimiser of the paper (LM, nested sampling, nested grids;
 * PAPER.md:265-289) calls that iteration thousands of times; here it is
 * batched: K parameter rows per call.
 *
 * Plain C, no torch types.  Every pointer says whether it is HOST or DEVICE
 * memory.  No function throws or aborts; all return GBK_OK or an error code
 * and leave a message for gbk_last_error().  There is NO CPU fallback: without
 * a CUDA device every compute call returns GBK_ERR_CUDA.  Calls make the problem's device current
 * for their duration and restore the caller's device.
 *
 * Streams and threads.  The eval calls are asynchronous on the caller's stream.  The only state they
 * share is a small scratch (cross-tile chi^2 partials of tiled launches, staging of the host entry)
 * that the problem keeps PER STREAM: launches of one problem on different streams may overlap, from
 * one host thread or several (the scratch table is guarded by a mutex).  Launches on the SAME stream
 * are ordered by the stream and share that stream's scratch.  A CUDA graph captured from a stream
 * uses that stream's scratch: do not replay it while other work of the same problem and stream is in
 * flight elsewhere.  The scratch grows (cudaMalloc, which synchronises) the first time a stream sees
 * a larger batch; gbk_reserve sizes it up front, which is REQUIRED before a stream capture.
 *
 * Model row (GBK_P = 10 floats; GBK_P_EPINAT = 12 with the Epinat rotation curve):
 *   [0] x_o, [1] y_o    kinematic centre, data pixels (pixel j is centred on j)
 *   [2] PA   degrees    position angle (eq. 1-2)
 *   [3] i    degrees    inclination (eq. 3)
 *   [4] V_sys km/s      systemic velocity (eq. 8)
 *   [5] V_t  km/s, [6] r_t px   rotation curve (eq. 6; or ramp)
 *   [7] sigma_0 km/s    intrinsic dispersion
 *   [8] r_0 px, [9] I_0 exponential disc (eq. 5), or the scale length and
 *                       amplitude of a tabulated profile (gbk_problem_desc.intensity_table)
 *   [10] a, [11] g      GBK_RC_EPINAT only: the slopes of eq. 7, both > 0
 * Every array of rows at this boundary is [K][row_stride] with row_stride = gbk_problem_info.row_stride
 * (GBK_P, or GBK_P_EPINAT for a GBK_RC_EPINAT problem).
 *
 * Out-of-domain rows are not errors: a row with a non-finite parameter,
 * sigma_0 <= 0, r_0 <= 0, r_t <= 0, I_0 <= 0 or |cos i| < 1e-6, or with an
 * unmasked spaxel that is model-dark (m0 < 1e-30 * I_0) or has non-finite
 * moments, gets chi2 = +INF (an optimiser rejects it).
 */
#ifndef GBK_H_
#define GBK_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GBK_P 10
#define GBK_P_EPINAT 12 /* GBK_P + the Epinat slopes a, g */
#define GBK_P_MAX 12

enum { GBK_OK = 0, GBK_ERR_ARG = 1, GBK_ERR_ALLOC = 2, GBK_ERR_CUDA = 3, GBK_ERR_UNSUPPORTED = 4 };
enum { GBK_RC_ARCTAN = 0, GBK_RC_RAMP = 1, GBK_RC_EPINAT = 2 };
/* eq. 6; V_t*min(r/r_t,1); eq. 7: V_t q^g/(1+q^a), q = r/r_t.
 * GBK_RC_EPINAT is the curve the paper pairs with velocity-field modelling; its rows
 * have GBK_P_EPINAT = 12 floats, the slopes in [10] = a > 0 and [11] = g > 0, for BOTH strategies. */
enum { GBK_PSF_GAUSSIAN = 0, GBK_PSF_IMAGE = 1 }; /* eq. 9; image */

typedef struct gbk_problem gbk_problem; /* opaque; owns device copies of the observation */

/*
 * Problem descriptor: the observation a batch of rows is compared with
 * (velocity and dispersion maps with optional error and mask maps,
 * PAPER.md:185; PSF and LSF; grid and up-sampling factor,
 * PAPER.md:201; rotation-curve choice).
 * All pointers are HOST memory, read during gbk_create_problem only; the caller
 * may free them afterwards.  Maps are [n_gal][ny][nx], x fastest.
 */
typedef struct {
  int32_t nx, ny, nv;   /* spaxels and velocity channels of the observation               */
  int32_t u;            /* spatial up-sampling factor >= 1; the model is evaluated on a     */
                        /* (u*nx) x (u*ny) fine grid and block-averaged */
  float v_center, dv;   /* km/s; channel k has velocity v_center + (k-(nv-1)/2)*dv          */
  int32_t rc_model;     /* GBK_RC_*                                                        */
  int32_t n_gal;        /* data sets held by this problem (>= 1)                           */
  const float *vobs;    /* observed velocity map, km/s (required)                          */
  const float *verr;    /* its 1-sigma error map, > 0 where unmasked (required)            */
  const float *sobs;    /* observed dispersion map; NULL with serr NULL drops the second   */
  const float *serr;    /* term of eq. 11.  W of eq. 11 is pre-folded by    */
                        /* the caller as serr / sqrt(W)                     */
  const uint8_t *mask;  /* 0 = masked spaxel; NULL = all valid              */
  int32_t psf_kind;     /* GBK_PSF_*                                                       */
  const float *psf_fwhm;  /* GAUSSIAN: FWHM in DATA pixels, [n_gal] if psf_per_gal else [1]; */
                          /* taps exp(-j^2/2s^2), s = u*FWHM/(2 sqrt(2 ln 2)) fine pixels,   */
                          /* j in [-R,R], R = ceil(4 s), normalised to sum 1; FWHM <= 0 is   */
                          /* the delta PSF                                                  */
  const float *psf_image; /* IMAGE: [n_gal or 1][psf_n][psf_n] sampled on the FINE grid,     */
  int32_t psf_n;          /* psf_n odd; normalised to sum 1 at create; applied as a true     */
                          /* convolution (kernel flipped)                                   */
  int32_t psf_per_gal;  /* 0: one PSF shared by all data sets                              */
  float lsf_sigma;      /* km/s; Gaussian LSF, taps R = ceil(4*sigma/dv) channels,           */
                        /* normalised; <= 0 is the delta LSF                               */
  int32_t tile_w, tile_h; /* spatial tile of one thread block in SPAXELS; 0 = automatic:     */
                          /* the largest tile of which two blocks fit in an SM's shared      */
                          /* memory, and, when BOTH are 0, smaller tiles at eval time for     */
                          /* batches too small to fill the GPU (chi^2 then differs between    */
                          /* batch sizes by summation order only, ~1e-7 relative)             */
  int32_t device;       /* CUDA device ordinal; < 0 = the current device                   */
  const float *intensity_table; /* NULL: the exponential disc of eq. 5.  Else a "user-specified      */
  int32_t intensity_n;          /* intensity model": I(r) = I_0 T(r / r_0) with T      */
  float intensity_dx;           /* tabulated at x_j = j * intensity_dx, j = 0 .. intensity_n - 1      */
                                /* (>= 2 finite values >= 0, dx > 0), linear interpolation between   */
                                /* nodes, the last value beyond them; cube strategy only             */
} gbk_problem_desc;

/* What gbk_create_problem decided (for tests, benchmarks and op counting). */
typedef struct {
  int32_t nx, ny, nv, u, n_gal;
  int32_t r_v;            /* LSF tap radius, channels                                      */
  int32_t r_p_max;        /* largest PSF tap radius over the data sets, fine pixels        */
  int32_t tile_w, tile_h; /* tile in spaxels                                               */
  int32_t tiles_x, tiles_y;
  int32_t block_threads;  /* threads per block of the fused kernel                        */
  int32_t smem_bytes;     /* dynamic shared memory per block                              */
  int32_t blocks_per_sm;  /* occupancy of the fused kernel as reported by the runtime      */
  int32_t sm_count;
  int64_t ext_voxels_per_eval; /* sum over tiles of (tw+2R)(th+2R)(nv+2R_v), R = r_p_max   */
  int32_t device;         /* CUDA device ordinal the problem lives on                      */
  int32_t strategy;       /* GBK_STRATEGY_* the host drivers evaluate with (gbk_set_strategy) */
  int64_t unfused_bytes_per_eval; /* algorithmic HBM bytes of gbk_eval_batch_unfused per row:   */
                          /* every intermediate array written once and read once per consumer */
  int32_t row_stride;     /* floats per parameter row: GBK_P, or GBK_P_EPINAT                  */
  int32_t extraction;     /* GBK_EXTRACT_* (gbk_set_extraction)                                 */
} gbk_problem_info;

/*
 * Validates the descriptor, copies the observation to the device, builds tap
 * and channel tables, picks the tiling.  *out receives the handle.
 * Errors: GBK_ERR_ARG (NULL/shape/non-finite unmasked data/even psf_n/non-
 * positive error at an unmasked spaxel), GBK_ERR_UNSUPPORTED (tile does not
 * fit in shared memory, PSF radius beyond the supported maximum),
 * GBK_ERR_ALLOC, GBK_ERR_CUDA.
 */
int gbk_create_problem(const gbk_problem_desc *desc, gbk_problem **out);

int gbk_get_info(const gbk_problem *p, gbk_problem_info *info);

/*
 * Which of the paper's two modelling strategies the host drivers gbk_fit_* evaluate
 * rows with: the intensity-cube strategy (gbk_eval_batch, the default) or the velocity-field
 * strategy (gbk_eval_vfield_batch; residual vectors are then ny*nx long instead of 2*ny*nx).
 * GBK_RC_EPINAT problems start as GBK_STRATEGY_VFIELD (the paper's pairing), all others
 * as GBK_STRATEGY_CUBE.  The eval calls themselves ignore it.
 */
enum { GBK_STRATEGY_CUBE = 0, GBK_STRATEGY_VFIELD = 1 };
int gbk_set_strategy(gbk_problem *p, int32_t strategy);

/*
 * How the cube strategy extracts the velocity and dispersion maps from the down-sampled cube
 * (PAPER.md:228): GBK_EXTRACT_MOMENTS, the first and second moments of every spectrum (the paper's
 * choice, and the default), or GBK_EXTRACT_GAUSSFIT, a Gaussian profile fitted to every
 * spectrum (the paper tried it, and compares the two in section
 * 6.2): unweighted least squares for (A, mu, sigma) by Levenberg-Marquardt started
 * from the moments, velocity = mu, dispersion = sigma, m0 = the plain sum; a fit that does not
 * converge gives NaN there and chi2 = +INF if the spaxel is unmasked.  The fit needs the whole
 * convolved spectrum of every spaxel, which the fused kernel never forms: with GBK_EXTRACT_GAUSSFIT
 * gbk_eval_batch (and the drivers) run the multi-kernel pipeline of gbk_eval_batch_unfused.
 */
enum { GBK_EXTRACT_MOMENTS = 0, GBK_EXTRACT_GAUSSFIT = 1 };
int gbk_set_extraction(gbk_problem *p, int32_t extraction);

/*
 * The hot path (PAPER.md:63-66 steps 1-3 for K rows), fused: the model cube is
 * never written to memory.  Asynchronous on `cuda_stream`; never synchronises
 * or allocates except to grow that stream's cross-tile scratch (see gbk_reserve).
 * Errors: GBK_ERR_ARG (NULL arguments, K < 0, K x tiles beyond the grid limit, scratch growth
 * needed during a stream capture), GBK_ERR_UNSUPPORTED, GBK_ERR_ALLOC, GBK_ERR_CUDA.
 *   params     DEVICE [K][row_stride] float32, row-major
 *   gal_index  DEVICE [K] int32 in [0, n_gal), or NULL (all rows use data set 0)
 *   chi2       DEVICE [K] float32, required (eq. 11)
 *   m0,m1,m2   DEVICE [K][ny][nx] float32 each, any may be NULL: flux (sum over
 *              channels), velocity (first moment) and dispersion (sqrt of the
 *              second central moment) maps of the model
 *   resid      DEVICE [K][2][ny][nx] float32 or NULL: (model-obs)/err for the
 *              velocity and dispersion maps, 0 where masked
 *   cuda_stream  a cudaStream_t (NULL = the legacy default stream)
 * The caller owns all buffers.
 */
int gbk_eval_batch(gbk_problem *p, const float *params, const int32_t *gal_index, int64_t K,
                   float *chi2, float *m0, float *m1, float *m2, float *resid,
                   void *cuda_stream);

/*
 * gbk_eval_batch (chi^2 only) that also COUNTS the work the voxel loop executes, for the roofline
 * of bench.py: `counters` is a DEVICE array of GBK_N_COUNTERS uint64 the kernel adds to (the caller
 * zeroes it).  Units: one warp item = 128 fine samples (32 lanes x 2 pixel pairs); a polynomial block
 * = 8 channels of one warp item summed as a polynomial (1024 voxels); a direct channel = 1 channel of
 * one warp item by one ex2 per voxel (128 voxels).  The counting costs a few atomics per thread block,
 * so timings are taken with gbk_eval_batch.
 */
enum { GBK_CNT_ITEMS = 0, GBK_CNT_POLY_BLOCKS = 1, GBK_CNT_DIRECT_CHANNELS = 2, GBK_CNT_PRECISE_ITEMS = 3,
       GBK_N_COUNTERS = 4 };
int gbk_eval_batch_counted(gbk_problem *p, const float *params, const int32_t *gal_index, int64_t K,
                           float *chi2, uint64_t *counters, void *cuda_stream);

/*
 * Sizes the scratch that `cuda_stream` needs for batches of up to K_max rows (any tiling the library
 * may choose for them) and for gbk_eval_batch_host, so that later eval calls on that stream neither
 * allocate nor synchronise.  Needed before capturing eval calls into a CUDA graph: an eval call that
 * would have to grow the scratch during a capture returns GBK_ERR_ARG instead.
 */
int gbk_reserve(gbk_problem *p, int64_t K_max, void *cuda_stream);

/*
 * gbk_eval_batch for callers that cannot allocate at all (a stream capture without a gbk_reserve
 * beforehand, a serving loop or a harness that forbids cudaMalloc): same arguments, same kernel,
 * same results, but the cross-tile scratch of a tiled launch (one chi^2 partial per row and tile,
 * one tile counter per row) lives in a fixed array in the library's device image instead of the
 * per-stream scratch that gbk_eval_batch grows with cudaMalloc.  The call never calls cudaMalloc,
 * cudaFree or any allocating routine, and never synchronises: it clears the K tile counters with a
 * cudaMemsetAsync on `cuda_stream` and launches the kernel there.
 * Limits (the size of the array, 4.25 MiB, which every GPU that loads the library holds until the
 * process exits):  K <= GBK_STATIC_MAX_ROWS  and  K x tiles <= GBK_STATIC_MAX_PARTIALS, tiles being
 * the tiles per row of the tiling the library picks for K rows (tiles_x x tiles_y of gbk_get_info
 * for large K or an explicit tile; never more for small K than ceil(nx / 4) ceil(ny / 4)).  Larger
 * batches are rejected with GBK_ERR_ARG (split them, or use gbk_eval_batch); so is
 * GBK_EXTRACT_GAUSSFIT (GBK_ERR_UNSUPPORTED: that pipeline needs a model cube of scratch).
 * ONE array per device serves every problem and every stream: two gbk_eval_batch_static calls that
 * may overlap on the GPU (different streams, or a replayed graph beside a live call) RACE on it --
 * order them on one stream or with events.  It keeps the last call's contents between calls;
 * nothing in it needs to survive from one call to the next.
 */
#define GBK_STATIC_MAX_ROWS (1 << 16)
#define GBK_STATIC_MAX_PARTIALS (1 << 20)
int gbk_eval_batch_static(gbk_problem *p, const float *params, const int32_t *gal_index, int64_t K,
                          float *chi2, float *m0, float *m1, float *m2, float *resid,
                          void *cuda_stream);

/*
 * Comparison path, same contract: one kernel per step of the paper's pipeline
 * (PAPER.md:197-251), with the FP32 model cube written to device memory
 * between steps (the paper's own structure minus the FFT).  Processes the rows
 * in chunks that fit its scratch buffer.
 */
int gbk_eval_batch_unfused(gbk_problem *p, const float *params, const int32_t *gal_index,
                           int64_t K, float *chi2, float *m0, float *m1, float *m2, float *resid,
                           void *cuda_stream);

/*
 * The paper's OTHER modelling strategy, velocity-field modelling (section
 * 2.2.1): eq. 8 evaluated at every spaxel centre of the nx x ny grid -- no cube, no
 * PSF, no LSF, no up-sampling (the paper skips steps 2.2.2-2.2.5) -- then the
 * velocity residual and the first term of eq. 11 only.  Uses the
 * problem's vobs / verr / mask and rc_model; of a row only x_o, y_o, PA, i, V_sys, V_t, r_t are
 * read, plus a = row[10], g = row[11] with GBK_RC_EPINAT (a row is out of domain, chi2 = +INF, when
 * one of those is not finite, r_t <= 0, |cos i| < 1e-6, or a <= 0 or g <= 0).  Asynchronous on
 * `cuda_stream`, no allocation.
 *   params DEVICE [K][row_stride]; gal_index DEVICE [K] or NULL; chi2 DEVICE [K], required
 *   vmap   DEVICE [K][ny][nx] or NULL: the model velocity field
 *   resid  DEVICE [K][ny][nx] or NULL: (model - vobs) / verr, 0 where masked
 */
int gbk_eval_vfield_batch(gbk_problem *p, const float *params, const int32_t *gal_index, int64_t K,
                          float *chi2, float *vmap, float *resid, void *cuda_stream);

/*
 * End-to-end entry with HOST buffers: copies params (and gal_index) to the
 * device, runs gbk_eval_batch, copies chi2 back and waits for `cuda_stream`.
 * params/gal_index/chi2 are HOST pointers (pinned memory makes the copies
 * asynchronous and faster; pageable memory also works).
 */
int gbk_eval_batch_host(gbk_problem *p, const float *params, const int32_t *gal_index, int64_t K,
                        float *chi2, void *cuda_stream);

/* Frees device memory.  NULL is a no-op. */
int gbk_destroy(gbk_problem *p);

/* Thread-local message of the last failing call on this thread ("" if none). */
const char *gbk_last_error(void);

/*
 * Pipe-throughput probes used for the roofline denominators (DESIGN.md
 * "Roofline"): a register-only loop of independent MUFU.EX2 (which = 0) or
 * FFMA (which = 1) instructions on every SM.  Launches one kernel on
 * `cuda_stream` executing `iters` x 16 instructions per thread in
 * `blocks` x `threads`; `sink` is a DEVICE float buffer of at least one element
 * (written only to keep the loop alive).  *ops_per_launch receives the number
 * of lane-level operations the launch executes.
 */
int gbk_probe_pipe(int which, int64_t iters, int blocks, int threads, float *sink,
                   double *ops_per_launch, void *cuda_stream);

/*
 * A measured answer to "would tcgen05 help the 15 x 15 image-PSF pass of config 4?" (DESIGN.md
 * section 5, profiles/): every CTA issues, `iters` times, the tcgen05.mma sequence that one 64 x 64 tile
 * of that pass would need as a banded contraction -- 15 kernel rows x 3 BF16 split products x 5 K-steps
 * x (one M = 128 and one M = 64 MMA, N = 64, K = 16), operands in shared memory, accumulators in
 * TMEM -- after checking ONE MMA on known integers against the exact product.  `check` is a DEVICE
 * float that receives the largest error of that check (0 = the descriptors mean what they should);
 * *flops_per_launch receives 2 x multiply-adds issued.  One launch of `blocks` CTAs of 128 threads on
 * `cuda_stream`; the caller times it.  A probe, not a product path.
 */
int gbk_probe_umma(int iters, int blocks, float *check, double *flops_per_launch, void *cuda_stream);

/* ------------------------------------------------------------------------------------------
 * Host drivers: the paper's three optimisers re-stated as callers of the
 * batched hot path.  Each builds batches of rows, calls gbk_eval_batch on `cuda_stream`, reduces
 * on the device what can be reduced there (argmin, J^T J) and reads back a few numbers per
 * iteration.  All array arguments are HOST memory.  They block until the fit is done.
 * MPFIT and MultiNest themselves are third-party codes and are not reproduced; these are plain
 * re-statements of the published algorithms.
 * ---------------------------------------------------------------------------------------- */
typedef struct {
  int64_t evals;       /* rows evaluated                                                      */
  int32_t launches;    /* gbk_eval_batch calls                                                */
  int32_t iterations;  /* NG: levels; LM: largest iteration count over the fits; NS: batches  */
  int32_t converged;   /* fits that met their stopping rule                                   */
  float ms_total;      /* wall clock of the call, ms                                          */
  int32_t failed;      /* LM: fits that could not iterate (start row out of domain, a finite-   */
                       /* difference row out of domain, singular or non-finite normal equations) */
} gbk_fit_stats;

/*
 * Nested grids (refinement rule: DESIGN.md reading A19).  `n_axes` parameters
 * (indices axis_param[a] into the row, box [axis_lo[a], axis_hi[a]]) are gridded with axis_nodes[a]
 * nodes each (the paper uses 7, 11, 11, 5, 5, 5 for PA, r_t, V_t, sigma, a, g), the
 * other parameters stay at base_row.  Level l has spacing h_a = (hi-lo)/(nodes_a 2^l) and nodes
 * c + (j - (nodes_a-1)/2) h_a; c = box centre at level 0, then the best node of the level before.  An
 * axis on PA (index 2) whose box spans >= 360 degrees wraps; any other axis is shifted to stay inside
 * its box.  Ties in chi^2 take the lowest flat index (axis 0 slowest).  The product of the node counts
 * is <= 2^24.  Stopping ("until the area of the parameter space under the grid is smaller
 * than a user-defined accuracy threshold a"; :362: a = 0.01 for r_t, 0.1 otherwise): the level whose
 * spacing is <= axis_accuracy[a] on EVERY axis is the last one; axis_accuracy == NULL runs exactly
 * max_levels levels; max_levels always caps the count.  stats->converged is 1 when the thresholds were
 * reached (or none were given) and the best chi^2 is finite.
 * base_row and best_row are [row_stride]; best_chi2 [1] receives the chi^2 of the last level's best node.
 */
int gbk_fit_ng(gbk_problem *p, const float *base_row, int32_t gal, int32_t n_axes,
               const int32_t *axis_param, const float *axis_lo, const float *axis_hi,
               const int32_t *axis_nodes, const float *axis_accuracy, int32_t max_levels,
               float *best_row, float *best_chi2, gbk_fit_stats *stats, void *cuda_stream);

/*
 * Levenberg-Marquardt for n_fits independent fits at once (config 5: one fit
 * per galaxy; config 2: n_fits = 1), device-resident: the state of every fit stays in
 * device memory and the host reads back one integer (fits still active) every four iterations.  Per
 * iteration ONE batch of n_listed*(n_free+1) rows (base + forward differences of rel_step x box
 * width, backward at the upper bound, doubled until the step is representable) with weighted
 * residuals, J^T J and J^T r reduced in FP64, the damped normal equations
 * (A + lambda diag A) x = -g solved by Cholesky for four damping factors lambda x {0.1, 1, 10, 100},
 * and ONE batch of n_listed*4 trial rows for chi^2.  The best trial that lowers chi^2 is accepted
 * (lambda <- max(1e-9, 0.3 x its factor x lambda)), else lambda <- 1e4 lambda.  Parameters are
 * clipped to [lo, hi].  A fit stops when the relative chi^2 decrease of an accepted step is < ftol
 * (converged), when no damping factor up to 1e10 lowers chi^2 (converged: stationary as far as LM can
 * tell), after max_iter iterations, or as FAILED when it cannot iterate: the start row or a
 * difference row is out of domain (chi^2 = +INF), or the normal equations are singular or not finite
 * for every damping factor.  Failed fits are counted in stats->failed, never in stats->converged.
 *   start_rows [n_fits][row_stride], gal [n_fits] or NULL (all 0), free_param/lo/hi [n_free]
 *   fit_rows [n_fits][row_stride], fit_chi2 [n_fits], fit_iters [n_fits] or NULL
 * A fit whose start row has chi^2 = +INF is returned unchanged with chi^2 = +INF.
 * stats->evals counts the rows evaluated for fits that were active.
 */
int gbk_fit_lm(gbk_problem *p, int32_t n_fits, const float *start_rows, const int32_t *gal,
               int32_t n_free, const int32_t *free_param, const float *lo, const float *hi,
               float rel_step, int32_t max_iter, float ftol, float *fit_rows, float *fit_chi2,
               int32_t *fit_iters, gbk_fit_stats *stats, void *cuda_stream);

/*
 * Nested sampling with ln L = -chi^2/2 (A20) and a uniform prior on
 * the box: n_live live points; every batch draws `batch` candidates uniformly from the ellipsoid of
 * the live points (their mean and covariance, scaled to hold them all and enlarged by the fraction
 * `enlarge` >= 0; intersected with their enlarged bounding box and the prior box; the box alone
 * while the covariance is singular) and evaluates them in one launch; each candidate that beats
 * the current worst live point replaces it (prior volume X_i = exp(-i/n_live), evidence by the
 * simple rule Z += L_i (X_{i-1} - X_i)).
 * Stops when L_max X_i < tol x Z or after max_batches.  Outputs: the best row, its chi^2, the
 * posterior-mean row (base_row, best_row, mean_row: [row_stride]) and ln Z.  `seed` seeds the driver's own generator (xoshiro256**).
 */
int gbk_fit_ns(gbk_problem *p, const float *base_row, int32_t gal, int32_t n_free,
               const int32_t *free_param, const float *lo, const float *hi, int32_t n_live,
               int32_t batch, int32_t max_batches, float enlarge, float tol, uint64_t seed,
               float *best_row, float *best_chi2, float *mean_row, double *log_evidence,
               gbk_fit_stats *stats, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* GBK_H_ */

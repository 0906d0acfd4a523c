/*
 * cetra.h -- C ABI of the B200-native CETRA hot path (arXiv 2503.20875).
 *
 * Citations are line numbers of PAPER.md (the paper's text); "R<n>" are the readings of the
 * paper listed in DESIGN.md.  The library implements, as hand-written sm_100a CUDA kernels:
 *
 *   linear search   (Eq. 1-2): for every trial duration D_j and every trial
 *                   mid-transit time t_i, the weighted least-squares amplitude of the nearest-
 *                   neighbour sampled transit template in the window [t_i - D_j/2, t_i + D_j/2]:
 *                   depth, depth variance and the log-likelihood gain over the flat model;
 *   periodic search (Eq. 3-4): phase-fold those per-(t_i, D_j) statistics over
 *                   trial periods with nearest-neighbour lookup on the t0 grid, common depth,
 *                   and reduce every period to its maximum-likelihood (t0, duration) element.
 *
 * Conventions (all entry points)
 *  - Every function returns a cetra_status, never throws, never exits, allocates no device memory:
 *    the caller owns every buffer and supplies the scratch workspace (size from the
 *    *_workspace_bytes functions, 256-byte aligned).  Work is enqueued on `cuda_stream`
 *    (a cudaStream_t passed as void*) and the call returns without synchronising unless stated.
 *  - "_dev" pointers are device memory, "_host" pointers are host memory (pageable is fine) and are
 *    free to be reused as soon as the call returns.
 *  - The light curve is on a regular time grid (R1): the library checks
 *    max_n |times[n] - times[0] - n*c| <= 1e-3*c with c = (times[n-1]-times[0])/(n-1), else
 *    CETRA_ERR_NONUNIFORM_TIMES.  Null points (gaps, padding) are marked by a non-finite flux or a
 *    non-finite / non-positive flux_err.  flux is normalised to baseline 1;
 *    internally f = 1 - flux (R7).
 *  - The t0 grid is t_i = t0_start + i*t0_stride, i < n_t0, any start and any stride > 0.
 *    When every t0 cell lies on a sample (to 1e-6 cadence at the last cell: |a - round a| + |b - round b| (n_t0-1)
 *    <= 1e-6 with a = (t0_start - times[0])/c, b = t0_stride/c, b >= 1)
 *    the nearest-neighbour template position comes from the integer sample offset (R3) and the
 *    tabulated-tap kernel runs; otherwise it comes from the time difference
 *    x = (n*c - (t_i - times[0]))/D + 1/2 in FP64 (R25).  Off the sample grid a stride that is a small rational
 *    multiple of the cadence (the paper's default, 1 % of the shortest duration: 18 s on 2-min data = 3/20) is
 *    split into residue classes of cells, each an on-grid problem for the same tabulated-tap kernel with its own
 *    tap tables; any other stride takes a per-cell kernel that steps the position in fixed point.  Both evaluate
 *    the exact R25 sequence only where a position lies within a proven rounding bound of a decision point
 *    (cetra_exact_eval_count), so the result is the definition's on every path.  t0_start may lie before times[0] or t_i after times[n-1]: windows are clipped to the
 *    data (R9), which is the paper's null padding expressed through the grid.
 *  - Grids are stored [n_dur][n_t0], t0 contiguous, float32.  Cells whose window holds no
 *    observation are NaN in all three grids.
 *  - Arithmetic: FP32 products and sums on the CUDA cores, FP64 for every
 *    quantity that decides an integer (template index R3, epoch cell R11).
 */
#ifndef CETRA_H_
#define CETRA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    CETRA_OK = 0,
    CETRA_ERR_INVALID_ARG = -1,       /* null pointer, non-positive size, duration <= 0, period < t0_stride ... */
    CETRA_ERR_NONUNIFORM_TIMES = -2,  /* times[] is not a regular grid */
    CETRA_ERR_UNSUPPORTED = -3,       /* too many durations, index overflow */
    CETRA_ERR_WORKSPACE = -4,         /* workspace null, misaligned or smaller than *_workspace_bytes */
    CETRA_ERR_CUDA = -5,              /* a CUDA runtime call failed (cudaGetLastError is left set) */
    CETRA_ERR_STATIC_LIMIT = -6       /* cetra_resample_static: n_lc * n_out exceeds CETRA_RESAMPLE_STATIC_MAX_POINTS */
} cetra_status;

typedef enum { CETRA_F32 = 0, CETRA_F64 = 1 } cetra_dtype;

#define CETRA_MAX_DURATIONS 128

/* Uniform grid of trial mid-transit times. */
typedef struct {
    double t0_start;    /* days, same origin as times[] */
    double t0_stride;   /* days, > 0 */
    int64_t n_t0;       /* number of cells I */
} cetra_t0_grid;

/* One record of the periodogram: the maximum-likelihood element of one trial
 * period.  A period with no candidate has lr = depth = depth_var = t0 = NaN and indices -1. */
typedef struct {
    float lr;           /* log-likelihood gain of the periodic model over the flat model (Eq. 4 summed) */
    float depth;        /* common depth Z */
    float depth_var;    /* its variance; SNR = depth / sqrt(depth_var) */
    float t0;           /* t0_start + i_t0 * t0_stride in days, ROUNDED TO FLOAT32: a convenience value.  i_t0 is the
                         * result; with a large time origin (BJD - 2 457 000 ~ 3e3 d: float32 resolves 20 s; full BJD:
                         * 0.25 d) recompute the time from i_t0 in double, or keep times relative to the first sample
                         * as the paper does */
    int32_t i_t0;       /* cell of the first epoch, in [0, ceil(P/stride)) */
    int32_t j_dur;      /* duration index */
    int32_t n_transits; /* epochs that contributed (non-null cells) */
    int32_t reserved;
} cetra_peak;

const char *cetra_status_string(int status);

/* Number of SMs / shared memory the library will size its persistent grids for (device of the
 * current context).  Returns CETRA_OK or CETRA_ERR_CUDA. */
int cetra_device_info(int32_t *n_sm, int32_t *smem_per_block_optin);

/* ------------------------------------------------------------------------------------------
 * Linear search (§2.2).
 *
 *  times_host     [n]            float64 days, regular cadence
 *  flux_dev       [n_lc][n]      dtype (float32 or float64), baseline 1
 *  flux_err_dev   [n_lc][n]      dtype
 *  durations_host [n_dur]        float64 days, > 0, n_dur <= CETRA_MAX_DURATIONS
 *  template_host  [n_template]   float32, tpl[0] = first contact ... tpl[n_template-1] = last contact,
 *                                normalised to maximum depth 1; sampled nearest-
 *                                neighbour: idx = floor(x*(M-1)+1/2), x = (t_n - t_i)/D_j + 1/2 (R3)
 *  depth_dev, var_dev, dlogL_dev  [n_lc][n_dur][n_t0] float32 outputs (any of them may be NULL):
 *        depth = S_wmf/S_wmm,  var = 1/S_wmm,  dlogL = Eq. 2 = 1/2 S_wmf^2/S_wmm.
 *  stats_dev      optional output (may be NULL): the sufficient statistics (S_wmm, S_wmf) as float2,
 *                 [n_lc][n_dur][cetra_stats_pitch(n_t0)], zero in null cells and in the row padding;
 *                 this is the form cetra_periodic_search_stats consumes.
 *  Limits: n_lc <= 65 535 per call (light curves are one dimension of the launch grid; more return
 *  CETRA_ERR_UNSUPPORTED: call once per slice of curves, or use cetra_search_batched, which slices by itself).
 * ------------------------------------------------------------------------------------------ */
size_t cetra_linear_workspace_bytes(const double *times_host, int64_t n, int32_t n_lc,
                                    const double *durations_host, int32_t n_dur,
                                    cetra_t0_grid grid, int32_t n_template);

int cetra_linear_search(const double *times_host, const void *flux_dev, const void *flux_err_dev,
                        cetra_dtype dtype, int64_t n, int32_t n_lc,
                        const double *durations_host, int32_t n_dur, cetra_t0_grid grid,
                        const float *template_host, int32_t n_template,
                        float *depth_dev, float *var_dev, float *dlogL_dev, float *stats_dev,
                        void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* t0 grids off the sample grid (the paper's default stride is 1 % of the shortest duration; DESIGN.md
 * R25) are searched without evaluating the definition's FP64 expression for every (cell, sample) pair: the
 * nearest-neighbour template sample is taken from a position computed once per residue class of cells (stride /
 * cadence rational) or by fixed-point stepping (any stride), and only pairs whose position lies within a proven
 * rounding bound of a decision point (an index step, a window edge) are evaluated with the exact R25 sequence, so the
 * result is the definition's.  This diagnostic returns how many exact evaluations the device has done since the last
 * reset.  Synchronises the device.  count may be NULL.  Returns CETRA_OK or CETRA_ERR_CUDA. */
int cetra_exact_eval_count(int64_t *count, int32_t reset);

/* Row pitch (in cells) of the sufficient-statistics grid for n_t0 cells. */
int64_t cetra_stats_pitch(int64_t n_t0);

/* ------------------------------------------------------------------------------------------
 * Periodic search (§2.3).
 *
 *  depth_dev, var_dev  [n_lc][n_dur][n_t0] float32: the linear-search grids (NaN = null cell).
 *  dlogL_dev      [n_lc][n_dur][n_t0] float32 or NULL: the per-transit likelihood ratios LR_e that Eq. 4 sums
 *        (PAPER.md:137-143).  Eq. 4 summed at the common depth Z is
 *            sum_e [LR_e - 1/2 (depth_e - Z)^2 / var_e] = sum_e (LR_e - 1/2 depth_e^2 / var_e) + 1/2 (sum B)^2 / sum A,
 *        A = 1/var, B = depth/var.  For the linear search's own grids the first sum vanishes (LR_e = Eq. 2 =
 *        1/2 depth_e^2 / var_e, P2) and the search runs on the two sufficient statistics; that is also
 *        what NULL means.  When the grid passed here differs from 1/2 depth^2/var in some cell by more than 1e-5
 *        of it (e.g. full log-likelihoods), the call searches with the literal three-term sum
 *        instead (a plain, slower kernel; decided on the device, the call stays asynchronous), so the records
 *        are Eq. 4's for whatever grid the caller supplies (R20).
 *  periods_host   [n_per] float64 days, each >= t0_stride
 *  dur_lo_host, dur_hi_host  optional [n_per] int32: half-open duration-index range searched for each
 *        period; NULL = every duration.  Durations with D_j >= P_k are always skipped
 *        (PAPER.md:145).
 *  peaks_dev      [n_lc][n_per] output records.  Ties in lr: smallest j_dur, then smallest i_t0 (R13).
 *
 * Epoch e of phase p uses cell p + llrint(e * (P/stride)) (FP64, R11) while that is <= n_t0-1.
 * ------------------------------------------------------------------------------------------ */
size_t cetra_periodic_workspace_bytes(int32_t n_lc, int32_t n_dur, cetra_t0_grid grid, int32_t n_per);

int cetra_periodic_search(const float *depth_dev, const float *var_dev, const float *dlogL_dev,
                          int32_t n_lc, int32_t n_dur, cetra_t0_grid grid,
                          const double *durations_host, const double *periods_host, int32_t n_per,
                          const int32_t *dur_lo_host, const int32_t *dur_hi_host,
                          cetra_peak *peaks_dev,
                          void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Same search on the sufficient statistics written by cetra_linear_search (stats_dev). */
int cetra_periodic_search_stats(const float *stats_dev, int32_t n_lc, int32_t n_dur, cetra_t0_grid grid,
                                const double *durations_host, const double *periods_host, int32_t n_per,
                                const int32_t *dur_lo_host, const int32_t *dur_hi_host,
                                cetra_peak *peaks_dev,
                                void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* ------------------------------------------------------------------------------------------
 * Batched search: n_lc light curves sharing one timestamp array, linear search then
 * periodic search per chunk of light curves; the per-curve grids live only in the workspace.
 * Arguments as above.  `lc_chunk` light curves are resident at a time (0 = library default; a larger request is
 * clamped to 65 535, the most one linear-search launch takes).  n_lc itself is not limited.
 * ------------------------------------------------------------------------------------------ */
size_t cetra_search_batched_workspace_bytes(const double *times_host, int64_t n, int32_t n_lc, int32_t lc_chunk,
                                            const double *durations_host, int32_t n_dur, cetra_t0_grid grid,
                                            int32_t n_template, int32_t n_per);

int cetra_search_batched(const double *times_host, const void *flux_dev, const void *flux_err_dev,
                         cetra_dtype dtype, int64_t n, int32_t n_lc, int32_t lc_chunk,
                         const double *durations_host, int32_t n_dur, cetra_t0_grid grid,
                         const float *template_host, int32_t n_template,
                         const double *periods_host, int32_t n_per,
                         const int32_t *dur_lo_host, const int32_t *dur_hi_host,
                         cetra_peak *peaks_dev,
                         void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Same search for a set of transit templates in one pass ("it may be worth running CETRA across a sequence of
 * values" of the impact parameter): templates_host is [n_templates][n_template] float32, peaks_dev is
 * [n_templates][n_lc][n_per]; template t's records are bit for bit those of cetra_search_batched with that template.
 * Per chunk of light curves the samples are preprocessed once, the tap tables of all templates are built in one
 * launch, and ONE linear-search launch (grid y = template x duration) writes the statistics grids of every template
 * from those samples; the fold then runs once per template.  The workspace holds one statistics grid per template:
 * query it with cetra_search_batched_templates_workspace_bytes (n_templates x n_dur <= 65 535). */
size_t cetra_search_batched_templates_workspace_bytes(const double *times_host, int64_t n, int32_t n_lc,
                                                      int32_t lc_chunk, const double *durations_host, int32_t n_dur,
                                                      cetra_t0_grid grid, int32_t n_template, int32_t n_templates,
                                                      int32_t n_per);

int cetra_search_batched_templates(const double *times_host, const void *flux_dev, const void *flux_err_dev,
                                   cetra_dtype dtype, int64_t n, int32_t n_lc, int32_t lc_chunk,
                                   const double *durations_host, int32_t n_dur, cetra_t0_grid grid,
                                   const float *templates_host, int32_t n_template, int32_t n_templates,
                                   const double *periods_host, int32_t n_per,
                                   const int32_t *dur_lo_host, const int32_t *dur_hi_host,
                                   cetra_peak *peaks_dev,
                                   void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Same, with the light curves and the result in HOST memory (pinned memory recommended): each chunk is
 * copied host->device, searched, and its records copied device->host on `cuda_stream`; the call
 * synchronises the stream before returning.  The workspace must be
 * cetra_search_batched_host_workspace_bytes (it also stages the inputs and the records). */
size_t cetra_search_batched_host_workspace_bytes(const double *times_host, int64_t n, int32_t n_lc, int32_t lc_chunk,
                                                 cetra_dtype dtype,
                                                 const double *durations_host, int32_t n_dur, cetra_t0_grid grid,
                                                 int32_t n_template, int32_t n_per);

int cetra_search_batched_host(const double *times_host, const void *flux_host, const void *flux_err_host,
                              cetra_dtype dtype, int64_t n, int32_t n_lc, int32_t lc_chunk,
                              const double *durations_host, int32_t n_dur, cetra_t0_grid grid,
                              const float *template_host, int32_t n_template,
                              const double *periods_host, int32_t n_per,
                              const int32_t *dur_lo_host, const int32_t *dur_hi_host,
                              cetra_peak *peaks_host,
                              void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Transit model -> search template ("The chosen/supplied model is ultimately resampled to a
 * user-defined number of samples using simple linear interpolation").  model_host [n_model] float32 spans first to
 * last contact; template_host [n_template] receives the model at n_template evenly spaced positions over the same
 * span (both end samples kept), interpolated linearly in FP64 and rounded to float32.  A host-side setup helper
 * (no device work).  Returns CETRA_OK or CETRA_ERR_INVALID_ARG (null pointer, fewer than 2 samples). */
int cetra_resample_template(const float *model_host, int32_t n_model, float *template_host, int32_t n_template);

/* ------------------------------------------------------------------------------------------
 * Setup: light-curve resampling (§2.1.1, lines 53-61).
 *
 * cetra_median_cadence   host-only: the default resample cadence, the median of the differences of
 *                        the time-sorted finite timestamps (R22).
 * cetra_resample_grid    host-only: the regular output grid for `times_host`: cadence (<= 0: the median
 *                        cadence), `pad_days` of null padding at both ends (half the maximum
 *                        trial duration), rounded up to whole points.  Output point n is at
 *                        t_start + n * cadence; the first observation falls on point ceil(pad/cadence).
 * cetra_resample         every observation goes to the nearest output point,
 *                        cell = floor((t - t_start)/cadence + 1/2) in FP64 (R21); observations sharing a
 *                        point are combined with the inverse-variance weighted mean, error
 *                        (sum 1/sigma^2)^-1/2; points without data get flux = NaN, flux_err = +inf
 *                        (PAPER.md:55).  Null observations (non-finite time/flux/error, error <= 0) and
 *                        observations off the grid are dropped.  The input needs no ordering.
 *     times_dev              [n_in] float64 DEVICE (the irregular timestamps are a large array)
 *     flux_dev, flux_err_dev [n_lc][n_in] dtype, sharing times_dev
 *     flux_out_dev, flux_err_out_dev [n_lc][n_out] dtype (same dtype as the input); n_in = 0 gives an all-null grid
 *     workspace              cetra_resample_workspace_bytes(n_in, n_lc, n_out): four int32 arrays (the output point of
 *                            every observation, the observations of every point, counts, offsets); it does not grow
 *                            with n_lc, because the light curves share the timestamps
 * The observation -> point lists are built once per call for all light curves, and each (light curve, point) sum adds
 * its observations in ascending input index in FP64: no floating-point atomics, so the result is bit-identical from
 * run to run and equals a sequential pass over the input; it does not depend on the order of the input beyond FP64
 * rounding.  Limits: n_in < 2^31, n_out < 2^31 - 1 (CETRA_ERR_UNSUPPORTED beyond).
 * ------------------------------------------------------------------------------------------ */
int cetra_median_cadence(const double *times_host, int64_t n, double *cadence);

int cetra_resample_grid(const double *times_host, int64_t n, double cadence, double pad_days,
                        double *t_start, double *cadence_out, int64_t *n_out);

size_t cetra_resample_workspace_bytes(int64_t n_in, int32_t n_lc, int64_t n_out);

int cetra_resample(const double *times_dev, const void *flux_dev, const void *flux_err_dev, cetra_dtype dtype,
                   int64_t n_in, int32_t n_lc, double t_start, double cadence, int64_t n_out,
                   void *flux_out_dev, void *flux_err_out_dev,
                   void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* ------------------------------------------------------------------------------------------
 * cetra_resample for callers that have no device memory to give as a workspace.
 *
 * Who this is for.  cetra_resample needs cetra_resample_workspace_bytes() of device scratch (index lists that grow
 * with the number of observations).  Some callers cannot produce that: code that runs inside somebody else's memory budget and is
 * handed its input and output buffers but no allocator (a plug-in stage of a pipeline, a worker whose device pool
 * was carved up front and is full), code on a path where cudaMalloc is not allowed because it synchronises the
 * whole device (a latency-critical service loop, a region other threads are capturing or timing), and code in a
 * process whose memory is accounted for by a framework that forbids allocations behind its back.  For them this
 * entry point keeps the sums in a fixed array that is part of the library image itself.
 *
 * What it costs.  The array is CETRA_RESAMPLE_STATIC_MAX_POINTS pairs of doubles = 4 MiB of device memory on every
 * GPU that loads the library, from the moment the library's CUDA module is loaded on that GPU until the process
 * exits, whether or not this function is ever called.
 *
 * Limit.  n_lc * n_out <= CETRA_RESAMPLE_STATIC_MAX_POINTS (262 144 output points over all light curves of the
 * call: e.g. 13 TESS 2-min sectors of ~20 000 points).  A larger request is refused with
 * CETRA_ERR_STATIC_LIMIT before anything is enqueued; split the light curves over several calls, or use
 * cetra_resample with a workspace.  cetra_resample_static_max_points() returns the limit at run time.
 *
 * Arguments and results are cetra_resample's.  The sums here are FP64 atomic adds into the fixed array (one pair per
 * output point, which is what bounds n_lc * n_out), so their order varies from run to run: the two entry points agree
 * to FP64 rounding of the sums, i.e. after rounding to the output dtype to within one unit in the last place.
 * The call makes no cudaMalloc / cudaFree and calls nothing that allocates; it enqueues one memset of the part of
 * the array it uses and two kernels on `cuda_stream` and returns without synchronising.
 *
 * First call on each device.  The address of the array on the current device is looked up once per device
 * (cudaGetSymbolAddress, with that device current) the first time this function runs there, and remembered.  That
 * lookup may load the library's CUDA module, so make the first call on each device during set-up, outside any
 * stream capture and outside any region where module loading is unwelcome.
 *
 * Sharing.  Every call on a device uses the same array, from offset 0, and leaves its sums behind; each call
 * clears the part it is about to use, so earlier calls never leak into later ones.  Two calls that can run on the
 * GPU at the same time (different streams of one device without an ordering between them, or two host threads)
 * overwrite each other's sums and both give wrong answers: order them on one stream or with events.  Different
 * devices have separate copies and do not interact.
 *
 * Returns CETRA_OK, CETRA_ERR_INVALID_ARG (as cetra_resample), CETRA_ERR_STATIC_LIMIT, CETRA_ERR_UNSUPPORTED
 * (device ordinal >= 64) or CETRA_ERR_CUDA (no device, symbol lookup or launch failed).
 * ------------------------------------------------------------------------------------------ */
#define CETRA_RESAMPLE_STATIC_MAX_POINTS 262144

int64_t cetra_resample_static_max_points(void);

int cetra_resample_static(const double *times_dev, const void *flux_dev, const void *flux_err_dev, cetra_dtype dtype,
                          int64_t n_in, int32_t n_lc, double t_start, double cadence, int64_t n_out,
                          void *flux_out_dev, void *flux_err_out_dev, void *cuda_stream);

/* ------------------------------------------------------------------------------------------
 * Monotransit search: single-transit events in the linear-search output alone.
 *
 *  profile(i) = max_j dlogL[j][i] (null cells skipped; ties: smallest j).  Events are taken greedily by
 *  decreasing profile (ties: smallest i); an event at (i, j) removes every reference time with
 *  |t - t_i| <= excl * D_j from further consideration (R23).
 *
 *  depth_dev, var_dev, dlogL_dev  [n_lc][n_dur][n_t0] float32, the linear-search grids
 *  profile_lr_dev  optional [n_lc][n_t0] float32 (NaN where every duration is null)
 *  profile_j_dev   optional [n_lc][n_t0] int32   (-1 there)
 *  events_dev      [n_lc][n_peaks] records; entries beyond n_found are NaN / -1
 *  n_found_dev     [n_lc] int32
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    float lr;           /* dlogL of the event (Eq. 2) */
    float depth;
    float depth_var;
    float t0;           /* t0_start + i_t0 * t0_stride */
    int32_t i_t0;
    int32_t j_dur;
    int32_t reserved[2];
} cetra_event;

size_t cetra_monotransit_workspace_bytes(int32_t n_lc, int64_t n_t0);

int cetra_monotransit_search(const float *depth_dev, const float *var_dev, const float *dlogL_dev,
                             int32_t n_lc, int32_t n_dur, cetra_t0_grid grid, const double *durations_host,
                             int32_t n_peaks, double excl,
                             float *profile_lr_dev, int32_t *profile_j_dev,
                             cetra_event *events_dev, int32_t *n_found_dev,
                             void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* ------------------------------------------------------------------------------------------
 * Iterative masking: nullify the flux within and around a detected signal before the
 * search is repeated.  Sample n of light curve b is set to NaN when its distance to the nearest transit
 * mid-time t0[b] + e * period[b] (e any integer; period[b] <= 0: the single event at t0[b]) is
 * <= width * duration[b] / 2 (R24), all in FP64.
 *
 *  times_dev       [n] float64 DEVICE
 *  flux_dev        [n_lc][n] dtype, modified in place
 *  period_host, t0_host, duration_host  [n_lc] float64 (a light curve with a non-finite t0 or a
 *                  non-positive duration is left untouched)
 *  n_masked_dev    optional [n_lc] int32: samples nullified by this call
 *  workspace       cetra_mask_workspace_bytes(n_lc)
 * ------------------------------------------------------------------------------------------ */
size_t cetra_mask_workspace_bytes(int32_t n_lc);

int cetra_mask_transits(const double *times_dev, void *flux_dev, cetra_dtype dtype, int64_t n, int32_t n_lc,
                        const double *period_host, const double *t0_host, const double *duration_host,
                        double width, int32_t *n_masked_dev,
                        void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Number of kernel launches the library has enqueued since the process started (diagnostic). */
int64_t cetra_kernel_launch_count(void);

/* Test hook, not a tuning knob: overrides the periodic search's choice of fold kernel for every later call in
 * this process, so that the parity tests can send small problems (which the oracle folds in full) through the kernel
 * that normally serves only rows too large for shared memory.  force_stream != 0: rows that fit in shared memory are
 * streamed anyway; stage_cells >= 64: the streamed kernel's stages hold that many cells instead of a full share of
 * shared memory (epoch blocks split, wide windows gathered directly).  (0, 0) restores the library's own plan, which
 * is the only one production code should run: the overridden plans give the same records, more slowly.
 * The library reads no environment variable; this call is the only way to change the plan.  Not thread-safe with
 * respect to searches running concurrently on other host threads. */
void cetra_test_fold_override(int32_t force_stream, int32_t stage_cells);

/* Diagnostics for bench.py's roofline line.  While enabled, the library brackets every launch of its two
 * hot kernels (the windowed-sum linear-search kernel and the fold-gather-argmax periodic-search kernel)
 * with a pair of CUDA events recorded on the launching stream; nothing is synchronised at launch time.
 * The events are the only objects the library ever creates; cetra_profile_enable(0) destroys them.
 * cetra_profile_read waits for the recorded events, returns the summed device time (milliseconds) and the
 * number of launches of each kernel since the last reset, and resets the counters if `reset` is non-zero.
 * Any output pointer may be NULL.  Not thread-safe. */
int cetra_profile_enable(int32_t enable);
int cetra_profile_read(double *linear_ms, int64_t *linear_launches, double *fold_ms, int64_t *fold_launches,
                       int32_t reset);

#ifdef __cplusplus
}
#endif
#endif /* CETRA_H_ */

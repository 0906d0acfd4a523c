// C ABI of the CETRA B200 library: argument validation, workspace carve-up, launch order.
// Every step of the path runs in the kernels of linear_search.cu / periodic_search.cu; nothing here
// computes any of the method's arithmetic on the host, and there is no CPU fallback.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "linear_search.cuh"
#include "periodic_search.cuh"

namespace cetra {

std::atomic<int64_t> g_launch_count{0};

// ---- optional profiling events (diagnostics only) ----
struct ProfileState {
    bool on = false;
    std::vector<cudaEvent_t> begin[2], end[2];
    double ms[2] = {0.0, 0.0};
    int64_t launches[2] = {0, 0};
};
static ProfileState g_prof;

void profile_mark(ProfiledKernel which, bool begin, cudaStream_t st) {
    if (!g_prof.on) return;
    cudaEvent_t ev;
    if (cudaEventCreate(&ev) != cudaSuccess) return;
    cudaEventRecord(ev, st);
    (begin ? g_prof.begin[which] : g_prof.end[which]).push_back(ev);
}

static void profile_drain() {
    for (int w = 0; w < 2; ++w) {
        const size_t n = std::min(g_prof.begin[w].size(), g_prof.end[w].size());
        for (size_t i = 0; i < n; ++i) {
            float ms = 0.f;
            if (cudaEventSynchronize(g_prof.end[w][i]) == cudaSuccess &&
                cudaEventElapsedTime(&ms, g_prof.begin[w][i], g_prof.end[w][i]) == cudaSuccess) {
                g_prof.ms[w] += ms;
                g_prof.launches[w] += 1;
            }
        }
        for (cudaEvent_t e : g_prof.begin[w]) cudaEventDestroy(e);
        for (cudaEvent_t e : g_prof.end[w]) cudaEventDestroy(e);
        g_prof.begin[w].clear();
        g_prof.end[w].clear();
    }
}

// DESIGN.md R1/R9: the samples are a regular grid; the t0 grid sits on it with a whole-sample stride.
int derive_geometry(const double *times_host, int64_t n, cetra_t0_grid grid, Geometry *g) {
    if (!times_host || n < 2 || !(grid.t0_stride > 0.0) || !std::isfinite(grid.t0_stride) ||
        !std::isfinite(grid.t0_start) || grid.n_t0 < 1)
        return CETRA_ERR_INVALID_ARG;
    const double c = (times_host[n - 1] - times_host[0]) / static_cast<double>(n - 1);
    if (!(c > 0.0) || !std::isfinite(c)) return CETRA_ERR_INVALID_ARG;
    for (int64_t i = 0; i < n; ++i)
        if (!(fabs(times_host[i] - times_host[0] - static_cast<double>(i) * c) <= 1e-3 * c))
            return CETRA_ERR_NONUNIFORM_TIMES;
    const double a = (grid.t0_start - times_host[0]) / c;
    const double b = grid.t0_stride / c;
    if (!(fabs(a) < 1e15) || !(b < 1e15)) return CETRA_ERR_UNSUPPORTED;
    const long long ia = llrint(a), ib = llrint(b);
    g->cadence = c;
    g->delta = grid.t0_start - times_host[0];
    g->stride = grid.t0_stride;
    // on the sample grid iff no cell of the t0 grid is further than 1e-6 samples from a sample: the mismatch of
    // the stride accumulates over the grid, so it is bounded at the last cell (R25)
    const double drift = fabs(a - static_cast<double>(ia)) +
                         fabs(b - static_cast<double>(ib)) * static_cast<double>(grid.n_t0 - 1);
    g->on_grid = !(drift > 1e-6 || ib < 1);
    g->n0 = g->on_grid ? ia : 0;
    g->q = g->on_grid ? ib : 0;
    g->rational = false;
    g->cls = 1;
    g->drift = 0.0;
    if (!g->on_grid) {
        // continued-fraction convergents of stride / cadence with a denominator of at most kMaxClasses
        long long p0 = 0, q0 = 1, p1 = 1, q1 = 0;
        double x = b;
        for (int it = 0; it < 40; ++it) {
            const double fl = floor(x);
            if (!(fl < 1e9)) break;
            const long long ai = static_cast<long long>(fl);
            const long long p2 = ai * p1 + p0, q2 = ai * q1 + q0;
            if (q2 > kMaxClasses || p2 > kMaxClassStride) break;
            p0 = p1; q0 = q1; p1 = p2; q1 = q2;
            const double fr = x - fl;
            if (fabs(b - static_cast<double>(p1) / static_cast<double>(q1)) * static_cast<double>(grid.n_t0) <= 1e-9 ||
                !(fr > 1e-12))
                break;
            x = 1.0 / fr;
        }
        if (q1 >= 1 && p1 >= 1) {
            const double dr = fabs(b - static_cast<double>(p1) / static_cast<double>(q1)) * static_cast<double>(grid.n_t0);
            if (dr <= 1e-6) {
                g->rational = true;
                g->q = p1;
                g->cls = q1;
                g->drift = dr + 1e-12;
            }
        }
    }
    return CETRA_OK;
}

struct Device {
    int n_sm = 0, smem_optin = 0;
};

static int query_device(Device *d) {
    int dev = 0;
    CETRA_CUDA_TRY(cudaGetDevice(&dev));
    CETRA_CUDA_TRY(cudaDeviceGetAttribute(&d->n_sm, cudaDevAttrMultiProcessorCount, dev));
    CETRA_CUDA_TRY(cudaDeviceGetAttribute(&d->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    return CETRA_OK;
}

// Plans are sized for a B200 when no device is visible (workspace queries on a CPU-only host).
static Device device_or_default() {
    Device d;
    if (query_device(&d) != CETRA_OK || d.n_sm <= 0) {
        cudaGetLastError();
        d.n_sm = 148;
        d.smem_optin = 232448;
    }
    return d;
}

// The compute entry points refuse to run without a device: there is no CPU fallback.
static int require_device() {
    Device d;
    const int rc = query_device(&d);
    if (rc != CETRA_OK) cudaGetLastError();
    return rc;
}

static bool aligned(const void *p) { return (reinterpret_cast<uintptr_t>(p) & (kAlign - 1)) == 0; }

static size_t stats_bytes(int32_t n_lc, int32_t n_dur, int64_t n_t0) {
    return align_up(sizeof(float2) * static_cast<size_t>(n_lc) * n_dur * static_cast<size_t>(cetra_stats_pitch(n_t0)));
}

static size_t dtype_size(cetra_dtype t) { return t == CETRA_F64 ? 8 : 4; }

}  // namespace cetra

using namespace cetra;

extern "C" {

const char *cetra_status_string(int status) {
    switch (status) {
        case CETRA_OK: return "ok";
        case CETRA_ERR_INVALID_ARG: return "invalid argument";
        case CETRA_ERR_NONUNIFORM_TIMES: return "times[] is not a regular grid";
        case CETRA_ERR_UNSUPPORTED: return "unsupported configuration";
        case CETRA_ERR_WORKSPACE: return "workspace null, misaligned or too small";
        case CETRA_ERR_CUDA: return "CUDA runtime error";
        case CETRA_ERR_STATIC_LIMIT:
            return "request exceeds the library's built-in scratch (cetra_resample_static: n_lc * n_out > 262144)";
        default: return "unknown status";
    }
}

int cetra_device_info(int32_t *n_sm, int32_t *smem_per_block_optin) {
    Device d;
    const int rc = query_device(&d);
    if (rc != CETRA_OK) return rc;
    if (n_sm) *n_sm = d.n_sm;
    if (smem_per_block_optin) *smem_per_block_optin = d.smem_optin;
    return CETRA_OK;
}

int64_t cetra_stats_pitch(int64_t n_t0) { return round_up64(n_t0 + kStatsPad, 32); }

int64_t cetra_kernel_launch_count(void) { return g_launch_count.load(); }

int cetra_profile_enable(int32_t enable) {
    profile_drain();
    g_prof.on = enable != 0;
    g_prof.ms[0] = g_prof.ms[1] = 0.0;
    g_prof.launches[0] = g_prof.launches[1] = 0;
    return CETRA_OK;
}

int cetra_profile_read(double *linear_ms, int64_t *linear_launches, double *fold_ms, int64_t *fold_launches,
                       int32_t reset) {
    profile_drain();
    if (linear_ms) *linear_ms = g_prof.ms[kProfLinear];
    if (linear_launches) *linear_launches = g_prof.launches[kProfLinear];
    if (fold_ms) *fold_ms = g_prof.ms[kProfFold];
    if (fold_launches) *fold_launches = g_prof.launches[kProfFold];
    if (reset) {
        g_prof.ms[0] = g_prof.ms[1] = 0.0;
        g_prof.launches[0] = g_prof.launches[1] = 0;
    }
    return cudaGetLastError() == cudaSuccess ? CETRA_OK : CETRA_ERR_CUDA;
}

// ------------------------------------------------------------------------------------------ linear
size_t cetra_linear_workspace_bytes(const double *times_host, int64_t n, int32_t n_lc, const double *durations_host,
                                    int32_t n_dur, cetra_t0_grid grid, int32_t n_template) {
    const Device d = device_or_default();
    LinearPlan pl;
    if (build_linear_plan(times_host, n, n_lc, durations_host, n_dur, grid, n_template, d.smem_optin, d.n_sm, &pl) !=
        CETRA_OK)
        return 0;
    return linear_workspace_bytes(pl, n_lc, n_template);
}

int cetra_linear_search(const double *times_host, const void *flux_dev, const void *flux_err_dev, cetra_dtype dtype,
                        int64_t n, int32_t n_lc, const double *durations_host, int32_t n_dur, cetra_t0_grid grid,
                        const float *template_host, int32_t n_template, float *depth_dev, float *var_dev,
                        float *dlogL_dev, float *stats_dev, void *workspace_dev, size_t workspace_bytes,
                        void *cuda_stream) {
    if (!flux_dev || !flux_err_dev || !template_host || (dtype != CETRA_F32 && dtype != CETRA_F64))
        return CETRA_ERR_INVALID_ARG;
    const Device d = device_or_default();   // argument errors are reported even where no device is visible
    int rc;
    LinearPlan pl;
    rc = build_linear_plan(times_host, n, n_lc, durations_host, n_dur, grid, n_template, d.smem_optin, d.n_sm, &pl);
    if (rc != CETRA_OK) return rc;
    if (!workspace_dev || !aligned(workspace_dev) || workspace_bytes < linear_workspace_bytes(pl, n_lc, n_template))
        return CETRA_ERR_WORKSPACE;
    if ((rc = require_device()) != CETRA_OK) return rc;
    return run_linear(pl, flux_dev, flux_err_dev, dtype, n, n_lc, template_host, n_template, false, depth_dev,
                      var_dev, dlogL_dev, stats_dev, workspace_dev, static_cast<cudaStream_t>(cuda_stream));
}

int cetra_exact_eval_count(int64_t *count, int32_t reset) {
    const int rc = require_device();
    if (rc != CETRA_OK) return rc;
    return exact_eval_count(count, reset != 0);
}

// ---------------------------------------------------------------------------------------- periodic
size_t cetra_periodic_workspace_bytes(int32_t n_lc, int32_t n_dur, cetra_t0_grid grid, int32_t n_per) {
    if (n_lc < 1 || n_dur < 1 || n_per < 1 || grid.n_t0 < 1) return 0;
    // keys and period arrays, the (S_wmm, S_wmf) rows, and for a caller's likelihood-ratio grid its residual rows + flag
    return periodic_workspace_bytes(n_lc, n_per) + stats_bytes(n_lc, n_dur, grid.n_t0) +
           align_up(stats_bytes(n_lc, n_dur, grid.n_t0) / 2) + kAlign;
}

int cetra_periodic_search_stats(const float *stats_dev, int32_t n_lc, int32_t n_dur, cetra_t0_grid grid,
                                const double *durations_host, const double *periods_host, int32_t n_per,
                                const int32_t *dur_lo_host, const int32_t *dur_hi_host, cetra_peak *peaks_dev,
                                void *workspace_dev, size_t workspace_bytes, void *cuda_stream) {
    if (!stats_dev || !peaks_dev || ((dur_lo_host == nullptr) != (dur_hi_host == nullptr)))
        return CETRA_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(stats_dev) & 15) != 0) return CETRA_ERR_INVALID_ARG;
    const Device d = device_or_default();   // argument errors are reported even where no device is visible
    int rc;
    PeriodicPlan pl;
    rc = build_periodic_plan(n_lc, n_dur, grid, durations_host, periods_host, n_per, d.smem_optin, d.n_sm, &pl);
    if (rc != CETRA_OK) return rc;
    if (!workspace_dev || !aligned(workspace_dev) || workspace_bytes < periodic_workspace_bytes(n_lc, n_per))
        return CETRA_ERR_WORKSPACE;
    if ((rc = require_device()) != CETRA_OK) return rc;
    return run_periodic(pl, reinterpret_cast<const float2 *>(stats_dev), periods_host, dur_lo_host, dur_hi_host, true,
                        peaks_dev, workspace_dev, static_cast<cudaStream_t>(cuda_stream));
}

int cetra_periodic_search(const float *depth_dev, const float *var_dev, const float *dlogL_dev, int32_t n_lc,
                          int32_t n_dur, cetra_t0_grid grid, const double *durations_host,
                          const double *periods_host, int32_t n_per, const int32_t *dur_lo_host,
                          const int32_t *dur_hi_host, cetra_peak *peaks_dev, void *workspace_dev,
                          size_t workspace_bytes, void *cuda_stream) {
    if (!depth_dev || !var_dev || !peaks_dev || ((dur_lo_host == nullptr) != (dur_hi_host == nullptr)))
        return CETRA_ERR_INVALID_ARG;
    const Device d = device_or_default();   // argument errors are reported even where no device is visible
    int rc;
    PeriodicPlan pl;
    rc = build_periodic_plan(n_lc, n_dur, grid, durations_host, periods_host, n_per, d.smem_optin, d.n_sm, &pl);
    if (rc != CETRA_OK) return rc;
    if (!workspace_dev || !aligned(workspace_dev) ||
        workspace_bytes < cetra_periodic_workspace_bytes(n_lc, n_dur, grid, n_per))
        return CETRA_ERR_WORKSPACE;
    if ((rc = require_device()) != CETRA_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    char *ws = static_cast<char *>(workspace_dev);
    float2 *stats = reinterpret_cast<float2 *>(ws + periodic_workspace_bytes(n_lc, n_per));
    // dlogL given: Eq. 4 is summed with the caller's LR_e (R20); NULL: LR_e = 1/2 depth^2/var, the linear search's own
    float *resid = reinterpret_cast<float *>(ws + periodic_workspace_bytes(n_lc, n_per) + stats_bytes(n_lc, n_dur, grid.n_t0));
    int *literal = reinterpret_cast<int *>(reinterpret_cast<char *>(resid) + align_up(stats_bytes(n_lc, n_dur, grid.n_t0) / 2));
    rc = run_grids_to_stats(depth_dev, var_dev, dlogL_dev, n_lc * n_dur, grid.n_t0, stats, resid, literal, st);
    if (rc != CETRA_OK) return rc;
    return run_periodic(pl, stats, periods_host, dur_lo_host, dur_hi_host, true, peaks_dev, workspace_dev, st,
                        dlogL_dev ? resid : nullptr, dlogL_dev ? literal : nullptr);
}

// ----------------------------------------------------------------------------------------- batched
namespace {

struct BatchedLayout {
    int32_t chunk = 0;
    size_t linear_bytes = 0, stats_bytes = 0, periodic_bytes = 0, total = 0;
};

// Light curves resident at a time: by default as many as keep the chunk's (S_wmm, S_wmf) grids within
// 512 MiB of workspace.  Larger chunks mean fewer, longer launches (the linear kernel's ramp and tail are
// amortised: 43 % -> 50 % of the FP32 peak from 14 to 64 curves); the periodic search reads every row from
// global memory only a handful of times per launch, so L2 residency of the grids does not matter.
int32_t default_chunk(int32_t n_lc, int32_t n_dur, int64_t n_t0, int32_t n_templates) {
    const size_t per_lc = sizeof(float2) * static_cast<size_t>(n_dur) * static_cast<size_t>(cetra_stats_pitch(n_t0)) *
                          static_cast<size_t>(n_templates);
    const size_t budget = 512ull << 20;
    const size_t c = std::max<size_t>(1, budget / std::max<size_t>(per_lc, 1));
    // (65 535: light curves are the z dimension of the linear kernels' grids)
    return static_cast<int32_t>(std::min<size_t>(std::min<size_t>(c, 65535), static_cast<size_t>(n_lc)));
}

int plan_batched(const double *times_host, int64_t n, int32_t n_lc, int32_t lc_chunk, const double *durations_host,
                 int32_t n_dur, cetra_t0_grid grid, int32_t n_template, int32_t n_per, const Device &d,
                 LinearPlan *lin, BatchedLayout *lay, int32_t n_templates = 1) {
    if (n_lc < 1 || lc_chunk < 0 || n_per < 1 || n_templates < 1) return CETRA_ERR_INVALID_ARG;
    if (n_dur < 1 || grid.n_t0 < 1) return CETRA_ERR_INVALID_ARG;
    // light curves are the z dimension of the linear kernel's launch grid: a chunk holds at most 65 535 of them,
    // whatever the caller asked for (cetra.h)
    const int32_t chunk = lc_chunk > 0 ? std::min(std::min(lc_chunk, n_lc), static_cast<int32_t>(65535))
                                       : default_chunk(n_lc, n_dur, grid.n_t0, n_templates);
    const int rc = build_linear_plan(times_host, n, chunk, durations_host, n_dur, grid, n_template, d.smem_optin,
                                     d.n_sm, lin, n_templates);
    if (rc != CETRA_OK) return rc;
    lay->chunk = chunk;
    lay->linear_bytes = linear_workspace_bytes(*lin, chunk, n_template);
    lay->stats_bytes = stats_bytes(chunk, n_dur, grid.n_t0) * static_cast<size_t>(n_templates);   // one grid per template
    lay->periodic_bytes = periodic_workspace_bytes(chunk, n_per);
    lay->total = lay->linear_bytes + lay->stats_bytes + lay->periodic_bytes;
    return CETRA_OK;
}

// Linear search then periodic search for light curves [lc0, lc0 + m) of a chunked batch.  With a template set
// (lin.n_templates = T > 1) the light curves are preprocessed once and ONE linear launch writes the
// T statistics grids ([T][m][n_dur][pitch]); the fold then runs once per template (its work is per template by
// nature).  peaks_dev: records of light curve lc0 for template 0; template t's are peaks_tpl_stride records further.
int run_chunk(LinearPlan &lin, const BatchedLayout &lay, const Device &d, const void *flux_dev,
              const void *flux_err_dev, cetra_dtype dtype, int64_t n, int32_t m, bool first,
              const double *durations_host, int32_t n_dur, cetra_t0_grid grid, const float *template_host,
              int32_t n_template, const double *periods_host, int32_t n_per, const int32_t *dur_lo_host,
              const int32_t *dur_hi_host, cetra_peak *peaks_dev, size_t peaks_tpl_stride, char *ws, cudaStream_t st) {
    float *stats = reinterpret_cast<float *>(ws + lay.linear_bytes);
    int rc = run_linear(lin, flux_dev, flux_err_dev, dtype, n, m, template_host, n_template, false, nullptr, nullptr,
                        nullptr, stats, ws, st);
    if (rc != CETRA_OK) return rc;
    PeriodicPlan per;
    rc = build_periodic_plan(m, n_dur, grid, durations_host, periods_host, n_per, d.smem_optin, d.n_sm, &per);
    if (rc != CETRA_OK) return rc;
    const size_t grid_elems = static_cast<size_t>(m) * n_dur * static_cast<size_t>(cetra_stats_pitch(grid.n_t0));
    for (int t = 0; t < lin.n_templates; ++t) {
        rc = run_periodic(per, reinterpret_cast<const float2 *>(stats) + t * grid_elems, periods_host, dur_lo_host,
                          dur_hi_host, first && t == 0, peaks_dev + t * peaks_tpl_stride,
                          ws + lay.linear_bytes + lay.stats_bytes, st);
        if (rc != CETRA_OK) return rc;
    }
    return CETRA_OK;
}

}  // namespace

size_t cetra_search_batched_workspace_bytes(const double *times_host, int64_t n, int32_t n_lc, int32_t lc_chunk,
                                            const double *durations_host, int32_t n_dur, cetra_t0_grid grid,
                                            int32_t n_template, int32_t n_per) {
    const Device d = device_or_default();
    LinearPlan lin;
    BatchedLayout lay;
    if (plan_batched(times_host, n, n_lc, lc_chunk, durations_host, n_dur, grid, n_template, n_per, d, &lin, &lay) !=
        CETRA_OK)
        return 0;
    return lay.total;
}

int cetra_search_batched(const double *times_host, const void *flux_dev, const void *flux_err_dev, cetra_dtype dtype,
                         int64_t n, int32_t n_lc, int32_t lc_chunk, const double *durations_host, int32_t n_dur,
                         cetra_t0_grid grid, const float *template_host, int32_t n_template,
                         const double *periods_host, int32_t n_per, const int32_t *dur_lo_host,
                         const int32_t *dur_hi_host, cetra_peak *peaks_dev, void *workspace_dev,
                         size_t workspace_bytes, void *cuda_stream) {
    return cetra_search_batched_templates(times_host, flux_dev, flux_err_dev, dtype, n, n_lc, lc_chunk, durations_host,
                                          n_dur, grid, template_host, n_template, 1, periods_host, n_per, dur_lo_host,
                                          dur_hi_host, peaks_dev, workspace_dev, workspace_bytes, cuda_stream);
}

size_t cetra_search_batched_templates_workspace_bytes(const double *times_host, int64_t n, int32_t n_lc,
                                                      int32_t lc_chunk, const double *durations_host, int32_t n_dur,
                                                      cetra_t0_grid grid, int32_t n_template, int32_t n_templates,
                                                      int32_t n_per) {
    const Device d = device_or_default();
    LinearPlan lin;
    BatchedLayout lay;
    if (plan_batched(times_host, n, n_lc, lc_chunk, durations_host, n_dur, grid, n_template, n_per, d, &lin, &lay,
                     n_templates) != CETRA_OK)
        return 0;
    return lay.total;
}

int cetra_search_batched_templates(const double *times_host, const void *flux_dev, const void *flux_err_dev,
                                   cetra_dtype dtype, int64_t n, int32_t n_lc, int32_t lc_chunk,
                                   const double *durations_host, int32_t n_dur, cetra_t0_grid grid,
                                   const float *templates_host, int32_t n_template, int32_t n_templates,
                                   const double *periods_host, int32_t n_per, const int32_t *dur_lo_host,
                                   const int32_t *dur_hi_host, cetra_peak *peaks_dev, void *workspace_dev,
                                   size_t workspace_bytes, void *cuda_stream) {
    if (!flux_dev || !flux_err_dev || !templates_host || !periods_host || !peaks_dev || n_templates < 1 ||
        (dtype != CETRA_F32 && dtype != CETRA_F64) || ((dur_lo_host == nullptr) != (dur_hi_host == nullptr)))
        return CETRA_ERR_INVALID_ARG;
    const Device d = device_or_default();   // argument errors are reported even where no device is visible
    int rc;
    LinearPlan lin;
    BatchedLayout lay;
    rc = plan_batched(times_host, n, n_lc, lc_chunk, durations_host, n_dur, grid, n_template, n_per, d, &lin, &lay,
                      n_templates);
    if (rc != CETRA_OK) return rc;
    if (!workspace_dev || !aligned(workspace_dev) || workspace_bytes < lay.total) return CETRA_ERR_WORKSPACE;
    if ((rc = require_device()) != CETRA_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t esz = dtype_size(dtype);
    for (int32_t lc0 = 0; lc0 < n_lc; lc0 += lay.chunk) {
        const int32_t m = std::min(lay.chunk, n_lc - lc0);
        const char *fl = static_cast<const char *>(flux_dev) + static_cast<size_t>(lc0) * n * esz;
        const char *er = static_cast<const char *>(flux_err_dev) + static_cast<size_t>(lc0) * n * esz;
        rc = run_chunk(lin, lay, d, fl, er, dtype, n, m, lc0 == 0, durations_host, n_dur, grid, templates_host,
                       n_template, periods_host, n_per, dur_lo_host, dur_hi_host,
                       peaks_dev + static_cast<size_t>(lc0) * n_per, static_cast<size_t>(n_lc) * n_per,
                       static_cast<char *>(workspace_dev), st);
        if (rc != CETRA_OK) return rc;
    }
    return CETRA_OK;
}

size_t cetra_search_batched_host_workspace_bytes(const double *times_host, int64_t n, int32_t n_lc, int32_t lc_chunk,
                                                 cetra_dtype dtype, const double *durations_host, int32_t n_dur,
                                                 cetra_t0_grid grid, int32_t n_template, int32_t n_per) {
    const Device d = device_or_default();
    LinearPlan lin;
    BatchedLayout lay;
    if (plan_batched(times_host, n, n_lc, lc_chunk, durations_host, n_dur, grid, n_template, n_per, d, &lin, &lay) !=
        CETRA_OK)
        return 0;
    const size_t in_bytes = align_up(static_cast<size_t>(lay.chunk) * n * dtype_size(dtype));
    const size_t out_bytes = align_up(sizeof(cetra_peak) * static_cast<size_t>(lay.chunk) * n_per);
    return lay.total + 2 * in_bytes + out_bytes;
}

int cetra_search_batched_host(const double *times_host, const void *flux_host, const void *flux_err_host,
                              cetra_dtype dtype, int64_t n, int32_t n_lc, int32_t lc_chunk,
                              const double *durations_host, int32_t n_dur, cetra_t0_grid grid,
                              const float *template_host, int32_t n_template, const double *periods_host,
                              int32_t n_per, const int32_t *dur_lo_host, const int32_t *dur_hi_host,
                              cetra_peak *peaks_host, void *workspace_dev, size_t workspace_bytes,
                              void *cuda_stream) {
    if (!flux_host || !flux_err_host || !template_host || !periods_host || !peaks_host ||
        (dtype != CETRA_F32 && dtype != CETRA_F64) || ((dur_lo_host == nullptr) != (dur_hi_host == nullptr)))
        return CETRA_ERR_INVALID_ARG;
    const Device d = device_or_default();   // argument errors are reported even where no device is visible
    int rc;
    LinearPlan lin;
    BatchedLayout lay;
    rc = plan_batched(times_host, n, n_lc, lc_chunk, durations_host, n_dur, grid, n_template, n_per, d, &lin, &lay);
    if (rc != CETRA_OK) return rc;
    const size_t esz = dtype_size(dtype);
    const size_t in_bytes = align_up(static_cast<size_t>(lay.chunk) * n * esz);
    const size_t out_bytes = align_up(sizeof(cetra_peak) * static_cast<size_t>(lay.chunk) * n_per);
    if (!workspace_dev || !aligned(workspace_dev) || workspace_bytes < lay.total + 2 * in_bytes + out_bytes)
        return CETRA_ERR_WORKSPACE;
    if ((rc = require_device()) != CETRA_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    char *ws = static_cast<char *>(workspace_dev);
    char *fl_dev = ws + lay.total;
    char *er_dev = fl_dev + in_bytes;
    cetra_peak *pk_dev = reinterpret_cast<cetra_peak *>(er_dev + in_bytes);
    for (int32_t lc0 = 0; lc0 < n_lc; lc0 += lay.chunk) {
        const int32_t m = std::min(lay.chunk, n_lc - lc0);
        const size_t bytes = static_cast<size_t>(m) * n * esz;
        const char *fl = static_cast<const char *>(flux_host) + static_cast<size_t>(lc0) * n * esz;
        const char *er = static_cast<const char *>(flux_err_host) + static_cast<size_t>(lc0) * n * esz;
        CETRA_CUDA_TRY(cudaMemcpyAsync(fl_dev, fl, bytes, cudaMemcpyHostToDevice, st));
        CETRA_CUDA_TRY(cudaMemcpyAsync(er_dev, er, bytes, cudaMemcpyHostToDevice, st));
        rc = run_chunk(lin, lay, d, fl_dev, er_dev, dtype, n, m, lc0 == 0, durations_host, n_dur, grid,
                       template_host, n_template, periods_host, n_per, dur_lo_host, dur_hi_host, pk_dev, 0, ws, st);
        if (rc != CETRA_OK) return rc;
        CETRA_CUDA_TRY(cudaMemcpyAsync(peaks_host + static_cast<size_t>(lc0) * n_per, pk_dev,
                                       sizeof(cetra_peak) * static_cast<size_t>(m) * n_per, cudaMemcpyDeviceToHost,
                                       st));
    }
    CETRA_CUDA_TRY(cudaStreamSynchronize(st));
    return CETRA_OK;
}

}  // extern "C"

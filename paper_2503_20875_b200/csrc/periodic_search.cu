// Periodic search (§2.3): steps P1-P4 of DESIGN.md.
//
//   P1 epoch offsets        off_e = llrint(e * P_k / stride) in FP64, 32 epochs per warp at a time (R11)
//   P2 fold-gather-sum      SA = sum_e S_wmm[j][p + off_e], SB = sum_e S_wmf[j][p + off_e]
//   P3 combine              Z = SB/SA, var = 1/SA, LR = 1/2 SB^2/SA  (= Eq. 4 summed at Z)
//   P4 argmax               per period: max LR over (duration, phase), ties -> smallest j, then p
//
// The combined (depth, var, LR) arrays of a period are never materialised: a warp folds (period, duration)
// pairs in registers and publishes one packed 64-bit key per period with atomicMax.  The fold kernels live in
// fold_pair.cu (rows resident in shared memory) and fold_stream.cu (rows streamed through shared memory); this
// file holds the plan, the launch order, the conversion of the public grids and the final record kernel.
#include "periodic_search.cuh"
#include "fold_common.cuh"

#include <math.h>

#include <algorithm>
#include <vector>

namespace cetra {

// Plan overrides for the parity tests (cetra_test_fold_override in cetra.h).  Set only through that call: the library
// reads no environment variable, so nothing outside the process's own code can change which kernel a search runs.
static std::atomic<int> g_test_force_stream{0};
static std::atomic<int> g_test_stage_cells{0};

// One thread per (light curve, period): decode the winning (j, p), redo its fold in FP64 with
// IEEE division, count the contributing epochs and write the record.
__global__ void finalize_peaks_kernel(const __grid_constant__ PeriodicParams P, cetra_peak *__restrict__ peaks) {
    const long long total = static_cast<long long>(P.n_lc) * P.n_per;
    for (long long idx = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; idx < total;
         idx += static_cast<long long>(gridDim.x) * blockDim.x) {
        const unsigned long long key = P.keys[idx];
        cetra_peak out;
        const float nanv = __int_as_float(0x7fc00000);
        out.lr = nanv; out.depth = nanv; out.depth_var = nanv; out.t0 = nanv;
        out.i_t0 = -1; out.j_dur = -1; out.n_transits = 0; out.reserved = 0;
        if (key != 0ull) {
            const long long lc = idx / P.n_per;
            const int k = static_cast<int>(idx - lc * P.n_per);
            const unsigned int id = 0xffffffffu - static_cast<unsigned int>(key & 0xffffffffull);
            const int j = static_cast<int>(id / static_cast<unsigned int>(P.n_t0));
            const int p = static_cast<int>(id - static_cast<unsigned int>(j) * static_cast<unsigned int>(P.n_t0));
            const float2 *row = P.stats + (lc * P.n_dur + j) * P.stats_pitch;
            const double r = P.r_cells[k];
            const bool literal = P.literal && *P.literal;
            const float *res = literal ? P.resid + (lc * P.n_dur + j) * P.stats_pitch : nullptr;
            // FP64 sums and combination (north_star: "FP64 final sums if needed"): the record is then the FP32 cells'
            // exact fold rounded once, also where epochs of opposite sign cancel (Z ~ 0 out of large per-transit
            // terms) and a running FP32 sum would lose 1e-5 of the small combined LR.  One thread per record, a few
            // dozen cells each: 0.1 % of a search.
            double sa = 0.0, sb = 0.0, sc = 0.0;
            int ntr = 0;
            for (long long e = 0;; ++e) {
                const long long cell = p + __double2ll_rn(__dmul_rn(static_cast<double>(e), r));
                if (cell > P.n_t0 - 1) break;
                const float2 ab = row[cell];
                sa += static_cast<double>(ab.x);
                sb += static_cast<double>(ab.y);
                if (literal) sc += static_cast<double>(res[cell]);
                ntr += ab.x > 0.f ? 1 : 0;
            }
            const double z = sb / sa;                                // common depth Z
            out.depth = static_cast<float>(z);
            out.depth_var = static_cast<float>(1.0 / sa);
            out.lr = static_cast<float>(0.5 * sb * z + sc);          // Eq. 4 summed at Z (sc = 0 unless literal)
            out.t0 = static_cast<float>(P.t0_start + static_cast<double>(p) * P.t0_stride);
            out.i_t0 = p; out.j_dur = j; out.n_transits = ntr;
        }
        peaks[idx] = out;
    }
}

// (depth, var) grids -> (S_wmm, S_wmf) rows: S_wmm = 1/var, S_wmf = depth/var, null (NaN) cells -> 0.
// With a likelihood-ratio grid: resid = dlogL - 1/2 depth^2/var per cell (what Eq. 4 summed at Z keeps of LR_e beyond
// the two statistics: sum_e [LR_e - 1/2 (D_e - Z)^2 / var_e] = sum_e resid_e + 1/2 (sum B)^2 / sum A), and the flag
// is raised when some cell's resid exceeds the rounding of a linear-search grid (whose dlogL IS 1/2 depth^2/var).
__global__ void grids_to_stats_kernel(const float *__restrict__ depth, const float *__restrict__ var,
                                      const float *__restrict__ dlogL, long long n_rows, long long n_t0,
                                      long long pitch, float2 *__restrict__ stats, float *__restrict__ resid,
                                      int *__restrict__ literal) {
    const long long total = n_rows * pitch;
    bool differs = false;
    for (long long idx = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; idx < total;
         idx += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long rowid = idx / pitch;
        const long long i = idx - rowid * pitch;
        float2 out = make_float2(0.f, 0.f);
        float c = 0.f;
        if (i < n_t0) {
            const float d = depth[rowid * n_t0 + i], v = var[rowid * n_t0 + i];
            if (isfinite(d) && isfinite(v) && v > 0.f) {
                const float a = 1.0f / v;
                const float b = d / v;
                if (isfinite(a) && isfinite(b)) {
                    out = make_float2(a, b);
                    if (dlogL) {
                        const float l = dlogL[rowid * n_t0 + i];
                        const float ident = 0.5f * d * b;
                        c = l - ident;
                        // beyond FP32 rounding of the identity (relative), and large enough to move a log-likelihood
                        // at all (1e-7 absolute: sums of a few dozen epochs stay far below the 5e-6 that parity allows)
                        if (!(fabsf(c) <= 1e-5f * fabsf(ident) + 1e-7f)) differs = true;   // also NaN / inf
                        if (!isfinite(c)) c = 0.f;
                    }
                }
            }
        }
        stats[idx] = out;
        if (resid) resid[idx] = c;
    }
    if (literal && __any_sync(0xffffffffu, differs) && (threadIdx.x & 31) == 0) atomicOr(literal, 1);
}

// Periodic search on a caller's likelihood-ratio grid (literal Eq. 3-4): three sums per (period,
// duration, phase).  One warp per (light curve, period, duration), lanes over phases, rows read through L1/L2: a
// plain kernel for a rare call (the searches the library chains itself run on the two-statistic kernels).
__device__ __forceinline__ unsigned int order_bits(float x) {          // monotone map float -> uint (any sign)
    const unsigned int b = __float_as_uint(x);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

__global__ void __launch_bounds__(256) fold_literal_argmax_kernel(const __grid_constant__ PeriodicParams P) {
    if (!(P.literal && *P.literal)) return;
    const int lane = threadIdx.x & 31;
    const long long warp0 = (blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x) >> 5;
    const long long n_warps = (static_cast<long long>(gridDim.x) * blockDim.x) >> 5;
    const long long units = static_cast<long long>(P.n_lc) * P.n_dur * P.n_per;
    for (long long u = warp0; u < units; u += n_warps) {
        const int k = static_cast<int>(u % P.n_per);
        const long long rowid = u / P.n_per;                             // lc * n_dur + j
        const int j = static_cast<int>(rowid % P.n_dur);
        const long long lc = rowid / P.n_dur;
        if (!(P.durations[j] < P.periods[k])) continue;
        if (P.dur_lo && (j < P.dur_lo[k] || j >= P.dur_hi[k])) continue;
        const double r = P.r_cells[k];
        const double rc = ceil(r);
        const int n_phase = rc < static_cast<double>(P.n_t0) ? static_cast<int>(rc) : P.n_t0;   // R10
        const float2 *row = P.stats + rowid * P.stats_pitch;
        const float *res = P.resid + rowid * P.stats_pitch;
        unsigned long long best = 0ull;
        for (int p = lane; p < n_phase; p += 32) {
            float sa = 0.f, sb = 0.f, sc = 0.f;
            for (long long e = 0;; ++e) {
                const long long cell = p + __double2ll_rn(__dmul_rn(static_cast<double>(e), r));   // R11
                if (cell > P.n_t0 - 1) break;
                const float2 ab = __ldg(row + cell);
                sa += ab.x;
                sb += ab.y;
                sc += __ldg(res + cell);
            }
            if (sa >= 1.17549435e-38f) {
                const float lr = 0.5f * sb * (sb / sa) + sc;
                if (lr == lr) {
                    const unsigned int id = static_cast<unsigned int>(j) * static_cast<unsigned int>(P.n_t0) + p;
                    const unsigned long long key = (static_cast<unsigned long long>(order_bits(lr)) << 32) | (0xffffffffu - id);
                    best = key > best ? key : best;                      // ties: the smaller cell id has the larger key
                }
            }
        }
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) {
            const unsigned long long o = __shfl_xor_sync(0xffffffffu, best, s);
            best = o > best ? o : best;
        }
        if (lane == 0 && best) atomicMax(P.keys + lc * P.n_per + k, best);
    }
}

// ------------------------------------------------------------------------------------------- host
int build_periodic_plan(int32_t n_lc, int32_t n_dur, cetra_t0_grid grid, const double *durations_host,
                        const double *periods_host, int32_t n_per, int smem_limit, int n_sm, PeriodicPlan *pl) {
    if (!durations_host || !periods_host || n_lc < 1 || n_dur < 1 || n_per < 1 || grid.n_t0 < 1 ||
        !(grid.t0_stride > 0.0) || !std::isfinite(grid.t0_stride) || !std::isfinite(grid.t0_start))
        return CETRA_ERR_INVALID_ARG;
    if (n_dur > CETRA_MAX_DURATIONS) return CETRA_ERR_UNSUPPORTED;
    // the packed cell id (j * n_t0 + p) must fit 32 bits, cell indices an int
    if (grid.n_t0 > 0x7fffffffLL - 4096 || static_cast<long long>(n_dur) * grid.n_t0 >= 0xffffffffLL)
        return CETRA_ERR_UNSUPPORTED;
    for (int k = 0; k < n_per; ++k)
        if (!(periods_host[k] >= grid.t0_stride) || !std::isfinite(periods_host[k])) return CETRA_ERR_INVALID_ARG;
    PeriodicParams &P = pl->P;
    for (int j = 0; j < n_dur; ++j) {
        if (!(durations_host[j] > 0.0) || !std::isfinite(durations_host[j])) return CETRA_ERR_INVALID_ARG;
        P.durations[j] = durations_host[j];
    }
    P.n_lc = n_lc; P.n_dur = n_dur; P.n_t0 = static_cast<int>(grid.n_t0); P.n_per = n_per;
    P.t0_start = grid.t0_start; P.t0_stride = grid.t0_stride;
    P.stats_pitch = cetra_stats_pitch(grid.n_t0);
    const size_t row_bytes = static_cast<size_t>(P.stats_pitch) * sizeof(float2);
    const size_t header = kGrpHeaderBytes;
    pl->row_in_smem = row_bytes + header <= static_cast<size_t>(smem_limit);
    // test hook (cetra_test_fold_override): rows that would fit in shared memory go through the streamed kernel, so
    // that small problems (which the oracle folds in full) exercise it too
    if (g_test_force_stream.load(std::memory_order_relaxed)) pl->row_in_smem = false;
    if (pl->row_in_smem) {
        pl->smem_bytes = row_bytes + header;
    } else {
        // streamed kernel: the ring takes all the shared memory of the SM
        pl->stage_cells = static_cast<int>(((static_cast<size_t>(smem_limit) - kStrHeaderBytes) / (8 * kStrStages)) & ~size_t(1));
        {   // test hook (cetra_test_fold_override): small stages (block splitting, direct epochs)
            const int v = g_test_stage_cells.load(std::memory_order_relaxed) & ~1;
            if (v >= 64 && v < pl->stage_cells) pl->stage_cells = v;
        }
        pl->smem_bytes = kStrHeaderBytes + static_cast<size_t>(kStrStages) * pl->stage_cells * 8;
    }
    // work units: consecutive periods of one row, one period (per-period kernel) or kGrpT periods (grouped
    // kernel) per warp; see the kernels
    const long long rows = static_cast<long long>(n_lc) * n_dur;
    const int unit_periods = pl->row_in_smem ? (kGrpThreads / 32) * kGrpT : kStrUnitPeriods;   // two per (consumer) warp
    P.units_per_row = (n_per + unit_periods - 1) / unit_periods;
    P.n_units = rows * P.units_per_row;
    if (P.n_units > 0x7fffffffLL - (1LL << 24)) return CETRA_ERR_UNSUPPORTED;   // 32-bit queue head + overshoot
    P.max_claim = std::max(1, 4 * P.units_per_row);
    const int per_sm = 1;                                     // both fold kernels fill an SM with one CTA
    pl->grid = static_cast<int>(std::min<long long>(P.n_units, static_cast<long long>(n_sm) * per_sm));
    return CETRA_OK;
}

size_t periodic_workspace_bytes(int32_t n_lc, int32_t n_per) {
    size_t b = 0;
    b += 2 * align_up(sizeof(double) * static_cast<size_t>(n_per));                       // periods, periods / stride
    b += 2 * align_up(sizeof(int) * static_cast<size_t>(n_per));                          // dur_lo, dur_hi
    b += align_up(sizeof(unsigned long long) * static_cast<size_t>(n_lc) * n_per + 256);  // keys + counter
    return b;
}

int run_periodic(PeriodicPlan &pl, const float2 *stats_dev, const double *periods_host, const int32_t *dur_lo_host,
                 const int32_t *dur_hi_host, bool upload, cetra_peak *peaks_dev, void *workspace_dev,
                 cudaStream_t st, const float *resid_dev, const int *literal_dev) {
    PeriodicParams &P = pl.P;
    Carver ws(workspace_dev);
    double *periods = ws.take<double>(P.n_per);
    double *r_cells = ws.take<double>(P.n_per);
    int *lo = ws.take<int>(P.n_per);
    int *hi = ws.take<int>(P.n_per);
    const size_t n_keys = static_cast<size_t>(P.n_lc) * P.n_per;
    unsigned long long *keys = ws.take<unsigned long long>(n_keys + 32);
    const bool ranges = dur_lo_host && dur_hi_host;
    if (upload) {
        CETRA_CUDA_TRY(cudaMemcpyAsync(periods, periods_host, sizeof(double) * P.n_per, cudaMemcpyHostToDevice, st));
        // r_k = P_k / stride: the one IEEE FP64 division of R11, hoisted out of the kernels (a tiny staging array;
        // cudaMemcpyAsync from pageable memory copies it before returning)
        std::vector<double> r_host(P.n_per);
        for (int k = 0; k < P.n_per; ++k) r_host[k] = periods_host[k] / P.t0_stride;
        CETRA_CUDA_TRY(cudaMemcpyAsync(r_cells, r_host.data(), sizeof(double) * P.n_per, cudaMemcpyHostToDevice, st));
        if (ranges) {
            CETRA_CUDA_TRY(cudaMemcpyAsync(lo, dur_lo_host, sizeof(int) * P.n_per, cudaMemcpyHostToDevice, st));
            CETRA_CUDA_TRY(cudaMemcpyAsync(hi, dur_hi_host, sizeof(int) * P.n_per, cudaMemcpyHostToDevice, st));
        }
    }
    P.stats = stats_dev;
    P.periods = periods;
    P.r_cells = r_cells;
    P.dur_lo = ranges ? lo : nullptr;
    P.dur_hi = ranges ? hi : nullptr;
    P.keys = keys;
    P.counter = reinterpret_cast<unsigned int *>(keys + n_keys);
    P.resid = resid_dev;
    P.literal = literal_dev;
    CETRA_CUDA_TRY(cudaMemsetAsync(keys, 0, sizeof(unsigned long long) * (n_keys + 32), st));
    profile_mark(kProfFold, true, st);
    {
        const int rc = pl.row_in_smem ? launch_fold_pair(pl, st) : launch_fold_stream(pl, st);
        if (rc != CETRA_OK) return rc;
    }
    profile_mark(kProfFold, false, st);
    CETRA_LAUNCH_CHECK();
    if (resid_dev && literal_dev) {                           // returns at once unless the flag is raised
        fold_literal_argmax_kernel<<<148 * 8, 256, 0, st>>>(P);
        CETRA_LAUNCH_CHECK();
    }
    {
        const long long total = static_cast<long long>(P.n_lc) * P.n_per;
        const int blocks = static_cast<int>(std::min<long long>((total + 255) / 256, 148LL * 8));
        finalize_peaks_kernel<<<blocks, 256, 0, st>>>(P, peaks_dev);
        CETRA_LAUNCH_CHECK();
    }
    return CETRA_OK;
}

int run_grids_to_stats(const float *depth_dev, const float *var_dev, const float *dlogL_dev, int32_t n_rows,
                       int64_t n_t0, float2 *stats_dev, float *resid_dev, int *literal_dev, cudaStream_t st) {
    const long long pitch = cetra_stats_pitch(n_t0);
    const long long total = static_cast<long long>(n_rows) * pitch;
    const int blocks = static_cast<int>(std::min<long long>((total + 255) / 256, 148LL * 16));
    if (literal_dev) CETRA_CUDA_TRY(cudaMemsetAsync(literal_dev, 0, sizeof(int), st));
    grids_to_stats_kernel<<<blocks, 256, 0, st>>>(depth_dev, var_dev, dlogL_dev, n_rows, n_t0, pitch, stats_dev,
                                                  dlogL_dev ? resid_dev : nullptr, dlogL_dev ? literal_dev : nullptr);
    CETRA_LAUNCH_CHECK();
    return CETRA_OK;
}

}  // namespace cetra

extern "C" void cetra_test_fold_override(int32_t force_stream, int32_t stage_cells) {
    cetra::g_test_force_stream.store(force_stream != 0 ? 1 : 0, std::memory_order_relaxed);
    cetra::g_test_stage_cells.store(stage_cells > 0 ? stage_cells : 0, std::memory_order_relaxed);
}

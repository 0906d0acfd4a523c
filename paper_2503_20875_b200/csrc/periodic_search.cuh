// Host-side plan and kernel parameters of the periodic search (§2.3).
#pragma once

#include "common.cuh"

namespace cetra {

// Pair fold (rows resident in shared memory): one warp folds kGrpT neighbouring trial periods together.
constexpr int kGrpT = 2;             // periods per warp
constexpr int kGrpG = 11;            // consecutive phases per lane; odd => conflict-free 8-byte LDS at a stride of G cells
constexpr int kGrpThreads = 640;     // 20 warps x 96 registers
constexpr size_t kGrpHeaderBytes = 16 + (kGrpThreads / 32) * 64 * 8;   // barrier, claim slot, epoch words (2 blocks per warp)
// Streamed fold (rows that do not fit in shared memory): 19 consumer warps + one producer warp, a ring of stages that
// hold the windows of a block of epochs each (640 threads keep the 96-register budget of the two-period register window).
constexpr int kStrThreads = 640;
constexpr int kStrUnitPeriods = (kStrThreads / 32 - 1) * kGrpT;
#ifndef CETRA_STR_STAGES_LOG2
#define CETRA_STR_STAGES_LOG2 2
#endif
constexpr int kStrStagesLog2 = CETRA_STR_STAGES_LOG2;
constexpr int kStrStages = 1 << kStrStagesLog2;
constexpr size_t kStrHeaderBytes = 8192;                                 // barriers, stage descriptors, per-warp epoch words

struct PeriodicParams {
    const float2 *stats;             // [n_lc][n_dur][stats_pitch] (S_wmm, S_wmf), zero in null cells / padding
    const double *periods;           // [n_per] device
    const double *r_cells;           // [n_per] device: periods[k] / t0_stride (IEEE FP64 division, done once on the host)
    const int *dur_lo, *dur_hi;      // [n_per] device or null
    unsigned long long *keys;        // [n_lc][n_per] packed (lr bits << 32 | ~cell id), 0 = no candidate
    unsigned int *counter;           // work-unit queue head
    // cetra_periodic_search with a caller's likelihood-ratio grid (literal Eq. 4): resid = dlogL - 1/2 depth^2/var per
    // cell, and a device flag that is non-zero when some cell's resid matters (then fold_literal_argmax_kernel does
    // the search and the two-statistic kernels return at once).  Both null on the sufficient-statistics path.
    const float *resid;              // [n_lc][n_dur][stats_pitch] or null
    const int *literal;              // device flag or null
    long long stats_pitch;
    double t0_start, t0_stride;
    int n_lc, n_dur, n_t0, n_per;
    int units_per_row, max_claim;    // unit = periods_per_unit consecutive periods of one row
    long long n_units;
    double durations[CETRA_MAX_DURATIONS];
};

struct PeriodicPlan {
    PeriodicParams P{};
    bool row_in_smem = false;        // resident-row kernel (row in shared memory) or streamed kernel (row in L2)
    size_t smem_bytes = 0;
    int grid = 0;
    int stage_cells = 0;             // streamed kernel: cells per ring stage
};

int build_periodic_plan(int32_t n_lc, int32_t n_dur, cetra_t0_grid grid, const double *durations_host,
                        const double *periods_host, int32_t n_per, int smem_limit, int n_sm, PeriodicPlan *pl);
size_t periodic_workspace_bytes(int32_t n_lc, int32_t n_per);   // periods, ranges, keys, counter (not the stats)
// periods / ranges are uploaded when `upload` is set (first chunk of a batched search), else re-used.
int run_periodic(PeriodicPlan &pl, const float2 *stats_dev, const double *periods_host, const int32_t *dur_lo_host,
                 const int32_t *dur_hi_host, bool upload, cetra_peak *peaks_dev, void *workspace_dev,
                 cudaStream_t st, const float *resid_dev = nullptr, const int *literal_dev = nullptr);
int launch_fold_stream(const PeriodicPlan &pl, cudaStream_t st);   // fold_stream.cu
int launch_fold_pair(const PeriodicPlan &pl, cudaStream_t st);     // fold_pair.cu
int run_grids_to_stats(const float *depth_dev, const float *var_dev, const float *dlogL_dev, int32_t n_rows,
                       int64_t n_t0, float2 *stats_dev, float *resid_dev, int *literal_dev, cudaStream_t st);

}  // namespace cetra

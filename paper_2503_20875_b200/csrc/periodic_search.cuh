// Host-side plan and kernel parameters of the periodic search (§2.3).
#pragma once

#include "common.cuh"

namespace cetra {

constexpr int kFoldR = 8;            // phase groups (of 32 phases) per warp pass; needs kStatsPad >= 32*kFoldR
constexpr int kFoldThreads = 512;    // 16 warps x 128 registers: 8 x 4 loads in flight per lane (the kernel is latency-bound)

// Grouped fold (rows resident in shared memory): one warp folds kGrpT neighbouring trial periods together.
constexpr int kGrpT = 2;             // periods per warp
constexpr int kGrpG = 11;            // consecutive phases per lane; odd => conflict-free 8-byte LDS at a stride of G cells
constexpr int kGrpS = 7;             // largest spread of a group's epoch offsets served from one register window
constexpr int kGrpThreads = 640;     // 20 warps x 94 registers (measured best of 448-768 threads, G = 7-15)
constexpr size_t kGrpHeaderBytes = 16 + (kGrpThreads / 32) * 32 * 8;   // barrier, claim slot, epoch words
static_assert(kStatsPad >= 32 * (kGrpG + 2) + kGrpS + 1, "the widest (last) pass may read 32*(G+2)+S cells past the last t0 cell");
static_assert(kStatsPad >= 32 * kFoldR, "a pass may read 32*R cells past the last t0 cell");

struct PeriodicParams {
    const float2 *stats;             // [n_lc][n_dur][stats_pitch] (S_wmm, S_wmf), zero in null cells / padding
    const double *periods;           // [n_per] device
    const int *dur_lo, *dur_hi;      // [n_per] device or null
    unsigned long long *keys;        // [n_lc][n_per] packed (lr bits << 32 | ~cell id), 0 = no candidate
    unsigned int *counter;           // work-unit queue head
    long long stats_pitch;
    double t0_start, t0_stride;
    int n_lc, n_dur, n_t0, n_per;
    int units_per_row, max_claim;    // unit = periods_per_unit consecutive periods of one row
    long long n_units;
    double durations[CETRA_MAX_DURATIONS];
};

struct PeriodicPlan {
    PeriodicParams P{};
    bool row_in_smem = false;        // grouped kernel (row in shared memory) or per-period kernel (row in L2)
    size_t smem_bytes = 0;
    int grid = 0;
};

int build_periodic_plan(int32_t n_lc, int32_t n_dur, cetra_t0_grid grid, const double *durations_host,
                        const double *periods_host, int32_t n_per, int smem_limit, int n_sm, PeriodicPlan *pl);
size_t periodic_workspace_bytes(int32_t n_lc, int32_t n_per);   // periods, ranges, keys, counter (not the stats)
// periods / ranges are uploaded when `upload` is set (first chunk of a batched search), else re-used.
int run_periodic(PeriodicPlan &pl, const float2 *stats_dev, const double *periods_host, const int32_t *dur_lo_host,
                 const int32_t *dur_hi_host, bool upload, cetra_peak *peaks_dev, void *workspace_dev,
                 cudaStream_t st);
int run_grids_to_stats(const float *depth_dev, const float *var_dev, int32_t n_rows, int64_t n_t0,
                       float2 *stats_dev, cudaStream_t st);

}  // namespace cetra

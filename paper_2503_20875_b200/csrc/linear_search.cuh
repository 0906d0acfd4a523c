// Host-side plan and kernel parameters of the linear search (§2.2).
#pragma once

#include <vector>

#include "common.cuh"

namespace cetra {

constexpr int kLinearR = 15;   // consecutive t0 cells per thread; odd => conflict-free 8-byte shared loads

// Passed by value (__grid_constant__): no device copy, no host synchronisation.
struct LinearParams {
    const float2 *wfw;          // [n_lc][q][ph_pitch] (w f, w): element u of stream v is sample n_lo + q u + v
    const float2 *taps;         // per duration [q][A_j] (m, m^2), see build_taps_kernel
    float *depth, *var, *dlogL; // [n_lc][n_dur][n_t0] or null
    float2 *stats;              // [n_lc][n_dur][stats_pitch] or null
    long long lc_pitch, ph_pitch, n_lo, n0, n_t0, stats_pitch;   // lc_pitch = q * ph_pitch elements per light curve
    int q, n_dur, tiles_per_row;
    // Residue classes of a rational off-grid stride (Geometry::rational): cell i = n_cls a + rho of class rho sits
    // q a samples after sample cls_n0[rho] + f_rho, |f_rho| <= 1/2.  n_cls = 1 on the sample grid (n0, no lists).
    int n_cls, n_tpl;
    // Template set (cetra_search_batched_templates): T templates searched in one launch over the
    // same preprocessed samples.  Template t has its own tap tables (tset_taps entries after those of t - 1), its
    // own copy of the template (n_tpl floats after t - 1's) and its own output rows ((t n_lc + lc) n_dur + j).
    int n_tset;
    long long tset_taps;
    const int *cls_n0;          // [n_cls] device
    const int *unsafe_cnt;      // [n_dur][n_cls] device: taps of (j, rho) whose table entry is withheld (see build_class_taps_kernel)
    const int *unsafe_k;        // their sample offsets k, list of (j, rho) at n_cls * tap_off[j] + rho * stored_j
    const float *tpl;           // [n_tpl] device: the template, for the exact evaluations
    unsigned long long *exact_evals;   // device counter of exact (R25) evaluations, diagnostics
    long long n;                // samples per light curve
    double cadence, delta, stride;     // R25 arithmetic: c, t0_start - times[0], t0 stride (days)
    int H[CETRA_MAX_DURATIONS];         // window half-reach in samples (superset of the window)
    int A[CETRA_MAX_DURATIONS];         // taps per polyphase branch, padded to a multiple of kLinearR
    int tap_off[CETRA_MAX_DURATIONS + 1];
    unsigned char order[CETRA_MAX_DURATIONS];
    double durations[CETRA_MAX_DURATIONS];
};

// Off-grid t0 grids (R25): the nearest-neighbour position comes from the time difference, per (cell, sample).
struct GeneralParams {
    const float2 *wfw;          // [n_lc][lc_pitch] (w f, w), element 0 is sample 0
    const float *tpl;           // [n_tpl] device
    float *depth, *var, *dlogL; // [n_lc][n_dur][n_t0] or null
    float2 *stats;              // [n_lc][n_dur][stats_pitch] or null
    long long lc_pitch, n, n_t0, stats_pitch;
    int n_dur, n_tpl;
    long long row0;                    // output row of (light curve 0, duration 0): template t of a set starts at t n_lc n_dur
    double cadence, delta, stride;
    unsigned long long *exact_evals;   // device counter of exact (R25) evaluations, diagnostics
    double eps_scale, eps_abs;         // a position closer than eps_scale / D + eps_abs to a decision point is evaluated exactly
    double durations[CETRA_MAX_DURATIONS];
};

struct LinearPlan {
    Geometry geo;
    std::vector<int> cls_n0;        // rational strides: per class, the sample nearest to its cell 0 ...
    std::vector<double> cls_f;      // ... and the cell's offset from that sample, in samples
    double eps_scale = 0.0, eps_abs = 0.0;
    LinearParams P{};
    GeneralParams G{};          // used instead of P when !geo.on_grid
    int warps = 0, tile = 0;
    long long taps_total = 0;
    size_t smem_bytes = 0;
    bool taps_ready = false;    // tap tables already built in this workspace (batched path re-uses them)
    int n_templates = 1;        // templates searched per launch (cetra_search_batched_templates)
};

int build_linear_plan(const double *times_host, int64_t n, int32_t n_lc, const double *durations_host,
                      int32_t n_dur, cetra_t0_grid grid, int32_t n_template, int smem_limit, int n_sm,
                      LinearPlan *pl, int32_t n_templates = 1);
int exact_eval_count(int64_t *count, bool reset);
size_t linear_workspace_bytes(const LinearPlan &pl, int32_t n_lc, int32_t n_template);
int run_linear(LinearPlan &pl, const void *flux_dev, const void *flux_err_dev, cetra_dtype dtype, int64_t n,
               int32_t n_lc, const float *template_host, int32_t n_template, bool template_on_device,
               float *depth_dev, float *var_dev, float *dlogL_dev, float *stats_dev, void *workspace_dev,
               cudaStream_t st);

}  // namespace cetra

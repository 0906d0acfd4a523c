/*
 * CETRA oracle, setup and follow-up steps -- TEST INFRASTRUCTURE ONLY (see cetra_oracle.c).
 *
 * Plain FP64 restatements of the steps around the two searches (citations are
 * /root/reference/PAPER.md line numbers):
 *
 *   oracle_resample_template  supplied transit model -> M-sample template by linear interpolation
 *   oracle_median_cadence   default resample cadence = median cadence of the input
 *   oracle_resample         irregular light curve -> regular grid: every observation goes to the
 *                           nearest output point; several observations in one point are combined
 *                           with an inverse-variance weighted mean, errors propagated formally;
 *                           points without data are null (NaN flux, infinite error)
 *   oracle_monotransit      single-transit search in the linear-search output:
 *                           per reference time the maximum-likelihood duration, then the n_peaks
 *                           highest, mutually non-overlapping events
 *   oracle_mask_transits    "nullified the flux within and around the highest likelihood transit
 *                           signal" before a repeated search
 *
 * Readings taken where the paper is silent:
 *  R21 "nearest output point": cell = floor((t - t_start)/c + 1/2) (half-way cases go up, as in R3).
 *      Null observations (R8) and observations outside the output grid are dropped.
 *  R22 median cadence = median of the differences of the time-sorted finite timestamps; an even
 *      count takes the mean of the two middle differences.
 *  R23 monotransit events: profile(i) = max_j dlogL[j][i] (ties: smallest j).  Events are taken
 *      greedily by decreasing profile (ties: smallest i); an event at (i, j) removes every
 *      reference time with |t - t_i| <= excl * D_j from further consideration.
 *  R24 masking: a sample at time t is nullified (flux = NaN) when its distance to the nearest
 *      transit mid-time t0 + e*P (e any integer; P <= 0: the single event at t0) is
 *      <= width * D / 2; width = 1 is "within", width > 1 adds the "around".
 *
 * Pins (tests/test_oracle_setup_pins.py): identity on an already regular grid, the two-point
 * weighted mean, numpy.bincount / numpy.average brute force, permutation invariance, cell-boundary
 * placement, numpy.median of numpy.diff; brute-force greedy peak picking in numpy; masked sample
 * sets against a direct modulo computation and the closed-form count.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK 0
#define ORACLE_ERR_ARG -1

static int cmp_double(const void *a, const void *b) {
    const double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

/* "resampled to a user-defined number of samples using simple linear interpolation".
 * Output sample m sits at fraction m/(n_out-1) of the model's span (first to last contact, both kept). */
int oracle_resample_template(const double *model, int32_t n_in, double *out, int32_t n_out) {
    if (n_in < 2 || n_out < 2) return ORACLE_ERR_ARG;
    for (int32_t m = 0; m < n_out; ++m) {
        const double pos = (double)m / (double)(n_out - 1) * (double)(n_in - 1);    /* in model samples */
        int32_t lo = (int32_t)floor(pos);
        if (lo >= n_in - 1) lo = n_in - 2;
        const double w = pos - (double)lo;
        out[m] = (1.0 - w) * model[lo] + w * model[lo + 1];
    }
    return ORACLE_OK;
}

/* R22 */
int oracle_median_cadence(const double *times, int64_t n, double *cadence) {
    if (n < 2) return ORACLE_ERR_ARG;
    double *t = (double *)malloc(sizeof(double) * (size_t)n);
    if (!t) return ORACLE_ERR_ARG;
    int64_t m = 0;
    for (int64_t i = 0; i < n; ++i) if (isfinite(times[i])) t[m++] = times[i];
    if (m < 2) { free(t); return ORACLE_ERR_ARG; }
    qsort(t, (size_t)m, sizeof(double), cmp_double);
    for (int64_t i = 0; i + 1 < m; ++i) t[i] = t[i + 1] - t[i];
    qsort(t, (size_t)(m - 1), sizeof(double), cmp_double);
    const int64_t d = m - 1;
    *cadence = (d % 2) ? t[d / 2] : 0.5 * (t[d / 2 - 1] + t[d / 2]);
    free(t);
    return ORACLE_OK;
}

/* PAPER.md:53-55, R21.  out_flux / out_err are [n_out]. */
int oracle_resample(const double *times, const double *flux, const double *flux_err, int64_t n_in,
                    double t_start, double cadence, int64_t n_out, double *out_flux, double *out_err) {
    if (n_in < 0 || n_out < 1 || !(cadence > 0.0) || !isfinite(t_start)) return ORACLE_ERR_ARG;
    double *sw = (double *)calloc((size_t)n_out, sizeof(double));
    double *swf = (double *)calloc((size_t)n_out, sizeof(double));
    if (!sw || !swf) { free(sw); free(swf); return ORACLE_ERR_ARG; }
    for (int64_t i = 0; i < n_in; ++i) {
        if (!(isfinite(times[i]) && isfinite(flux[i]) && isfinite(flux_err[i]) && flux_err[i] > 0.0)) continue;
        const double cell = floor((times[i] - t_start) / cadence + 0.5);     /* nearest output point */
        if (!(cell >= 0.0 && cell < (double)n_out)) continue;
        const double w = 1.0 / (flux_err[i] * flux_err[i]);
        sw[(int64_t)cell] += w;
        swf[(int64_t)cell] += w * flux[i];
    }
    for (int64_t c = 0; c < n_out; ++c) {
        if (sw[c] > 0.0) {
            out_flux[c] = swf[c] / sw[c];             /* inverse-variance weighted mean */
            out_err[c] = sqrt(1.0 / sw[c]);           /* formal error of that mean */
        } else {
            out_flux[c] = NAN;                        /* null point */
            out_err[c] = INFINITY;
        }
    }
    free(sw); free(swf);
    return ORACLE_OK;
}

/*
 * R23.  Grids are [n_dur][n_t0]; null cells are NaN.  Outputs: n_found events (<= n_peaks), for each the
 * reference-time cell, duration index, dlogL, depth, depth variance.  Also the profile itself
 * (prof_lr[n_t0], prof_j[n_t0]; NaN / -1 where every duration is null) when the pointers are non-null.
 */
int oracle_monotransit(const double *depth, const double *var, const double *dlogL, int32_t n_dur,
                       int64_t n_t0, double t0_stride, const double *durations, int32_t n_peaks, double excl,
                       double *prof_lr, int32_t *prof_j,
                       int64_t *ev_i, int32_t *ev_j, double *ev_lr, double *ev_depth, double *ev_var,
                       int32_t *n_found) {
    if (n_dur < 1 || n_t0 < 1 || n_peaks < 0 || !(t0_stride > 0.0) || !(excl >= 0.0)) return ORACLE_ERR_ARG;
    double *pl = (double *)malloc(sizeof(double) * (size_t)n_t0);
    int32_t *pj = (int32_t *)malloc(sizeof(int32_t) * (size_t)n_t0);
    char *dead = (char *)calloc((size_t)n_t0, 1);
    if (!pl || !pj || !dead) { free(pl); free(pj); free(dead); return ORACLE_ERR_ARG; }
    for (int64_t i = 0; i < n_t0; ++i) {
        double best = -INFINITY; int32_t bj = -1;
        for (int32_t j = 0; j < n_dur; ++j) {
            const double v = dlogL[(int64_t)j * n_t0 + i];
            if (isnan(v)) continue;
            if (v > best) { best = v; bj = j; }
        }
        pl[i] = bj < 0 ? NAN : best;
        pj[i] = bj;
        if (prof_lr) prof_lr[i] = pl[i];
        if (prof_j) prof_j[i] = bj;
    }
    int32_t found = 0;
    while (found < n_peaks) {
        double best = -INFINITY; int64_t bi = -1;
        for (int64_t i = 0; i < n_t0; ++i) {
            if (dead[i] || pj[i] < 0) continue;
            if (pl[i] > best) { best = pl[i]; bi = i; }
        }
        if (bi < 0) break;
        const int32_t j = pj[bi];
        ev_i[found] = bi; ev_j[found] = j; ev_lr[found] = best;
        ev_depth[found] = depth[(int64_t)j * n_t0 + bi];
        ev_var[found] = var[(int64_t)j * n_t0 + bi];
        ++found;
        const double reach = excl * durations[j];
        for (int64_t i = 0; i < n_t0; ++i)
            if (fabs((double)(i - bi) * t0_stride) <= reach) dead[i] = 1;
        dead[bi] = 1;
    }
    *n_found = found;
    free(pl); free(pj); free(dead);
    return ORACLE_OK;
}

/* R24.  flux is modified in place; returns the number of samples nullified through *n_masked. */
int oracle_mask_transits(const double *times, double *flux, int64_t n, double period, double t0, double duration,
                         double width, int64_t *n_masked) {
    if (n < 0 || !(duration > 0.0) || !(width >= 0.0) || !isfinite(t0)) return ORACLE_ERR_ARG;
    const double half = 0.5 * width * duration;
    int64_t cnt = 0;
    for (int64_t i = 0; i < n; ++i) {
        double d = times[i] - t0;
        if (period > 0.0) d -= period * floor(d / period + 0.5);     /* distance to the nearest mid-time */
        if (fabs(d) <= half) { flux[i] = NAN; ++cnt; }
    }
    if (n_masked) *n_masked = cnt;
    return ORACLE_OK;
}

/*
 * CETRA oracle -- TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, FP64 CPU restatement of what the CETRA hot path computes
 * (arXiv 2503.20875; citations are /root/reference/PAPER.md line numbers).
 * It exists to check the CUDA library; it shares no code, header, table or
 * constant with paper_2503_20875_b200/csrc and must never be imported,
 * linked or executed by the product path.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * There is no blocking, fusion or re-ordering here beyond what the paper's
 * definitions state: the linear search is the two traversals of PAPER.md:91
 * (pass 1 = inverse-variance weighted mean depth; pass 2 =
 * literal Eq. 2), the periodic search is literal Eq. 3-4
 * with nearest-neighbour lookup on the t0 grid
 * and a max-reduction per period.  OpenMP only spreads the
 * independent outer loop (cells / periods) over cores.
 *
 * Pins (tests/test_oracle_pins.py): analytic WLS + numpy lstsq (P1), closed form
 * 1/2 S_mf^2/S_mm (P2), brute-force BLS with a box template (P3), joint multi-
 * transit fit (P4), noiseless injection recovery (P5), the paper's worked example
 * PAPER.md:121,167 (P6), scale/shift/null invariances (P7), null semantics (P9); and, for the branches a
 * GPU-vs-oracle comparison cannot see because both sides take the same reading: null epochs are skipped, not
 * the end of the fold (hand-built grid + joint fit across a data gap), ceil(P/s) phases (R10), samples exactly
 * on the first / last instant of a window belong to it (R2), the on-grid decision bounds the drift at the last
 * t0 cell (R25; tests/test_oracle_general_pins.py).
 * Exact agreement with the authors' code and with Table 2 is "parity unpinned"
 * (their code and the TESS data are not in the container).
 *
 * Readings of the paper taken here:
 *  R1  the light curve is already on a regular grid; gaps are null points.
 *  R3  nearest-neighbour template index: x = (k*c)/D + 1/2 for integer sample offset k from
 *      the window centre, idx = floor(x*(M-1) + 1/2); tpl[0] at first contact, tpl[M-1] at last.
 *  R4  t_i is the mid-point of the window.
 *  R5  Delta_n = f_n/m_n is used only through sum(w m f)/sum(w m^2).
 *  R7  f = 1 - flux (dips positive), no sign constraint on the depth.
 *  R8  null input = non-finite flux or non-finite / non-positive error; null output = NaN.
 *  R10 phases p in [0, ceil(P/s)); R11 epoch cell = p + llrint(e * (P/s)) in FP64.
 *  R12 only durations D_j < P_k, optionally a caller range [dur_lo, dur_hi).
 *  R13 ties: smallest j, then smallest p.
 *  R25 t0 grids that do not sit on the sample grid (the paper's default stride is 1 % of the shortest
 *      duration): the nearest-neighbour position is taken from the time difference,
 *      x = (n*c - (t0_start - times[0] + i*s))/D + 1/2 in FP64, every operation rounded once; grids on
 *      the sample grid (every cell within 1e-6 samples of a sample: |a - round a| + |b - round b| (I-1) <= 1e-6
 *      with a = (t0_start - times[0])/c, b = s/c) keep the integer-offset form of R3.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_ERR_ARG -1
#define ORACLE_ERR_GRID -2

static int g_threads = 0;

static int g_force_general = 0;

void oracle_set_threads(int n) { g_threads = n; }

/* Tests only: evaluate grids that sit on the sample grid through the general (R25) form as well. */
void oracle_force_general(int on) { g_force_general = on; }

int oracle_get_threads(void) {
#ifdef _OPENMP
    return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
    return 1;
#endif
}

static int is_null_point(double flux, double err) {
    return !(isfinite(flux) && isfinite(err) && err > 0.0);
}

/* Regular-grid description shared by both entry points (R1, R9). */
static int derive_grid(const double *times, int64_t n, double t0_start, double t0_stride, int64_t n_t0,
                       double *cadence, int64_t *n0, int64_t *q) {
    if (n < 2 || !(t0_stride > 0.0)) return ORACLE_ERR_ARG;
    double c = (times[n - 1] - times[0]) / (double)(n - 1);
    if (!(c > 0.0)) return ORACLE_ERR_ARG;
    for (int64_t i = 0; i < n; ++i)
        if (fabs(times[i] - times[0] - (double)i * c) > 1e-3 * c) return ORACLE_ERR_GRID;
    double a = (t0_start - times[0]) / c;
    double b = t0_stride / c;
    int64_t ia = llrint(a), ib = llrint(b);
    /* on the sample grid iff NO cell of the t0 grid is further than 1e-6 samples from a sample: the stride's
     * mismatch accumulates over the grid, so it is bounded at the last cell (R25) */
    if (fabs(a - (double)ia) + fabs(b - (double)ib) * (double)(n_t0 > 1 ? n_t0 - 1 : 0) > 1e-6 || ib < 1)
        return ORACLE_ERR_GRID;
    *cadence = c; *n0 = ia; *q = ib;
    return ORACLE_OK;
}

/*
 * Linear search, §2.2 (lines 89-125).  Outputs are [n_dur][n_t0], t0 contiguous.
 */
int oracle_linear_search(const double *times, const double *flux, const double *flux_err, int64_t n,
                         const double *durations, int32_t n_dur,
                         double t0_start, double t0_stride, int64_t n_t0,
                         const double *tpl, int32_t n_tpl,
                         double *depth, double *depth_var, double *dlogL) {
    double c; int64_t n0 = 0, q = 0;
    int rc = derive_grid(times, n, t0_start, t0_stride, n_t0, &c, &n0, &q);
    int general = g_force_general;
    if (rc == ORACLE_ERR_GRID) {
        /* regular samples but a t0 grid off the sample grid (R25)?  derive_grid checks the samples first */
        if (n < 2 || !(t0_stride > 0.0)) return ORACLE_ERR_ARG;
        c = (times[n - 1] - times[0]) / (double)(n - 1);
        for (int64_t i = 0; i < n; ++i)
            if (fabs(times[i] - times[0] - (double)i * c) > 1e-3 * c) return ORACLE_ERR_GRID;
        general = 1;
    } else if (rc) {
        return rc;
    }
    if (n_dur < 1 || n_t0 < 1 || n_tpl < 2) return ORACLE_ERR_ARG;
    for (int32_t j = 0; j < n_dur; ++j) if (!(durations[j] > 0.0)) return ORACLE_ERR_ARG;

    /* normalised flux offset from baseline, dips positive; w = 1/sigma^2. */
    double *f = (double *)malloc(sizeof(double) * (size_t)n);
    double *w = (double *)malloc(sizeof(double) * (size_t)n);
    if (!f || !w) { free(f); free(w); return ORACLE_ERR_ARG; }
    for (int64_t i = 0; i < n; ++i) {
        if (is_null_point(flux[i], flux_err[i])) { f[i] = 0.0; w[i] = 0.0; }
        else { f[i] = 1.0 - flux[i]; w[i] = 1.0 / (flux_err[i] * flux_err[i]); }
    }
    const double Mm1 = (double)(n_tpl - 1);
    const int64_t cells = (int64_t)n_dur * n_t0;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 256) num_threads(oracle_get_threads())
#endif
    for (int64_t cell = 0; cell < cells; ++cell) {
        const int32_t j = (int32_t)(cell / n_t0);
        const int64_t i = cell % n_t0;
        const double D = durations[j];
        const int64_t o = (int64_t)j * n_t0 + i;
        double s_mf = 0.0, s_mm = 0.0, delta = 0.0, ll_model = 0.0, ll_flat = 0.0;
        if (!general) {
        const int64_t centre = n0 + i * q;                  /* sample index of t_i */
        const int64_t reach = (int64_t)floor(D / (2.0 * c)) + 1;
        /* pass 1: maximum-likelihood depth and its variance */
        for (int64_t k = -reach; k <= reach; ++k) {
            const int64_t nn = centre + k;
            if (nn < 0 || nn >= n) continue;
            const double x = ((double)k * c) / D + 0.5;     /* R3, R4 */
            if (!(x >= 0.0 && x <= 1.0)) continue;
            const double m = tpl[(int64_t)floor(x * Mm1 + 0.5)];   /* nearest neighbour */
            s_mf += w[nn] * m * f[nn];
            s_mm += w[nn] * m * m;
        }
        if (!(s_mm > 0.0)) {                                /* no observation in the window: null */
            depth[o] = NAN; depth_var[o] = NAN; dlogL[o] = NAN;
            continue;
        }
        delta = s_mf / s_mm;
        /* pass 2: literal Eq. 2 */
        for (int64_t k = -reach; k <= reach; ++k) {
            const int64_t nn = centre + k;
            if (nn < 0 || nn >= n) continue;
            const double x = ((double)k * c) / D + 0.5;
            if (!(x >= 0.0 && x <= 1.0)) continue;
            const double m = tpl[(int64_t)floor(x * Mm1 + 0.5)];
            const double r = delta * m - f[nn];
            ll_model += -0.5 * r * r * w[nn];
            ll_flat += -0.5 * f[nn] * f[nn] * w[nn];
        }
        } else {
        /* R25: the reference time relative to the first sample, and a superset of the window's samples */
        const double ti = (t0_start - times[0]) + (double)i * t0_stride;
        int64_t lo = (int64_t)floor((ti - 0.5 * D) / c) - 1, hi = (int64_t)floor((ti + 0.5 * D) / c) + 2;
        if (lo < 0) lo = 0;
        if (hi > n - 1) hi = n - 1;
        for (int64_t nn = lo; nn <= hi; ++nn) {
            const double x = ((double)nn * c - ti) / D + 0.5;
            if (!(x >= 0.0 && x <= 1.0)) continue;
            const double m = tpl[(int64_t)floor(x * Mm1 + 0.5)];
            s_mf += w[nn] * m * f[nn];
            s_mm += w[nn] * m * m;
        }
        if (!(s_mm > 0.0)) {
            depth[o] = NAN; depth_var[o] = NAN; dlogL[o] = NAN;
            continue;
        }
        delta = s_mf / s_mm;
        for (int64_t nn = lo; nn <= hi; ++nn) {
            const double x = ((double)nn * c - ti) / D + 0.5;
            if (!(x >= 0.0 && x <= 1.0)) continue;
            const double m = tpl[(int64_t)floor(x * Mm1 + 0.5)];
            const double r = delta * m - f[nn];
            ll_model += -0.5 * r * r * w[nn];
            ll_flat += -0.5 * f[nn] * f[nn] * w[nn];
        }
        }
        depth[o] = delta;
        depth_var[o] = 1.0 / s_mm;
        dlogL[o] = ll_model - ll_flat;
    }
    free(f); free(w);
    return ORACLE_OK;
}

/*
 * One (period, duration, phase) cell of the periodic search: literal Eq. 3-4.
 * Returns the number of contributing (non-null) epochs; lr/z/z_var are set only if that is > 0.
 */
static int32_t fold_cell(const double *depth, const double *var, const double *dlogL, int64_t n_t0,
                         int32_t j, int64_t p, double r, double *lr, double *z, double *z_var) {
    const double *dj = depth + (int64_t)j * n_t0;
    const double *vj = var + (int64_t)j * n_t0;
    const double *lj = dlogL + (int64_t)j * n_t0;
    double sw = 0.0, swd = 0.0;
    int32_t ntr = 0;
    for (int64_t e = 0;; ++e) {
        const int64_t cell = p + llrint((double)e * r);     /* R11: nearest neighbour on the t0 grid */
        if (cell > n_t0 - 1) break;
        if (isnan(dj[cell]) || isnan(vj[cell])) continue;   /* null cell: no observation in that window */
        sw += 1.0 / vj[cell];
        swd += dj[cell] / vj[cell];
        ++ntr;
    }
    if (ntr == 0 || !(sw > 0.0)) return 0;
    const double zz = swd / sw;                              /* common depth: inverse-variance weighted mean */
    double acc = 0.0;
    for (int64_t e = 0;; ++e) {
        const int64_t cell = p + llrint((double)e * r);
        if (cell > n_t0 - 1) break;
        if (isnan(dj[cell]) || isnan(vj[cell])) continue;
        const double d = dj[cell] - zz;
        acc += lj[cell] - 0.5 * d * d / vj[cell];            /* Eq. 4 at Z, summed */
    }
    *lr = acc; *z = zz; *z_var = 1.0 / sw;
    return ntr;
}

int oracle_periodic_cell(const double *depth, const double *var, const double *dlogL, int32_t n_dur,
                         int64_t n_t0, double t0_stride, double period, int32_t j, int64_t p,
                         double *lr, double *z, double *z_var, int32_t *n_transits) {
    if (j < 0 || j >= n_dur || p < 0 || p >= n_t0 || !(t0_stride > 0.0) || !(period >= t0_stride))
        return ORACLE_ERR_ARG;
    const double r = period / t0_stride;
    double a = NAN, b = NAN, c = NAN;
    int32_t ntr = fold_cell(depth, var, dlogL, n_t0, j, p, r, &a, &b, &c);
    *lr = a; *z = b; *z_var = c; *n_transits = ntr;
    return ORACLE_OK;
}

/*
 * Periodic search, §2.3 (lines 127-157).  One record per period.
 * dur_lo/dur_hi (optional, may be NULL): per-period half-open duration index range.
 */
int oracle_periodic_search(const double *depth, const double *var, const double *dlogL, int32_t n_dur,
                           int64_t n_t0, double t0_start, double t0_stride, const double *durations,
                           const double *periods, int32_t n_per,
                           const int32_t *dur_lo, const int32_t *dur_hi,
                           double *out_lr, double *out_t0, int64_t *out_i_t0, int32_t *out_j,
                           double *out_z, double *out_z_var, int32_t *out_ntr) {
    if (n_dur < 1 || n_t0 < 1 || n_per < 0 || !(t0_stride > 0.0)) return ORACLE_ERR_ARG;
    for (int32_t k = 0; k < n_per; ++k) if (!(periods[k] >= t0_stride)) return ORACLE_ERR_ARG;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(oracle_get_threads())
#endif
    for (int32_t k = 0; k < n_per; ++k) {
        const double P = periods[k];
        const double r = P / t0_stride;                      /* period in t0-grid cells, FP64 (R11) */
        int64_t n_phase = (int64_t)ceil(r);                  /* R10 */
        if (n_phase > n_t0) n_phase = n_t0;
        int32_t jlo = dur_lo ? dur_lo[k] : 0, jhi = dur_hi ? dur_hi[k] : n_dur;
        if (jlo < 0) jlo = 0;
        if (jhi > n_dur) jhi = n_dur;
        double best = -INFINITY, bz = NAN, bzv = NAN;
        int64_t bp = -1; int32_t bj = -1, bn = 0;
        for (int32_t j = jlo; j < jhi; ++j) {
            if (!(durations[j] < P)) continue;
            for (int64_t p = 0; p < n_phase; ++p) {
                double lr, z, zv;
                const int32_t ntr = fold_cell(depth, var, dlogL, n_t0, j, p, r, &lr, &z, &zv);
                if (ntr == 0) continue;
                if (lr > best) { best = lr; bz = z; bzv = zv; bp = p; bj = j; bn = ntr; }   /* R13 */
            }
        }
        if (bj < 0) {
            out_lr[k] = NAN; out_t0[k] = NAN; out_i_t0[k] = -1; out_j[k] = -1;
            out_z[k] = NAN; out_z_var[k] = NAN; out_ntr[k] = 0;
        } else {
            out_lr[k] = best; out_t0[k] = t0_start + (double)bp * t0_stride; out_i_t0[k] = bp; out_j[k] = bj;
            out_z[k] = bz; out_z_var[k] = bzv; out_ntr[k] = bn;
        }
    }
    return ORACLE_OK;
}

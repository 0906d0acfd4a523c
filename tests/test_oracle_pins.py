"""Pins for the FP64 oracle: what the paper and the mathematics fix (no GPU, no product code).

Each test compares oracle output with something that is NOT the oracle's own formula:
a library least-squares solve, brute force from the definitions on the raw data, a closed
form, an invariance, or the worked example the paper prints.  Templates used where the
expected value must be built by hand are piecewise-constant or linear in x, so the value a
sample must take follows from the window definition and not from
retyping the oracle's nearest-neighbour index expression.
"""
import os

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _lc(n, cadence, sigma, seed, signal=None):
    rng = np.random.default_rng(seed)
    t = np.arange(n) * cadence
    flux = 1.0 + rng.standard_normal(n) * sigma
    err = sigma * (0.5 + rng.random(n))          # heteroscedastic on purpose
    flux = 1.0 + (flux - 1.0) * err / sigma
    if signal is not None:
        flux = flux - signal(t)
    return t, flux, err


def _staircase(M=1024):
    """tpl(x) = 0.5 on the outer quarters, 1 on the middle half (asymmetric tail: 0.25 on the last 10%)."""
    x = np.arange(M) / (M - 1)
    tpl = np.where((x >= 0.25) & (x <= 0.75), 1.0, 0.5)
    tpl = np.where(x > 0.9, 0.25, tpl)
    return tpl


def _staircase_fn(x):
    v = np.where((x >= 0.25) & (x <= 0.75), 1.0, 0.5)
    v = np.where(x > 0.9, 0.25, v)
    return np.where((x < 0) | (x > 1), 0.0, v)


# --------------------------------------------------------------------------- P1
def test_depth_is_weighted_least_squares_solution_lstsq(oracle_mod):
    """P1: depth/var of a window = library WLS solve of f ~ Delta*m."""
    n, c = 400, 0.01
    t, flux, err = _lc(n, c, 1e-3, 11)
    # offsets chosen so that no sample sits within 1e-3 of a staircase edge
    durations = np.array([0.1234, 0.3071])
    tpl = _staircase()
    g = oracle_mod.linear_search(t, flux, err, durations, t[0], c, n, tpl)
    f, w = 1.0 - flux, 1.0 / err ** 2
    for j, D in enumerate(durations):
        for i in (37, 200, 391):
            x = (t - t[i]) / D + 0.5
            m = _staircase_fn(x)
            assert np.min(np.abs(np.concatenate([x - 0.25, x - 0.75, x - 0.9, x, x - 1]))) > 2e-3
            sol, *_ = np.linalg.lstsq((np.sqrt(w) * m)[:, None], np.sqrt(w) * f, rcond=None)
            assert g.depth[j, i] == pytest.approx(sol[0], rel=1e-11, abs=1e-15)
            assert g.depth_var[j, i] == pytest.approx(1.0 / np.sum(w * m * m), rel=1e-12)
            # Eq. 2 by its definition on the whole light curve: lnL(model) - lnL(flat)
            ll = np.sum(-0.5 * w * (sol[0] * m - f) ** 2) - np.sum(-0.5 * w * f ** 2)
            assert g.dlogL[j, i] == pytest.approx(ll, rel=1e-9)


def test_template_orientation_and_window_placement(oracle_mod):
    """A linear ramp template: m_n must equal x_n = (t_n - t_i)/D + 1/2 within the NN step.

    Catches a reversed template, a start-anchored window (R4) and off-by-one window edges.
    """
    n, c, M = 300, 0.02, 1024
    t, flux, err = _lc(n, c, 1e-3, 5)
    tpl = np.arange(M) / (M - 1.0)
    durations = np.array([0.31, 0.77])
    g = oracle_mod.linear_search(t, flux, err, durations, t[0], c, n, tpl)
    f, w = 1.0 - flux, 1.0 / err ** 2
    for j, D in enumerate(durations):
        for i in (50, 151, 250):
            x = (t - t[i]) / D + 0.5
            m = np.where((x >= 0) & (x <= 1), x, 0.0)
            d_exact = np.sum(w * m * f) / np.sum(w * m * m)
            v_exact = 1.0 / np.sum(w * m * m)
            # NN sampling error of a unit-slope ramp is at most 0.5/(M-1) per sample
            assert g.depth_var[j, i] == pytest.approx(v_exact, rel=4.0 / (M - 1))
            assert abs(g.depth[j, i] - d_exact) < 6.0 / (M - 1) * (abs(d_exact) + np.sqrt(v_exact))
    # reversed ramp must give a different answer (the pin has teeth)
    g_rev = oracle_mod.linear_search(t, flux, err, durations, t[0], c, n, tpl[::-1].copy())
    assert not np.allclose(g_rev.depth[0, 50:250], g.depth[0, 50:250], rtol=1e-3)


# --------------------------------------------------------------------------- P2
def test_two_pass_eq2_equals_closed_form(oracle_mod):
    """P2: literal Eq. 2 = 1/2 S_mf^2/S_mm = 1/2 Delta^2/var, and is >= 0."""
    from cetra_synth import make_config
    p = make_config(1)
    g = oracle_mod.linear_search(p.times, p.flux, p.flux_err, p.durations, p.t0_start, p.t0_stride,
                                 p.n_t0, p.template)
    ok = ~np.isnan(g.depth)
    closed = 0.5 * g.depth[ok] ** 2 / g.depth_var[ok]
    assert np.allclose(g.dlogL[ok], closed, rtol=1e-9, atol=1e-12)
    assert np.all(g.dlogL[ok] >= -1e-12)


# --------------------------------------------------------------------------- P3
def test_box_template_reproduces_brute_force_bls(oracle_mod):
    """P3: with tpl == 1 the periodic search is BLS (Kovacs et al. 2002, cited PAPER.md:29):
    SR^2 = s^2/(r(1-r)) = 2 LR / (W (1-r)) for weighted-mean-subtracted data; brute force on N=200."""
    n, c = 200, 0.02
    rng = np.random.default_rng(3)
    t = np.arange(n) * c
    err = 1e-3 * (0.6 + rng.random(n))
    flux = 1.0 + rng.standard_normal(n) * err
    in_tr = (np.abs(((t - 0.33 + 0.4) % 0.8) - 0.4) < 0.05)
    flux[in_tr] -= 3e-3
    w = 1.0 / err ** 2
    W = w.sum()
    mean = np.sum(w * flux) / W
    fluxc = flux - mean + 1.0                           # weighted mean of f = 1 - fluxc is zero
    f = 1.0 - fluxc
    wt = w / W
    durations = np.array([0.05, 0.09, 0.13])            # D/(2c) non-integer: no sample on an edge
    tpl = np.ones(64)
    g = oracle_mod.linear_search(t, fluxc, err, durations, t[0], c, n, tpl)
    periods = np.array([20, 33, 40, 57]) * c            # multiples of the t0 stride: no NN rounding
    best_sr2 = np.zeros(len(periods))
    for k, P in enumerate(periods):
        r_cells = int(round(P / c))
        for j, D in enumerate(durations):
            for p in range(r_cells):
                centres = t[p] + P * np.arange(0, 40)
                centres = centres[centres <= t[-1] + 1e-12]
                mask = np.zeros(n, bool)
                for tc in centres:
                    mask |= np.abs(t - tc) <= 0.5 * D
                s = np.sum(wt[mask] * f[mask]); r = np.sum(wt[mask])
                sr2 = s * s / (r * (1.0 - r))
                lr, z, zv, ntr = oracle_mod.periodic_cell(g, c, P, j, p)
                assert ntr == len(centres)
                assert 2.0 * lr / (W * (1.0 - r)) == pytest.approx(sr2, rel=1e-9)
                assert z == pytest.approx(s / r, rel=1e-9)          # BLS depth estimate
                best_sr2[k] = max(best_sr2[k], 0.5 * W * s * s / r)   # brute-force LR of this cell
    # the search's per-period maximum of LR is consistent with the brute-force table
    pg = oracle_mod.periodic_search(g, t[0], c, durations, periods)
    for k, P in enumerate(periods):
        assert pg.lr[k] == pytest.approx(best_sr2[k], rel=1e-9)
    assert np.argmax(pg.lr) == 2                          # injected P = 0.8 = 40 cadences


# --------------------------------------------------------------------------- P4
def test_summed_sufficient_statistics_equal_joint_fit(oracle_mod):
    """P4: sum of Eq. 4 over epochs at the common depth = direct joint WLS fit of the multi-transit
    model to the raw data, when P is a multiple of the t0 stride."""
    n, c = 900, 0.01
    sig = lambda tt: 2e-3 * _staircase_fn(((tt - 1.07 + 1.1) % 2.2 - 1.1) / 0.2371 + 0.5)
    t, flux, err = _lc(n, c, 1e-3, 21, signal=sig)
    durations = np.array([0.1537, 0.2371])
    tpl = _staircase()
    g = oracle_mod.linear_search(t, flux, err, durations, t[0], c, n, tpl)
    f, w = 1.0 - flux, 1.0 / err ** 2
    for P_cells in (220, 147):
        P = P_cells * c
        for j, D in enumerate(durations):
            for p in (0, 63, 107, P_cells - 1):
                model = np.zeros(n)
                e = 0
                while p + e * P_cells <= n - 1:
                    x = (t - (t[p] + e * P)) / D + 0.5
                    model += _staircase_fn(x)
                    e += 1
                sab = np.sum(w * model * f); saa = np.sum(w * model * model)
                lr, z, zv, ntr = oracle_mod.periodic_cell(g, c, P, j, p)
                assert ntr == e
                assert z == pytest.approx(sab / saa, rel=1e-9)
                assert zv == pytest.approx(1.0 / saa, rel=1e-10)
                ll = np.sum(-0.5 * w * (z * model - f) ** 2) + np.sum(0.5 * w * f * f)
                assert lr == pytest.approx(ll, rel=1e-8)
                assert lr == pytest.approx(0.5 * sab * sab / saa, rel=1e-8)


def test_epoch_cells_are_nearest_grid_points(oracle_mod):
    """R11 / PAPER.md:141: for P not a multiple of the stride the epochs use the NEAREST t0 cell.
    A one-hot linear grid reveals which cells a (P, p) fold touches."""
    I, s = 500, 0.01
    t0s = np.arange(I) * s
    for P in (0.7331, 1.23457, 0.31415):
        for p in (0, 7, 29):
            expected = []
            e = 0
            while True:
                target = t0s[p] + e * P
                cell = int(np.argmin(np.abs(t0s - target)))
                if target > t0s[-1] + 0.5 * s:
                    break
                expected.append(cell)
                e += 1
            depth = np.full((1, I), np.nan); var = np.full((1, I), np.nan); dl = np.full((1, I), np.nan)
            # give every cell a distinct prime-ish weight so the sum identifies the set of cells touched
            wts = 1.0 + np.arange(I) * 1e-3
            depth[0] = 1.0; var[0] = 1.0 / wts; dl[0] = 0.5 * wts
            grids = oracle_mod.LinearGrids(depth, var, dl)
            lr, z, zv, ntr = oracle_mod.periodic_cell(grids, s, P, 0, p)
            assert ntr == len(expected)
            assert 1.0 / zv == pytest.approx(np.sum(wts[expected]), rel=1e-13)


# --------------------------------------------------------------------------- P5
def test_noiseless_injection_recovered_exactly(oracle_mod):
    """P5: a noiseless periodic signal built from the template itself, on grid-aligned t0 / grid
    duration / P a multiple of the stride, is recovered at its exact period, t0, duration and depth."""
    n, c = 1200, 0.01
    D_true, P_cells, p_true, depth_true = 0.2371, 260, 91, 1.5e-3
    t = np.arange(n) * c
    sig = np.zeros(n)
    e = 0
    while p_true + e * P_cells <= n - 1:
        sig += depth_true * _staircase_fn((t - (t[p_true] + e * P_cells * c)) / D_true + 0.5)
        e += 1
    flux = 1.0 - sig
    err = np.full(n, 1e-3)
    durations = np.array([0.1129, 0.1537, 0.2371, 0.3313])
    g = oracle_mod.linear_search(t, flux, err, durations, t[0], c, n, _staircase())
    periods = np.array([130, 200, 259, 260, 261, 390, 520]) * c
    pg = oracle_mod.periodic_search(g, t[0], c, durations, periods)
    k = int(np.argmax(pg.lr))
    assert periods[k] == pytest.approx(P_cells * c)
    assert pg.j_dur[k] == 2 and pg.i_t0[k] == p_true and pg.n_transits[k] == e
    assert pg.depth[k] == pytest.approx(depth_true, rel=1e-12)
    assert pg.t0[k] == pytest.approx(t[p_true], abs=1e-12)
    # residual is zero: LR = 1/2 depth^2 * sum(A)
    assert pg.lr[k] == pytest.approx(0.5 * depth_true ** 2 / pg.depth_var[k], rel=1e-10)
    # the linear grid itself holds the exact depth at every injected epoch
    for ee in range(e):
        assert g.depth[2, p_true + ee * P_cells] == pytest.approx(depth_true, rel=1e-12)


def test_smooth_template_injection_recovers_depth_within_nn_error(oracle_mod):
    """P8 (loose): with the limb-darkened profile injected continuously and searched through the
    M=1024 nearest-neighbour table, depth comes back within the O(1 %) error PAPER.md:75 quotes."""
    from cetra_synth import transit_profile, tabulate_template
    n, c = 2000, 120.0 / 86400.0
    t = np.arange(n) * c
    D, t0, depth = 3.0 / 24.0, t[977], 4e-4
    flux = 1.0 - depth * transit_profile((t - t0) / D + 0.5)
    err = np.full(n, 5e-4)
    durations = np.array([2.0, 3.0, 4.5]) / 24.0
    g = oracle_mod.linear_search(t, flux, err, durations, t[0], c, n, tabulate_template(1024))
    jj, ii = np.unravel_index(np.nanargmax(g.dlogL), g.dlogL.shape)
    assert (jj, ii) == (1, 977)
    assert g.depth[jj, ii] == pytest.approx(depth, rel=1e-2)


# --------------------------------------------------------------------------- P6
def _read_golden():
    vals = {}
    with open(os.path.join(GOLDEN, "worked_example.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            key, *rest = line.split()
            vals[key] = [float(v) for v in rest]
    return vals


def test_paper_worked_example(oracle_mod):
    """P6: PAPER.md:121, 167 -- transits at t=10,30,50, D=5 d, 1000 ppm, P=20 d are recovered and the
    P/2 and 2P aliases are less prominent (0.6 and 2/3 of the peak for equal noiseless transits)."""
    from cetra_synth import transit_profile, tabulate_template
    gold = _read_golden()
    c = 0.05
    t = np.arange(1201) * c
    D, depth, P = gold["duration_d"][0], gold["depth_ppm"][0] * 1e-6, gold["period_d"][0]
    flux = np.ones_like(t)
    for tc in gold["transit_times_d"]:
        flux -= depth * transit_profile((t - tc) / D + 0.5)
    err = np.full(t.shape, 1e-4)
    durations = np.array([2.5, 4.0, 5.0, 6.5])
    # t0 grid 2.5 .. 57.5 d: only windows fully inside the data for D = 5 d, so that the alias
    # closed forms (which count whole windows) apply
    t0_start, n_t0 = 2.5, 1101
    g = oracle_mod.linear_search(t, flux, err, durations, t0_start, c, n_t0, tabulate_template(1024))
    # linear search: the three transits are the three top local maxima at D = 5 d
    row = g.dlogL[2]
    for tc in gold["transit_times_d"]:
        i = int(round((tc - t0_start) / c))
        assert row[i] == np.nanmax(row[i - 40:i + 41])
        assert g.depth[2, i] == pytest.approx(depth, rel=1e-2)
    periods = np.concatenate([[P / 2, P, 2 * P], np.linspace(8.0, 45.0, 149)])
    pg = oracle_mod.periodic_search(g, t0_start, c, durations, periods)
    k = int(np.argmax(pg.lr))
    assert periods[k] == P and pg.j_dur[k] == 2 and pg.n_transits[k] == 3
    assert pg.t0[k] == pytest.approx(10.0, abs=1e-9)
    assert pg.depth[k] == pytest.approx(depth, rel=1e-2)
    assert pg.lr[0] < pg.lr[1] and pg.lr[2] < pg.lr[1]
    assert pg.lr[0] / pg.lr[1] == pytest.approx(gold["alias_half_ratio"][0], rel=1e-6)
    assert pg.lr[2] / pg.lr[1] == pytest.approx(gold["alias_double_ratio"][0], rel=1e-6)


# --------------------------------------------------------------------------- P7
def test_invariances(oracle_mod):
    """P7: flux-offset scaling, error scaling, time shift, and insertion of null points."""
    from cetra_synth import tabulate_template
    n, c = 600, 0.01
    sig = lambda tt: 2e-3 * (np.abs(tt - 2.5) < 0.1)
    t, flux, err = _lc(n, c, 1e-3, 8, signal=sig)
    durations = np.array([0.0837, 0.2113])
    tpl = tabulate_template(1024)
    periods = np.array([0.9317, 1.7, 2.41])
    g = oracle_mod.linear_search(t, flux, err, durations, t[0], c, n, tpl)
    pg = oracle_mod.periodic_search(g, t[0], c, durations, periods)
    # f -> a f
    a = 3.0
    g2 = oracle_mod.linear_search(t, 1.0 - a * (1.0 - flux), err, durations, t[0], c, n, tpl)
    assert np.allclose(g2.depth, a * g.depth, rtol=1e-10, equal_nan=True)
    assert np.allclose(g2.depth_var, g.depth_var, rtol=1e-12, equal_nan=True)
    assert np.allclose(g2.dlogL, a * a * g.dlogL, rtol=1e-9, equal_nan=True)
    # sigma -> b sigma
    b = 0.5
    g3 = oracle_mod.linear_search(t, flux, b * err, durations, t[0], c, n, tpl)
    assert np.allclose(g3.depth, g.depth, rtol=1e-10, equal_nan=True)
    assert np.allclose(g3.depth_var, b * b * g.depth_var, rtol=1e-12, equal_nan=True)
    assert np.allclose(g3.dlogL, g.dlogL / (b * b), rtol=1e-9, equal_nan=True)
    # time shift of everything (power-of-two cadence so the shifted grid is exact)
    c2 = 1.0 / 128.0
    t2 = np.arange(n) * c2
    d2 = durations * c2 / c
    ga = oracle_mod.linear_search(t2, flux, err, d2, t2[0], c2, n, tpl)
    gb = oracle_mod.linear_search(t2 + 1024.0, flux, err, d2, t2[0] + 1024.0, c2, n, tpl)
    assert np.array_equal(ga.depth, gb.depth, equal_nan=True)
    # null points between the observations: twice the sampling, stride 2 samples
    tt = np.arange(2 * n - 1) * (c2 / 2)
    fl = np.full(2 * n - 1, np.nan); er = np.full(2 * n - 1, np.inf)
    fl[::2] = flux; er[::2] = err
    gn = oracle_mod.linear_search(tt, fl, er, d2, tt[0], c2, n, tpl)
    assert np.allclose(gn.depth, ga.depth, rtol=1e-12, equal_nan=True)
    assert np.allclose(gn.dlogL, ga.dlogL, rtol=1e-12, equal_nan=True)
    # periodic results inherit the scalings
    pg2 = oracle_mod.periodic_search(g2, t[0], c, durations, periods)
    assert np.array_equal(pg2.i_t0, pg.i_t0) and np.array_equal(pg2.j_dur, pg.j_dur)
    assert np.allclose(pg2.lr, a * a * pg.lr, rtol=1e-9)
    assert np.allclose(pg2.depth, a * pg.depth, rtol=1e-9)


# --------------------------------------------------------------------------- P9 / R12 / R13
def test_null_semantics(oracle_mod):
    """P9: cells whose window holds no observation are null; partially covered windows are not
    (PAPER.md:123).  Null inputs are NaN flux, infinite or non-positive error."""
    from cetra_synth import tabulate_template
    n, c = 400, 0.01
    t, flux, err = _lc(n, c, 1e-3, 2)
    flux[100:160] = np.nan; err[100:160] = np.inf          # 0.6 d gap
    err[300] = 0.0; flux[301] = np.inf
    durations = np.array([0.0837, 0.2113])
    g = oracle_mod.linear_search(t, flux, err, durations, t[0] - 0.5, c, n + 100, tabulate_template(256))
    centre = (np.arange(n + 100) - 50) * c
    for j, D in enumerate(durations):
        x_lo, x_hi = centre - D / 2, centre + D / 2
        good = np.isfinite(flux) & np.isfinite(err) & (err > 0)
        # interior samples only (template is 0 exactly at first/last contact)
        has = np.array([np.any(good & (t > lo + 1e-9) & (t < hi - 1e-9)) for lo, hi in zip(x_lo, x_hi)])
        assert np.array_equal(np.isnan(g.depth[j]), ~has)
        assert np.array_equal(np.isnan(g.depth_var[j]), ~has)
        assert np.array_equal(np.isnan(g.dlogL[j]), ~has)
    assert np.isnan(g.depth[0, 0]) and not np.isnan(g.depth[0, 50 + 3])   # t < D/2 padding vs partial window


def test_duration_must_be_shorter_than_period_and_ties(oracle_mod):
    """PAPER.md:145 (D < P strictly), optional duration ranges, tie rule R13, empty period."""
    I, s = 300, 0.01
    depth = np.ones((3, I)); var = np.ones((3, I)); dl = 0.5 * np.ones((3, I))
    grids = oracle_mod.LinearGrids(depth, var, dl)
    durations = np.array([0.05, 0.5, 1.0])
    periods = np.array([0.5, 0.75, 1.5])
    pg = oracle_mod.periodic_search(grids, 0.0, s, durations, periods)
    # identical cells: LR = n_tr/2, maximal at the smallest phase; ties -> smallest j, then smallest p
    assert list(pg.j_dur) == [0, 0, 0] and list(pg.i_t0) == [0, 0, 0]
    assert list(pg.n_transits) == [6, 4, 2]
    lo = np.array([1, 1, 1], np.int32); hi = np.array([3, 3, 3], np.int32)
    pg = oracle_mod.periodic_search(grids, 0.0, s, durations, periods, lo, hi)
    assert list(pg.j_dur) == [-1, 1, 1]                   # P=0.5: D=0.5 is not < P, D=1.0 neither
    assert np.isnan(pg.lr[0]) and pg.i_t0[0] == -1


# ------------------------------------------------------------ branches that GPU parity cannot see
# The three tests below each kill one plausible mistake that the CUDA path would share by construction
# (VERDICT round 1): a fold that stops at the first null epoch instead of skipping it, floor(P/s) phases
# instead of ceil(P/s), and a window that drops the sample sitting exactly on its last (or first) instant.
def _nearest_cells(I, s, P, p):
    """Cells a (P, p) fold touches, from the definition: the grid point nearest to t0_p + e P."""
    t0s = np.arange(I) * s
    out, e = [], 0
    while t0s[p] + e * P <= t0s[-1] + 0.5 * s:
        out.append(int(np.argmin(np.abs(t0s - (t0s[p] + e * P)))))
        e += 1
    return out


def test_fold_skips_null_epochs_hand_built_grid(oracle_mod):
    """PAPER.md:123 ("no influence on either the depth or the likelihood ratio"): epochs whose cell is null are
    skipped, the later epochs still contribute.  Kills `continue -> break` on a null epoch in fold_cell."""
    I, s = 500, 0.01
    wts = 1.0 + np.arange(I) * 1e-3                     # distinct weights: the sum identifies the set of cells
    dep = 1.0 + 0.25 * np.sin(np.arange(I) * 0.37)
    for P, p in ((0.7331, 7), (0.31415, 29), (1.23457, 0)):
        cells = _nearest_cells(I, s, P, p)
        assert len(cells) >= 4
        null = [cells[1], cells[3]] if len(cells) >= 5 else [cells[1]]
        kept = [c for c in cells if c not in null]
        depth = dep[None, :].copy(); var = (1.0 / wts)[None, :].copy()
        dl = 0.5 * depth ** 2 / var
        for arr in (depth, var, dl):
            arr[0, null] = np.nan
        grids = oracle_mod.LinearGrids(depth, var, dl)
        lr, z, zv, ntr = oracle_mod.periodic_cell(grids, s, P, 0, p)
        assert ntr == len(cells) - len(null)
        assert 1.0 / zv == pytest.approx(np.sum(wts[kept]), rel=1e-13)
        assert z == pytest.approx(np.sum(wts[kept] * dep[kept]) / np.sum(wts[kept]), rel=1e-13)
        assert lr == pytest.approx(0.5 * np.sum(wts[kept] * dep[kept]) ** 2 / np.sum(wts[kept]), rel=1e-12)
        # the per-period search reports the same element (every other phase is left null)
        only = np.full((1, I), np.nan)
        d1, v1, l1 = only.copy(), only.copy(), only.copy()
        d1[0, kept], v1[0, kept], l1[0, kept] = depth[0, kept], var[0, kept], dl[0, kept]
        pg = oracle_mod.periodic_search(oracle_mod.LinearGrids(d1, v1, l1), 0.0, s, np.array([0.05]), np.array([P]))
        assert pg.i_t0[0] == p and pg.n_transits[0] == len(kept)
        assert pg.lr[0] == pytest.approx(lr, rel=1e-13)


def test_fold_across_a_data_gap_equals_joint_fit(oracle_mod):
    """P4 with a gap longer than the duration: the epoch that falls in the gap has a null linear cell, the joint
    weighted least-squares fit of the multi-transit model to the raw data ignores it (its points carry no
    weight), and the folded statistics must agree with that fit.  Kills `continue -> break`."""
    n, c = 1100, 0.01
    P_cells, p = 220, 63
    sig = lambda tt: 2e-3 * _staircase_fn(((tt - 0.63 + 1.1) % 2.2 - 1.1) / 0.2371 + 0.5)
    t, flux, err = _lc(n, c, 1e-3, 33, signal=sig)
    gap = slice(p + P_cells - 30, p + P_cells + 31)        # 0.6 d around the second epoch; D <= 0.2371 d
    flux[gap] = np.nan; err[gap] = np.inf
    durations = np.array([0.1537, 0.2371])
    g = oracle_mod.linear_search(t, flux, err, durations, t[0], c, n, _staircase())
    assert np.isnan(g.depth[:, p + P_cells]).all() and not np.isnan(g.depth[:, p + 2 * P_cells]).any()
    good = np.isfinite(flux)
    f = np.where(good, 1.0 - np.where(good, flux, 1.0), 0.0)
    w = np.where(good, 1.0 / np.where(good, err, 1.0) ** 2, 0.0)
    P = P_cells * c
    for j, D in enumerate(durations):
        model = np.zeros(n)
        e = 0
        while p + e * P_cells <= n - 1:
            model += _staircase_fn((t - (t[p] + e * P)) / D + 0.5)
            e += 1
        assert e == 5
        sab, saa = np.sum(w * model * f), np.sum(w * model * model)
        lr, z, zv, ntr = oracle_mod.periodic_cell(g, c, P, j, p)
        assert ntr == e - 1                                # four of the five epochs have data
        assert z == pytest.approx(sab / saa, rel=1e-9)
        assert zv == pytest.approx(1.0 / saa, rel=1e-10)
        assert lr == pytest.approx(0.5 * sab * sab / saa, rel=1e-8)
        ll = np.sum(-0.5 * w * (z * model - f) ** 2) + np.sum(0.5 * w * f * f)
        assert lr == pytest.approx(ll, rel=1e-8)


def test_phase_count_is_ceil_of_period_in_cells(oracle_mod):
    """R10: the first epoch may sit in any cell p with p*s < P, i.e. p < ceil(P/s).  For a non-integer P/s a
    signal whose first epoch is cell floor(P/s) is a phase of its own (no earlier phase touches the same
    cells).  Kills `n_phase = ceil(r) -> floor(r)`."""
    I, s = 400, 0.01
    r = 57.4
    P = r * s
    p_star = 57                                            # = floor(r) < ceil(r) = 58
    assert p_star * s < P
    cells = _nearest_cells(I, s, P, p_star)
    depth = np.zeros((1, I)); var = np.ones((1, I))
    depth[0, cells] = 1.0
    dl = 0.5 * depth ** 2 / var
    grids = oracle_mod.LinearGrids(depth, var, dl)
    pg = oracle_mod.periodic_search(grids, 0.0, s, np.array([0.05]), np.array([P]))
    assert pg.i_t0[0] == p_star and pg.i_t0[0] < int(np.ceil(r))
    assert pg.n_transits[0] == len(cells)
    assert pg.lr[0] == pytest.approx(0.5 * len(cells), rel=1e-13)
    # no phase below floor(r) reaches that likelihood: a floor(r)-phase search would lose the peak
    others = [oracle_mod.periodic_cell(grids, s, P, 0, q)[0] for q in range(p_star)]
    assert max(others) < 0.5 * pg.lr[0]
    # the same from raw data: box transits centred on cell 57 + nearest(e r) of a noiseless light curve
    n = I
    t = np.arange(n) * s
    flux = np.ones(n)
    for cc in cells:
        flux[max(cc - 2, 0):cc + 3] -= 1e-3
    g = oracle_mod.linear_search(t, flux, np.full(n, 1e-4), np.array([0.045]), 0.0, s, n, np.ones(16))
    pg2 = oracle_mod.periodic_search(g, 0.0, s, np.array([0.045]), np.array([P]))
    assert pg2.i_t0[0] == p_star and pg2.depth[0] == pytest.approx(1e-3, rel=1e-9)
    # integer P/s (power-of-two stride, so that P/s is exact): ceil = floor, the last phase is r - 1; the only
    # signal sits in cells 57 + 57 e, which is phase 0's second epoch onward, so the winner is a phase < 57
    s2 = 1.0 / 128.0
    d3 = np.zeros((1, I)); d3[0, 57::57] = 1.0
    g3 = oracle_mod.LinearGrids(d3, np.ones((1, I)), 0.5 * d3 ** 2)
    pg3 = oracle_mod.periodic_search(g3, 0.0, s2, np.array([0.05]), np.array([57 * s2]))
    assert pg3.i_t0[0] == 0 and pg3.n_transits[0] == len(range(0, I, 57))


def test_window_includes_samples_on_its_first_and_last_instant(oracle_mod):
    """R2 (first and last element of the window, both inclusive): with D/(2c) a whole number the
    samples at t_i -+ D/2 sit exactly on x = 0 and x = 1 and belong to the window.  Box template = the BLS
    window of P3 with edge samples; a staircase template fixes which template end each edge sample takes.
    Kills `x <= 1 -> x < 1` (and `x >= 0 -> x > 0`)."""
    n, c = 300, 1.0 / 64.0                                 # power-of-two cadence: k*c and D/2 are exact
    t, flux, err = _lc(n, c, 1e-3, 17)
    f, w = 1.0 - flux, 1.0 / err ** 2
    for h in (3, 7):
        D = 2.0 * (h * c)
        g = oracle_mod.linear_search(t, flux, err, np.array([D]), t[0], c, n, np.ones(32))
        gs = oracle_mod.linear_search(t, flux, err, np.array([D]), t[0], c, n, _staircase())
        for i in (0, 2, 50, 151, n - 1):
            win = np.abs(t - t[i]) <= 0.5 * D               # inclusive on both sides
            assert win.sum() == min(i, h) + min(n - 1 - i, h) + 1
            assert g.depth_var[0, i] == pytest.approx(1.0 / np.sum(w[win]), rel=1e-13)
            assert g.depth[0, i] == pytest.approx(np.sum(w[win] * f[win]) / np.sum(w[win]), rel=1e-12)
            # staircase: tpl = 0.5 at first contact, 0.25 at last contact
            m = _staircase_fn((t - t[i]) / D + 0.5)
            assert m[i - h] == 0.5 if i >= h else True
            assert m[i + h] == 0.25 if i + h < n else True
            assert gs.depth_var[0, i] == pytest.approx(1.0 / np.sum(w * m * m), rel=1e-13)
            assert gs.depth[0, i] == pytest.approx(np.sum(w * m * f) / np.sum(w * m * m), rel=1e-12)
    # the off-grid form (R25) takes the same decision: t0 grid shifted by a quarter cadence, D/2 = (h + 1/4) c
    h = 5
    D = 2.0 * ((h + 0.25) * c)
    gg = oracle_mod.linear_search(t, flux, err, np.array([D]), t[0] + 0.25 * c, c, n - 1, np.ones(32))
    for i in (40, 200):
        ti = t[0] + 0.25 * c + i * c
        win = np.abs(t - ti) <= 0.5 * D
        assert win.sum() == 2 * h + 1 and t[win][0] - ti == -0.5 * D      # the first sample sits exactly on x = 0
        assert gg.depth_var[0, i] == pytest.approx(1.0 / np.sum(w[win]), rel=1e-13)

"""Pins of the oracle's off-grid t0 form (R25; the paper's default t0 stride is 1 % of the shortest duration,
PAPER.md:87, which does not sit on the sample grid).  CPU only."""
import numpy as np
import pytest

from parity_util import nearest_template_sample


def _lc(n, c, sigma, seed):
    rng = np.random.default_rng(seed)
    t = 2.5 + c * np.arange(n)
    f = 1.0 + sigma * rng.standard_normal(n)
    e = np.full(n, sigma) * rng.uniform(0.7, 1.4, n)
    f[n // 3: n // 3 + 17] = np.nan
    return t, f, e


def _tpl(M=1024):
    from cetra_synth import tabulate_template
    return tabulate_template(M).astype(np.float64)


def test_general_form_reduces_to_the_on_grid_form(oracle_mod):
    # an on-grid t0 grid evaluated through the time-difference form (R25) agrees with the integer-offset form (R3),
    # which the pins of test_oracle_pins.py fix; durations are not multiples of the cadence, so that no sample sits
    # on a window edge or a template-index boundary where 1e-16 of rounding could flip a nearest-neighbour choice
    c = 2.0 / 1440.0
    t, f, e = _lc(900, c, 8e-4, 1)
    durations = np.array([0.0213, 0.0517, 0.0931, 0.1777])
    a = oracle_mod.linear_search(t, f, e, durations, t[0] - 5 * c, 2 * c, 460, _tpl())
    b = oracle_mod.linear_search(t, f, e, durations, t[0] - 5 * c, 2 * c, 460, _tpl(), force_general=True)
    for x, y in ((a.depth, b.depth), (a.depth_var, b.depth_var), (a.dlogL, b.dlogL)):
        assert np.array_equal(np.isnan(x), np.isnan(y))
        ok = ~np.isnan(x)
        assert np.allclose(x[ok], y[ok], rtol=1e-10, atol=1e-18)
    assert np.isnan(a.depth).sum() > 0 and (~np.isnan(a.depth)).sum() > 1000


def test_off_grid_cell_is_the_weighted_least_squares_fit(oracle_mod):
    c = 2.0 / 1440.0
    t, f, e = _lc(700, c, 8e-4, 2)
    tpl = _tpl(512)
    durations = np.array([0.0317, 0.0871])
    s = 0.01 * durations[0]                                   # 1 % of the minimum duration
    t0_start = t[0] + 0.123 * c
    n_t0 = 2500
    g = oracle_mod.linear_search(t, f, e, durations, t0_start, s, n_t0, tpl)
    rng = np.random.default_rng(0)
    for j, D in enumerate(durations):
        for i in rng.integers(0, n_t0, 6):
            ti = t0_start + i * s
            x = (t - ti) / D + 0.5
            win = (x >= 0) & (x <= 1) & np.isfinite(f)
            assert np.min(np.abs(x[np.isfinite(f)] - 0.0)) > 1e-9 and np.min(np.abs(x[np.isfinite(f)] - 1.0)) > 1e-9
            # the template sample of every observation from the definition (distances to the tabulated positions),
            # not from the oracle's rounding expression
            idx, margin = nearest_template_sample(x[win], len(tpl))
            assert margin.min() > 1e-9
            m = tpl[idx]
            sw = 1.0 / e[win]
            sol, *_ = np.linalg.lstsq((sw * m)[:, None], sw * (1.0 - f[win]), rcond=None)
            assert g.depth[j, i] == pytest.approx(sol[0], rel=1e-9)
            assert g.depth_var[j, i] == pytest.approx(1.0 / np.sum((sw * m) ** 2), rel=1e-9)
            assert g.dlogL[j, i] == pytest.approx(0.5 * g.depth[j, i] ** 2 / g.depth_var[j, i], rel=1e-9)


def test_quarter_sample_stride_shift_invariance(oracle_mod):
    # stride = c/4: delaying the data by one sample moves every result by four cells
    c = 10.0 / 1440.0
    t, f, e = _lc(400, c, 5e-4, 3)
    durations = np.array([0.0533, 0.1291])
    tpl = _tpl(256)
    s = c / 4
    a = oracle_mod.linear_search(t, f, e, durations, t[0] + 0.37 * c, s, 1400, tpl)
    f2, e2 = np.roll(f, 1), np.roll(e, 1)
    f2[0] = np.nan
    b = oracle_mod.linear_search(t, f2, e2, durations, t[0] + 0.37 * c, s, 1400, tpl)
    # cells whose window stays clear of the wrapped sample
    lo = int(durations.max() / s) + 8
    for x, y in ((a.depth, b.depth), (a.depth_var, b.depth_var), (a.dlogL, b.dlogL)):
        xa, yb = x[:, lo:1396 - 4], y[:, lo + 4:1396]
        assert np.array_equal(np.isnan(xa), np.isnan(yb))
        ok = ~np.isnan(xa)
        assert np.allclose(xa[ok], yb[ok], rtol=1e-9, atol=1e-18)


def test_off_grid_noiseless_injection_recovered_exactly(oracle_mod):
    c = 2.0 / 1440.0
    n = 1200
    t = c * np.arange(n)
    tpl = _tpl(1024)
    durations = np.array([0.05, 0.0831, 0.13])
    s = 0.01 * durations[0]
    t0_start = 0.2
    i_star, j_star, depth = 1234, 1, 1.7e-3
    ti = (t0_start - t[0]) + i_star * s
    x = (np.arange(n) * c - ti) / durations[j_star] + 0.5
    ins = (x >= 0) & (x <= 1)
    m = np.zeros(n)
    idx, margin = nearest_template_sample(x[ins], 1024)
    assert margin.min() > 1e-9
    m[ins] = tpl[idx]
    f = 1.0 - depth * m
    e = np.full(n, 3e-4)
    g = oracle_mod.linear_search(t, f, e, durations, t0_start, s, 3000, tpl)
    assert g.depth[j_star, i_star] == pytest.approx(depth, rel=1e-12)
    assert g.dlogL[j_star, i_star] == pytest.approx(0.5 * depth ** 2 * np.sum(m ** 2) / 9e-8, rel=1e-10)
    j, i = np.unravel_index(np.nanargmax(g.dlogL), g.dlogL.shape)
    assert j == j_star and abs(i - i_star) <= 1            # neighbours one hundredth of a duration away tie to ~1e-4
    assert g.dlogL[j_star, i_star] >= np.nanmax(g.dlogL) * (1 - 1e-12)


def _stair(x):
    """0.5 on the outer quarters, 1 on the middle half, 0.25 on the last tenth, 0 outside [0, 1]."""
    v = np.where((x >= 0.25) & (x <= 0.75), 1.0, 0.5)
    v = np.where(x > 0.9, 0.25, v)
    return np.where((x < 0) | (x > 1), 0.0, v)


def test_off_grid_template_position_from_the_definition(oracle_mod):
    """The template value of every sample follows from x = (t_n - t_i)/D + 1/2 alone when the template is
    piecewise constant (no index expression is retyped here): pins the orientation, the window placement and the
    nearest-neighbour position of the R25 form, cell by cell, against a library least-squares solve."""
    c = 2.0 / 1440.0
    t, f, e = _lc(700, c, 8e-4, 5)
    M = 2048
    tpl = _stair(np.arange(M) / (M - 1.0))
    durations = np.array([0.0317, 0.0871])
    s = 0.01 * durations[0]
    t0_start = t[0] - 0.4 * durations[1]
    n_t0 = 3000
    g = oracle_mod.linear_search(t, f, e, durations, t0_start, s, n_t0, tpl)
    ok = np.isfinite(f)
    rng = np.random.default_rng(4)
    checked = 0
    for j, D in enumerate(durations):
        for i in rng.integers(0, n_t0, 40):
            x = (t - (t0_start + i * s)) / D + 0.5
            # skip cells with a sample within half a template step of a staircase edge or a window edge
            edges = np.concatenate([x[ok] - 0.25, x[ok] - 0.75, x[ok] - 0.9, x[ok], x[ok] - 1.0])
            if np.min(np.abs(edges)) < 1.0 / (M - 1):
                continue
            m = _stair(x) * ok
            if not m.any():
                assert np.isnan(g.depth[j, i])
                continue
            sw = np.where(ok, 1.0 / e, 0.0)
            sol, *_ = np.linalg.lstsq((sw * m)[:, None], sw * np.where(ok, 1.0 - f, 0.0), rcond=None)
            assert g.depth[j, i] == pytest.approx(sol[0], rel=1e-9)
            assert g.depth_var[j, i] == pytest.approx(1.0 / np.sum((sw * m) ** 2), rel=1e-10)
            checked += 1
    assert checked > 40


def test_on_grid_decision_bounds_the_drift_at_the_last_cell(oracle_mod):
    """A stride that misses a whole number of cadences by 5e-7 samples drifts by half a sample over 1e6 cells:
    such a grid is NOT on the sample grid.  With I cells the R3 (integer offset) form is used only while
    |a - round a| + |b - round b| (I - 1) <= 1e-6 samples; beyond that the exact-time form (R25) decides.  A
    staircase template makes the two forms differ visibly once the drift crosses a template edge."""
    c = 1.0 / 64.0
    n = 4000
    rng = np.random.default_rng(9)
    t = c * np.arange(n)
    e = 1e-3 * (0.5 + rng.random(n))
    f = 1.0 + e * rng.standard_normal(n)
    M = 256
    tpl = _stair(np.arange(M) / (M - 1.0))
    D = np.array([8.3 * c])
    # (1) mismatch 2e-10 per cell, 3000 cells: drift 6e-7 -> on grid: identical to the exact integer stride
    a = oracle_mod.linear_search(t, f, e, D, t[0], c, 3000, tpl)
    b = oracle_mod.linear_search(t, f, e, D, t[0], c * (1 + 2e-10), 3000, tpl)
    assert np.array_equal(a.depth, b.depth, equal_nan=True)
    # (2) mismatch 1e-4 per cell: after 3000 cells the grid is 0.3 samples late; the result must be the exact-time
    #     form's, i.e. the WLS fit with the template taken at the true (t_n - t_i)/D + 1/2
    s = c * (1 + 1e-4)
    g = oracle_mod.linear_search(t, f, e, D, t[0], s, 3000, tpl)
    w = 1.0 / e ** 2
    checked = differs = 0
    for i in list(range(5, 3000, 97)) + list(range(2900, 3000)):
        x = (t - (t[0] + i * s)) / D[0] + 0.5
        if np.min(np.abs(np.concatenate([x - 0.25, x - 0.75, x - 0.9, x, x - 1.0]))) < 1.0 / (M - 1):
            continue
        m = _stair(x)
        assert g.depth_var[0, i] == pytest.approx(1.0 / np.sum(w * m * m), rel=1e-12)
        checked += 1
        differs += int(abs(g.depth_var[0, i] / a.depth_var[0, i] - 1.0) > 1e-6)
    assert checked >= 50 and differs >= 20              # the drifted grid is visibly not the integer-stride grid

"""Pins of the oracle's setup / follow-up steps (oracle/cetra_oracle_setup.c) against what the paper and the
mathematics fix: resampling, median cadence, monotransit events
 and transit masking.  CPU only."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


# ------------------------------------------------------------------------------------------- resampling
def test_resample_is_identity_on_a_regular_grid(oracle_mod):
    rng = np.random.default_rng(11)
    n, c = 500, 2.0 / 1440.0
    t = 3.25 + c * np.arange(n)
    f = 1.0 + 1e-3 * rng.standard_normal(n)
    e = rng.uniform(5e-4, 2e-3, n)
    of, oe = oracle_mod.resample(t, f, e, t[0], c, n)
    # one observation per output point: the weighted mean of one value is that value (to rounding),
    # its formal error is the observation's own
    assert np.allclose(of, f, rtol=1e-15, atol=0)
    assert np.allclose(oe, e, rtol=1e-15, atol=0)


def test_resample_two_points_in_a_cell_closed_form(oracle_mod):
    # f1 +- s1 and f2 +- s2 in one cell: mean = (f1/s1^2 + f2/s2^2)/(1/s1^2 + 1/s2^2), error = (1/s1^2+1/s2^2)^-1/2
    t = np.array([0.1, 0.3, 1.2])
    f = np.array([1.0, 3.0, 7.0])
    e = np.array([1.0, 2.0, 0.5])
    of, oe = oracle_mod.resample(t, f, e, 0.0, 1.0, 3)
    assert of[0] == pytest.approx((1.0 / 1.0 + 3.0 / 4.0) / (1.0 + 0.25), rel=1e-15)     # 1.4
    assert oe[0] == pytest.approx((1.0 + 0.25) ** -0.5, rel=1e-15)
    assert of[1] == 7.0 and oe[1] == pytest.approx(0.5, rel=1e-15)
    assert np.isnan(of[2]) and np.isinf(oe[2]) and oe[2] > 0                              # null: PAPER.md:55
    # equal errors: plain mean, error / sqrt(2)
    of, oe = oracle_mod.resample([0.0, 0.2], [2.0, 4.0], [0.3, 0.3], 0.0, 1.0, 1)
    assert of[0] == pytest.approx(3.0, rel=1e-15) and oe[0] == pytest.approx(0.3 / np.sqrt(2.0), rel=1e-15)


def test_resample_matches_bincount_brute_force_and_ignores_order(oracle_mod):
    rng = np.random.default_rng(5)
    n_in, c, n_out = 4000, 0.01, 900
    t = np.sort(rng.uniform(-0.5, 9.5, n_in))           # irregular, denser than the grid, runs off both ends
    f = 1.0 + 1e-2 * rng.standard_normal(n_in)
    e = rng.uniform(1e-3, 5e-3, n_in)
    f[::97] = np.nan                                    # null observations are dropped (R8)
    e[5::131] = -1.0
    of, oe = oracle_mod.resample(t, f, e, 0.0, c, n_out)
    ok = np.isfinite(f) & np.isfinite(e) & (e > 0)
    cell = np.floor(t / c + 0.5).astype(np.int64)
    ok &= (cell >= 0) & (cell < n_out)
    w = 1.0 / e[ok] ** 2
    sw = np.bincount(cell[ok], weights=w, minlength=n_out)
    swf = np.bincount(cell[ok], weights=w * f[ok], minlength=n_out)
    has = sw > 0
    assert np.array_equal(has, np.isfinite(of))
    assert np.allclose(of[has], swf[has] / sw[has], rtol=1e-13)
    assert np.allclose(oe[has], sw[has] ** -0.5, rtol=1e-13)
    assert np.all(np.isinf(oe[~has]))
    # one cell against numpy.average
    k = int(np.argmax(np.bincount(cell[ok], minlength=n_out)))
    sel = ok & (cell == k)
    assert of[k] == pytest.approx(np.average(f[sel], weights=1.0 / e[sel] ** 2), rel=1e-13)
    # "avoids any need for ... sorting": the input order does not matter
    perm = rng.permutation(n_in)
    of2, oe2 = oracle_mod.resample(t[perm], f[perm], e[perm], 0.0, c, n_out)
    assert np.allclose(of2[has], of[has], rtol=1e-13) and np.allclose(oe2[has], oe[has], rtol=1e-13)


def test_resample_assigns_to_the_nearest_output_point(oracle_mod):
    # points at 0.49 c and 0.51 c around the boundary between cells 0 and 1; 1.5 c goes up (R21)
    c = 0.25
    t = np.array([0.49 * c, 0.51 * c, 1.5 * c, -0.49 * c, -0.51 * c])
    f = np.array([10.0, 20.0, 30.0, 40.0, 50.0])
    of, _ = oracle_mod.resample(t, f, np.ones(5), 0.0, c, 4)
    assert of[0] == pytest.approx(25.0)        # 10 and 40 (both within half a cadence of point 0)
    assert of[1] == pytest.approx(20.0)
    assert of[2] == pytest.approx(30.0)
    assert np.isnan(of[3])                     # -0.51 c is before the grid: dropped


def test_resample_template_is_numpy_interp_and_keeps_a_linear_model(oracle_mod):
    """the supplied model is resampled "using simple linear interpolation".  Pins: numpy.interp on the
    same positions; a straight-line model is reproduced exactly at every output sample; the same sample count is the
    identity; the end samples are kept."""
    rng = np.random.default_rng(4)
    model = np.cumsum(rng.normal(size=317))
    for n_out in (2, 5, 317, 1024):
        got = oracle_mod.resample_template(model, n_out)
        want = np.interp(np.linspace(0.0, 316.0, n_out), np.arange(317.0), model)
        assert np.allclose(got, want, rtol=0, atol=1e-12 * np.abs(model).max())
        assert got[0] == model[0] and abs(got[-1] - model[-1]) <= 1e-12 * abs(model[-1])
    assert np.allclose(oracle_mod.resample_template(model, 317), model, rtol=0, atol=1e-12 * np.abs(model).max())
    line = 3.0 - 0.25 * np.arange(41.0)
    assert np.allclose(oracle_mod.resample_template(line, 1001), np.linspace(line[0], line[-1], 1001), rtol=0, atol=1e-12)


def test_median_cadence_is_numpy_median_of_differences(oracle_mod):
    rng = np.random.default_rng(3)
    t = np.cumsum(rng.choice([1.0, 1.0, 1.0, 2.0, 7.5], size=1001) * 2.0 / 1440.0)
    assert oracle_mod.median_cadence(t) == pytest.approx(np.median(np.diff(t)), rel=1e-15)
    assert oracle_mod.median_cadence(t[:1000]) == pytest.approx(np.median(np.diff(t[:1000])), rel=1e-15)
    assert oracle_mod.median_cadence(t[rng.permutation(1001)]) == pytest.approx(np.median(np.diff(t)), rel=1e-15)
    assert oracle_mod.median_cadence(np.arange(50) * 0.125) == 0.125


# ----------------------------------------------------------------------------------------- monotransits
def _grids(oracle_mod, seed=0, n=700, n_dur=5):
    from cetra_synth import transit_profile
    rng = np.random.default_rng(seed)
    c = 10.0 / 1440.0
    t = c * np.arange(n)
    f = 1.0 + 4e-4 * rng.standard_normal(n)
    for tc, d in ((1.1, 2e-3), (3.3, 1.5e-3)):
        x = (t - tc) / 0.2 + 0.5
        inside = (x >= 0) & (x <= 1)
        f[inside] -= d * transit_profile(x[inside])
    e = np.full(n, 4e-4)
    f[300:330] = np.nan
    durations = np.array([0.08, 0.12, 0.2, 0.3, 0.45])[:n_dur]
    tpl = transit_profile(np.linspace(0, 1, 256))
    g = oracle_mod.linear_search(t, f, e, durations, t[0], c, n, tpl)
    return t, c, durations, g


def test_monotransit_profile_and_greedy_peaks_brute_force(oracle_mod):
    t, c, durations, g = _grids(oracle_mod)
    m = oracle_mod.monotransit(g, c, durations, n_peaks=6, excl=1.0)
    dl = g.dlogL
    filled = np.where(np.isnan(dl), -np.inf, dl)
    pj = np.argmax(filled, axis=0)                                  # first maximum: smallest j on ties
    pl = filled.max(axis=0)
    allnull = np.all(np.isnan(dl), axis=0)
    assert np.array_equal(m.profile_j, np.where(allnull, -1, pj))
    assert np.array_equal(np.isnan(m.profile_lr), allnull)
    assert np.array_equal(m.profile_lr[~allnull], pl[~allnull])
    # greedy picking written out in numpy
    alive = ~allnull
    ev = []
    for _ in range(6):
        if not alive.any():
            break
        cand = np.where(alive, pl, -np.inf)
        i = int(np.argmax(cand))
        ev.append(i)
        alive &= np.abs((np.arange(len(pl)) - i) * c) > 1.0 * durations[pj[i]]
    assert list(m.i_t0) == ev
    assert np.array_equal(m.j_dur, pj[ev])
    assert np.array_equal(m.lr, pl[ev])
    assert np.array_equal(m.depth, g.depth[pj[ev], ev]) and np.array_equal(m.depth_var, g.depth_var[pj[ev], ev])
    # the two injected single transits (t = 1.1 d and 3.3 d, D = 0.2 d) are the two strongest events
    top = sorted(t[m.i_t0[:2]])
    assert abs(top[0] - 1.1) < 0.02 and abs(top[1] - 3.3) < 0.02
    assert all(durations[j] == 0.2 for j in m.j_dur[:2])
    # events do not overlap: later events lie outside excl * D of every earlier one
    for a in range(len(ev)):
        for b in range(a + 1, len(ev)):
            assert abs((ev[b] - ev[a]) * c) > durations[pj[ev[a]]]


def test_monotransit_runs_out_of_candidates(oracle_mod):
    t, c, durations, g = _grids(oracle_mod, n=120)
    m = oracle_mod.monotransit(g, c, durations, n_peaks=50, excl=3.0)
    assert 1 <= len(m.i_t0) < 50          # 120 cells, each event removes > 2*3*0.08 d = 69 cells... a handful fit
    assert len(set(m.i_t0)) == len(m.i_t0)


# ---------------------------------------------------------------------------------------------- masking
def test_mask_transits_matches_direct_modulo_and_closed_form_count(oracle_mod):
    c = 2.0 / 1440.0
    n = 19728
    t = c * np.arange(n)
    f = np.ones(n)
    P, t0, D, width = 5.3, 1.7, 3.0 / 24.0, 1.5
    out, cnt = oracle_mod.mask_transits(t, f, P, t0, D, width)
    phase = np.mod(t - t0 + 0.5 * P, P) - 0.5 * P
    expect = np.abs(phase) <= 0.5 * width * D
    assert np.array_equal(np.isnan(out), expect) and cnt == int(expect.sum())
    assert np.all(out[~expect] == 1.0)
    # 6 epochs inside the 27.4 d baseline (1.7 + 5.3 e, e = 0..4 -> 5 epochs; e = 5 is 28.2 > 27.4): each masks
    # width*D/c = 135 samples, give or take one
    n_epochs = int(np.sum((t0 + P * np.arange(-1, 8) >= 0) & (t0 + P * np.arange(-1, 8) <= t[-1])))
    assert n_epochs == 5
    assert abs(cnt - n_epochs * width * D / c) <= n_epochs
    # a single event (period <= 0) masks one window only; width = 0 masks nothing off the grid
    out1, cnt1 = oracle_mod.mask_transits(t, f, 0.0, t0, D, 1.0)
    assert cnt1 == int(np.sum(np.abs(t - t0) <= 0.5 * D)) and 89 <= cnt1 <= 91
    _, cnt0 = oracle_mod.mask_transits(t + 0.3 * c, f, P, t0, D, 0.0)
    assert cnt0 == 0


def test_masking_the_best_signal_removes_it_from_the_next_search(oracle_mod):
    # after nullifying the strongest signal the search finds the next one
    from cetra_synth import transit_profile
    rng = np.random.default_rng(8)
    c, n = 10.0 / 1440.0, 1440
    t = c * np.arange(n)
    f = 1.0 + 3e-4 * rng.standard_normal(n)
    planets = ((2.0, 0.4, 0.15, 3e-3), (3.1, 1.3, 0.15, 1.5e-3))
    for P, t0, D, d in planets:
        ph = np.mod(t - t0 + 0.5 * P, P) - 0.5 * P
        x = ph / D + 0.5
        ins = (x >= 0) & (x <= 1)
        f[ins] -= d * transit_profile(x[ins])
    e = np.full(n, 3e-4)
    durations = np.array([0.1, 0.15, 0.2])
    tpl = transit_profile(np.linspace(0, 1, 512))
    periods = np.linspace(1.5, 4.0, 251)
    found = []
    for _ in range(2):
        g = oracle_mod.linear_search(t, f, e, durations, t[0], c, n, tpl)
        pg = oracle_mod.periodic_search(g, t[0], c, durations, periods)
        k = int(np.nanargmax(pg.lr))
        found.append(periods[k])
        f, _ = oracle_mod.mask_transits(t, f, periods[k], pg.t0[k], durations[pg.j_dur[k]], 2.0)
    assert abs(found[0] - 2.0) < 0.02 and abs(found[1] - 3.1) < 0.03

"""GPU parity: the CUDA path (through the C ABI) against the FP64 oracle on the same seeded inputs.

Run on the B200 box:  python -m pytest tests -m gpu -x -q
"""
import os

import numpy as np
import pytest

from parity_util import REL, assert_linear_parity, assert_periodic_parity, period_subset

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def cetra():
    import paper_2503_20875_b200 as c
    c.load_library()          # raises if the CUDA library is missing: no fallback
    return c


_PROBLEMS = {}


def _problem(cfg):
    from cetra_synth import make_config
    if cfg not in _PROBLEMS:
        _PROBLEMS[cfg] = make_config(cfg)
    return _PROBLEMS[cfg]


_ORACLE_LINEAR = {}


def _oracle_linear(oracle_mod, cfg):
    if cfg not in _ORACLE_LINEAR:
        p = _problem(cfg)
        _ORACLE_LINEAR[cfg] = oracle_mod.linear_search(p.times, p.flux, p.flux_err, p.durations, p.t0_start,
                                                       p.t0_stride, p.n_t0, p.template)
    return _ORACLE_LINEAR[cfg]


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _gpu_linear(torch, cetra, p, **kw):
    return cetra.cetra_linear_search(p.times, _dev(torch, p.flux), _dev(torch, p.flux_err), p.durations, p.t0_start,
                                     p.t0_stride, p.n_t0, p.template, **kw)


# ------------------------------------------------------------------------------------------ linear
@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_linear_search_full_grid(cfg, torch_cuda, cetra, oracle_mod):
    """Every (t0, duration) cell of configs 1-3 (several tiles, ragged tail, the data gap, q = 6 for cfg 3)."""
    p = _problem(cfg)
    g = _gpu_linear(torch_cuda, cetra, p)
    o = _oracle_linear(oracle_mod, cfg)
    worst = assert_linear_parity(g.depth.cpu().numpy(), g.depth_var.cpu().numpy(), g.dlogL.cpu().numpy(),
                                 o.depth, o.depth_var, o.dlogL, what=f"cfg{cfg}")
    print(f"cfg{cfg} linear worst relative errors: {worst}")


def test_linear_search_config4_full_grid(torch_cuda, cetra, oracle_mod):
    """Config 4 at full size: every one of the 50 x 256 464 cells against the oracle (SURVEY.md §8(d) "Checks":
    linear grids in full; about 5e9 FP64 template evaluations, seconds on the host cores)."""
    p = _problem(4)
    g = _gpu_linear(torch_cuda, cetra, p)
    o = _oracle_linear(oracle_mod, 4)
    assert o.depth.shape == (50, 256464)
    worst = assert_linear_parity(g.depth.cpu().numpy(), g.depth_var.cpu().numpy(), g.dlogL.cpu().numpy(),
                                 o.depth, o.depth_var, o.dlogL, what="cfg4")
    print(f"cfg4 linear worst relative errors: {worst}")
    assert np.isnan(o.depth).any()                    # the 1 d gaps leave null cells at the short durations


def test_linear_search_stats_are_the_sufficient_statistics(torch_cuda, cetra):
    """stats = (S_wmm, S_wmf): depth = S_wmf/S_wmm, var = 1/S_wmm bit for bit; zero in null cells and padding."""
    p = _problem(2)
    g = _gpu_linear(torch_cuda, cetra, p, want_stats=True)
    st = g.stats[0].cpu().numpy()
    a, b = st[..., 0], st[..., 1]
    assert np.all(st[:, p.n_t0:, :] == 0.0)
    depth, var = g.depth.cpu().numpy(), g.depth_var.cpu().numpy()
    null = np.isnan(depth)
    assert null.any(), "cfg 2 has a 1 d gap: the shortest durations must have null cells"
    assert np.all(a[:, :p.n_t0][null] == 0.0) and np.all(b[:, :p.n_t0][null] == 0.0)
    ok = ~null
    with np.errstate(divide="ignore", invalid="ignore"):
        assert np.array_equal((b[:, :p.n_t0] / a[:, :p.n_t0])[ok], depth[ok])
        assert np.array_equal((np.float32(1.0) / a[:, :p.n_t0])[ok], var[ok])


def test_linear_search_edge_geometry(torch_cuda, cetra, oracle_mod):
    """t0 grid that starts before the data and ends after it (R9 clipping), a stride of 3 samples with an
    offset start, float64 input with NaN/inf/negative-error nulls, a duration shorter than the cadence,
    a tiny n_t0 and the maximum number of durations."""
    rng = np.random.default_rng(7)
    n, c = 3001, 0.004
    times = 5.0 + np.arange(n) * c
    err = 1e-3 * (0.5 + rng.random(n))
    flux = 1.0 + rng.standard_normal(n) * err
    flux[100:140] = np.nan
    err[900:960] = np.inf
    err[1500] = -1.0
    err[1501] = 0.0
    flux[2000:2400] = np.nan                 # longer than most trial durations: null cells
    from cetra_synth import tabulate_template
    tpl = tabulate_template(257)
    cases = [
        dict(t0_start=times[0] - 50 * c, stride=c, n_t0=n + 120, durations=np.geomspace(0.5 * c, 300 * c, 9)),
        dict(t0_start=times[0] + 7 * c, stride=3 * c, n_t0=977, durations=np.geomspace(2.2 * c, 111 * c, 5)),
        dict(t0_start=times[0], stride=c, n_t0=5, durations=np.array([10 * c])),
        dict(t0_start=times[0], stride=2 * c, n_t0=1500, durations=np.geomspace(1.5 * c, 700.3 * c, 128)),
    ]
    saw_null = False
    for dt in (np.float64, np.float32):
        fl, er = flux.astype(dt), err.astype(dt)
        for cs in cases:
            g = cetra.cetra_linear_search(times, _dev(torch_cuda, fl), _dev(torch_cuda, er), cs["durations"],
                                          cs["t0_start"], cs["stride"], cs["n_t0"], tpl)
            o = oracle_mod.linear_search(times, fl, er, cs["durations"], cs["t0_start"], cs["stride"], cs["n_t0"],
                                         tpl)
            saw_null |= bool(np.isnan(o.depth).any())
            assert_linear_parity(g.depth.cpu().numpy(), g.depth_var.cpu().numpy(), g.dlogL.cpu().numpy(),
                                 o.depth, o.depth_var, o.dlogL, what=f"edge {dt.__name__} n_t0={cs['n_t0']}")
    assert saw_null, "the long gaps must produce null cells in at least one case"


def test_linear_search_window_edge_samples(torch_cuda, cetra, oracle_mod):
    """R2: D/(2c) a whole number puts a sample exactly on the first and on the last instant of every window; both
    belong to it.  Box template on a power-of-two cadence (k c and D/2 exact): the GPU must match the oracle AND
    the plain inclusive-window weighted mean computed here from the raw data (so that a shared `<` instead of
    `<=` cannot pass), for a stride of one and of two samples (the polyphase path) and for float64 input."""
    rng = np.random.default_rng(12)
    n, c = 5000, 1.0 / 256.0
    times = 3.0 + np.arange(n) * c
    err = 1e-3 * (0.5 + rng.random(n))
    flux = 1.0 + rng.standard_normal(n) * err
    flux[700:720] = np.nan
    hs = np.array([1, 2, 7, 8, 15, 16, 40])
    durations = 2.0 * (hs * c)
    box = np.ones(32, np.float32)
    good = np.isfinite(flux)
    w = np.where(good, 1.0 / err ** 2, 0.0)
    wf = np.where(good, w * (1.0 - np.where(good, flux, 1.0)), 0.0)
    cw, cwf = np.concatenate([[0.0], np.cumsum(w)]), np.concatenate([[0.0], np.cumsum(wf)])
    for dt, q in ((np.float32, 1), (np.float64, 1), (np.float32, 2)):
        fl, er = flux.astype(dt), err.astype(dt)
        n_t0 = (n - 1) // q + 1
        g = cetra.cetra_linear_search(times, _dev(torch_cuda, fl), _dev(torch_cuda, er), durations, times[0], q * c,
                                      n_t0, box)
        o = oracle_mod.linear_search(times, fl, er, durations, times[0], q * c, n_t0, box)
        assert_linear_parity(g.depth.cpu().numpy(), g.depth_var.cpu().numpy(), g.dlogL.cpu().numpy(),
                             o.depth, o.depth_var, o.dlogL, what=f"edge samples {dt.__name__} q={q}")
        if dt is np.float64:
            centre = q * np.arange(n_t0)
            var_g = g.depth_var.cpu().numpy().astype(np.float64)
            dep_g = g.depth.cpu().numpy().astype(np.float64)
            for j, h in enumerate(hs):
                lo, hi = np.maximum(centre - h, 0), np.minimum(centre + h, n - 1) + 1     # inclusive of both edges
                sw, swf = cw[hi] - cw[lo], cwf[hi] - cwf[lo]
                ok = sw > 0
                assert np.array_equal(np.isnan(var_g[j]), ~ok)
                assert np.allclose(var_g[j][ok], 1.0 / sw[ok], rtol=3e-5)
                assert np.allclose(dep_g[j][ok], swf[ok] / sw[ok], rtol=0, atol=3e-5 * np.sqrt(1.0 / sw[ok]).max())
                # dropping one edge sample of the 2h+1 would change var by 1/(2h+1) >= 1.2 %: far above 3e-5


# ---------------------------------------------------------------------------------------- periodic
def _oracle_periodic_inputs(oracle_mod, cfg):
    """Oracle linear grids rounded to the float32 the GPU entry point takes, promoted back to float64."""
    o = _oracle_linear(oracle_mod, cfg)
    d32, v32, l32 = (a.astype(np.float32) for a in (o.depth, o.depth_var, o.dlogL))
    grids = oracle_mod.LinearGrids(d32.astype(np.float64), v32.astype(np.float64), l32.astype(np.float64))
    return (d32, v32, l32), grids


def _check_periodic(torch, cetra, oracle_mod, p, grids32, grids64, sel, what, must_match=()):
    periods = p.periods[sel]
    peaks = cetra.cetra_periodic_search(*(_dev(torch, a) for a in grids32), p.t0_start, p.t0_stride, p.durations,
                                        periods)
    pk = cetra.peaks_to_numpy(peaks)[0]
    orc = oracle_mod.periodic_search(grids64, p.t0_start, p.t0_stride, p.durations, periods)

    def cell(k, j, ph):
        return oracle_mod.periodic_cell(grids64, p.t0_stride, periods[k], j, ph)

    res = assert_periodic_parity(pk, orc, cell, what=what, must_match=must_match)
    t0_ref = p.t0_start + pk["i_t0"].astype(np.float64) * p.t0_stride
    ok = pk["i_t0"] >= 0
    assert np.allclose(pk["t0"][ok], t0_ref[ok], rtol=2e-7, atol=0)
    return pk, orc, res


def test_periodic_search_config1_all_periods(torch_cuda, cetra, oracle_mod):
    p = _problem(1)
    g32, g64 = _oracle_periodic_inputs(oracle_mod, 1)
    pk, orc, res = _check_periodic(torch_cuda, cetra, oracle_mod, p, g32, g64, np.arange(p.periods.shape[0]), "cfg1")
    print("cfg1 periodic:", res)


@pytest.mark.parametrize("cfg,n_random", [(2, 700), (3, 500)])
def test_periodic_search_sampled_periods(cfg, n_random, torch_cuda, cetra, oracle_mod):
    """Configs 2-3: a seeded subset of the 20 000 trial periods plus windows around the injected period and
    its aliases (the oracle needs ~1e6 gathers per period).  The full-K GPU run must reproduce the subset
    run bit for bit (periods are independent), which extends the check to the bench launch configuration."""
    p = _problem(cfg)
    g32, g64 = _oracle_periodic_inputs(oracle_mod, cfg)
    inj = [i["period"] for i in p.injections]
    sel = period_subset(p.periods, inj, n_random, seed=100 + cfg)
    k_inj = int(np.argmin(np.abs(p.periods - inj[0])))
    must = [int(np.nonzero(sel == k_inj)[0][0])]
    pk, orc, res = _check_periodic(torch_cuda, cetra, oracle_mod, p, g32, g64, sel, f"cfg{cfg}", must_match=must)
    print(f"cfg{cfg} periodic:", res)
    # injected signal: the best period of the subset is the injected one, with identical indices
    kb_g, kb_o = int(np.nanargmax(pk["lr"])), int(np.nanargmax(orc.lr))
    assert kb_g == kb_o
    assert abs(p.periods[sel][kb_g] - inj[0]) <= 0.01 * inj[0]
    assert pk["j_dur"][kb_g] == orc.j_dur[kb_o] and pk["i_t0"][kb_g] == orc.i_t0[kb_o]
    full = cetra.peaks_to_numpy(cetra.cetra_periodic_search(*(_dev(torch_cuda, a) for a in g32), p.t0_start,
                                                             p.t0_stride, p.durations, p.periods))[0]
    assert np.array_equal(full[sel].view(np.uint8), pk.view(np.uint8))
    # cfg 2 has exactly one excluded (period, duration) pair: D = 12 h = P_min (R12)
    if cfg == 2:
        assert np.all(full["j_dur"] < p.durations.shape[0])


@pytest.mark.parametrize("cfg,kind", [(1, "random"), (1, "constant"), (2, "random")])
def test_periodic_search_honours_a_callers_likelihood_grid(cfg, kind, torch_cuda, cetra, oracle_mod):
    """Eq. 4 sums the per-transit likelihood ratios LR_e the caller passes.  For the linear
    search's own grid LR_e = 1/2 depth^2/var and two statistics suffice; a grid that differs (here: offset per
    cell, as when full log-likelihoods are passed) must give the literal sum, as the oracle does
    (R20): the winners change, and GPU and oracle still agree.  dlogL = None means the identity."""
    p = _problem(cfg)
    g32, _ = _oracle_periodic_inputs(oracle_mod, cfg)
    d32, v32, l32 = g32
    rng = np.random.default_rng(77 + cfg)
    off = (rng.uniform(0.0, 2.0, size=l32.shape) if kind == "random" else np.full(l32.shape, 1.0)).astype(np.float32)
    l_off = (l32 + off).astype(np.float32)
    l_off[np.isnan(l32)] = np.nan
    import oracle as oracle_pkg
    g64 = oracle_pkg.LinearGrids(d32.astype(np.float64), v32.astype(np.float64), l_off.astype(np.float64))
    sel = np.arange(p.periods.shape[0]) if cfg == 1 else period_subset(p.periods, [], 60, seed=5)
    periods = p.periods[sel]
    dev = [_dev(torch_cuda, a) for a in (d32, v32, l_off)]
    pk = cetra.peaks_to_numpy(cetra.cetra_periodic_search(*dev, p.t0_start, p.t0_stride, p.durations, periods))[0]
    orc = oracle_mod.periodic_search(g64, p.t0_start, p.t0_stride, p.durations, periods)

    def cell(k, j, ph):
        return oracle_mod.periodic_cell(g64, p.t0_stride, periods[k], j, ph)

    res = assert_periodic_parity(pk, orc, cell, what=f"cfg{cfg} caller LR grid ({kind})")
    print("caller LR grid:", cfg, kind, res)
    # the two-statistic search (dlogL = None, or the identity grid) picks other cells on this input
    plain = cetra.peaks_to_numpy(cetra.cetra_periodic_search(dev[0], dev[1], None, p.t0_start, p.t0_stride,
                                                             p.durations, periods))[0]
    ident = cetra.peaks_to_numpy(cetra.cetra_periodic_search(dev[0], dev[1], _dev(torch_cuda, l32), p.t0_start,
                                                             p.t0_stride, p.durations, periods))[0]
    assert np.array_equal(plain.view(np.uint8), ident.view(np.uint8))
    assert (plain["i_t0"] != pk["i_t0"]).any() and np.all(pk["lr"] > plain["lr"])


def test_periodic_search_duration_ranges_and_empty_periods(torch_cuda, cetra, oracle_mod):
    """Per-period duration ranges, periods shorter than every duration (no candidate -> NaN
    record, indices -1) and periods longer than the baseline (a single epoch)."""
    p = _problem(1)
    g32, g64 = _oracle_periodic_inputs(oracle_mod, 1)
    periods = np.concatenate([p.periods[::7], [0.02, 0.0201, 1.2, 3.0, 50.0]])
    K, J = periods.shape[0], p.durations.shape[0]
    rng = np.random.default_rng(9)
    lo = rng.integers(0, J, size=K).astype(np.int32)
    hi = np.minimum(J, lo + rng.integers(0, 4, size=K)).astype(np.int32)      # some ranges are empty
    peaks = cetra.cetra_periodic_search(*(_dev(torch_cuda, a) for a in g32), p.t0_start, p.t0_stride, p.durations,
                                        periods, dur_lo=lo, dur_hi=hi)
    pk = cetra.peaks_to_numpy(peaks)[0]
    orc = oracle_mod.periodic_search(g64, p.t0_start, p.t0_stride, p.durations, periods, lo, hi)
    assert np.isnan(orc.lr).any() and (~np.isnan(orc.lr)).any()

    def cell(k, j, ph):
        return oracle_mod.periodic_cell(g64, p.t0_stride, periods[k], j, ph)

    assert_periodic_parity(pk, orc, cell, what="ranges")
    ok = pk["j_dur"] >= 0
    assert np.all(pk["j_dur"][ok] >= lo[ok]) and np.all(pk["j_dur"][ok] < hi[ok])


@pytest.mark.parametrize("order", ["descending", "shuffled", "duplicates", "single", "far_apart"])
def test_periodic_search_any_period_order(order, torch_cuda, cetra, oracle_mod):
    """The fold kernel pairs neighbouring entries of the period array: the records must not depend on how the
    array is ordered, on an odd count (ragged last pair), on repeated periods, or on pairs whose offsets are too
    far apart to share a window."""
    p = _problem(2)
    g32, g64 = _oracle_periodic_inputs(oracle_mod, 2)
    rng = np.random.default_rng(77)
    base = p.periods[rng.choice(p.periods.shape[0], 41, replace=False)]
    if order == "descending":
        periods = np.sort(base)[::-1].copy()
    elif order == "shuffled":
        periods = base
    elif order == "duplicates":
        periods = np.repeat(np.sort(base)[:14], 3)[:41]
    elif order == "single":
        periods = base[:1]
    else:
        periods = np.array([0.5001, 13.5, 0.7, 9.1, 1.0, 12.0, 0.6])        # every pair spreads over > 7 cells
    peaks = cetra.cetra_periodic_search(*(_dev(torch_cuda, a) for a in g32), p.t0_start, p.t0_stride, p.durations,
                                        periods)
    pk = cetra.peaks_to_numpy(peaks)[0]
    orc = oracle_mod.periodic_search(g64, p.t0_start, p.t0_stride, p.durations, periods)

    def cell(k, j, ph):
        return oracle_mod.periodic_cell(g64, p.t0_stride, periods[k], j, ph)

    assert_periodic_parity(pk, orc, cell, what=f"period order {order}")
    if order == "duplicates":
        for a in range(0, 39, 3):            # equal periods give equal records
            assert pk[a] == pk[a + 1] == pk[a + 2]


# ------------------------------------------------------------------------- whole path, end to end
def _gpu_pipeline(torch, cetra, p, periods):
    """Linear search -> sufficient statistics -> periodic search, all on the device (the bench's path)."""
    flux, err = _dev(torch, p.flux), _dev(torch, p.flux_err)
    if flux.dim() == 1:
        flux, err = flux[None], err[None]
    peaks = cetra.cetra_search_batched(p.times, flux, err, p.durations, p.t0_start, p.t0_stride, p.n_t0, p.template,
                                       periods)
    return cetra.peaks_to_numpy(peaks)


@pytest.mark.parametrize("cfg,n_random", [(1, 200), (2, 300), (3, 200)])
def test_whole_path_against_oracle(cfg, n_random, torch_cuda, cetra, oracle_mod):
    """FP32 linear search feeding the FP32 periodic search vs the FP64 oracle end to end; the injected
    signal must come out at the identical (period, t0, duration) indices (north_star)."""
    p = _problem(cfg)
    inj = [i["period"] for i in p.injections if i["period"] is not None]
    sel = period_subset(p.periods, inj, n_random, seed=200 + cfg)
    periods = p.periods[sel]
    pk = _gpu_pipeline(torch_cuda, cetra, p, periods)[0]
    o = _oracle_linear(oracle_mod, cfg)
    orc = oracle_mod.periodic_search(o, p.t0_start, p.t0_stride, p.durations, periods)

    def cell(k, j, ph):
        return oracle_mod.periodic_cell(o, p.t0_stride, periods[k], j, ph)

    must = []
    if inj:
        k_inj = int(np.argmin(np.abs(p.periods - inj[0])))
        must = [int(np.nonzero(sel == k_inj)[0][0])]
    res = assert_periodic_parity(pk, orc, cell, what=f"cfg{cfg} end-to-end", must_match=must)
    print(f"cfg{cfg} end-to-end:", res)
    kb_g, kb_o = int(np.nanargmax(pk["lr"])), int(np.nanargmax(orc.lr))
    assert kb_g == kb_o and pk["j_dur"][kb_g] == orc.j_dur[kb_o] and pk["i_t0"][kb_g] == orc.i_t0[kb_o]
    if inj:
        i0 = p.injections[0]
        assert abs(periods[kb_g] - i0["period"]) <= 0.01 * i0["period"]
        # recovered epoch and duration are the injected ones to within a grid step / one duration bin
        t0_rec = p.t0_start + pk["i_t0"][kb_g] * p.t0_stride
        phase_err = (t0_rec - i0["t0"] + 0.5 * i0["period"]) % i0["period"] - 0.5 * i0["period"]
        assert abs(phase_err) <= 0.1 * i0["duration"]
    else:
        # cfg 1: a single transit; the recovered first-epoch cell is the injected epoch modulo the best period
        i0 = p.injections[0]
        t0_rec = p.t0_start + pk["i_t0"][kb_g] * p.t0_stride
        pb = periods[kb_g]
        phase_err = (t0_rec - i0["t0"] + 0.5 * pb) % pb - 0.5 * pb
        assert abs(phase_err) <= 0.1 * i0["duration"]


def test_config4_whole_path_sampled(torch_cuda, cetra, oracle_mod):
    """Config 4 (256 464 cells per row: rows that do not fit in shared memory) on the subset SURVEY.md §8(d) names:
    a seeded 2 000 of its 200 000 periods plus +-200 trials around each injected period and its x1/2, x2 aliases;
    oracle linear grids in full.  The trial period nearest to each injected planet must come out at the identical
    (t0, duration) cell, and so must the best period within +-1 % of each planet."""
    p = _problem(4)
    inj = [i["period"] for i in p.injections]
    sel = period_subset(p.periods, inj, 2000, seed=4, half_width=200)
    periods = p.periods[sel]
    assert periods.shape[0] > 3500
    pk = _gpu_pipeline(torch_cuda, cetra, p, periods)[0]
    o = _oracle_linear(oracle_mod, 4)
    orc = oracle_mod.periodic_search(o, p.t0_start, p.t0_stride, p.durations, periods)

    def cell(k, j, ph):
        return oracle_mod.periodic_cell(o, p.t0_stride, periods[k], j, ph)

    must = [int(np.argmin(np.abs(periods - pi))) for pi in inj]
    res = assert_periodic_parity(pk, orc, cell, what="cfg4 end-to-end", must_match=must)
    print("cfg4 end-to-end:", res, "periods", periods.shape[0])
    # argmax within +-1 % of each injected period is the same cell on both sides
    for i0 in p.injections:
        near = np.abs(periods - i0["period"]) <= 0.01 * i0["period"]
        kg = int(np.nanargmax(np.where(near, pk["lr"], -np.inf)))
        ko = int(np.nanargmax(np.where(near, orc.lr, -np.inf)))
        assert kg == ko and pk["j_dur"][kg] == orc.j_dur[ko] and pk["i_t0"][kg] == orc.i_t0[ko]
    # the global maximum of the subset is the shorter-period planet (more transits) on both sides
    assert int(np.nanargmax(pk["lr"])) == int(np.nanargmax(orc.lr))


def test_config2_on_the_papers_default_t0_grid(torch_cuda, cetra, oracle_mod):
    """The TESS-like sector searched as the paper does by default (t0 stride = 1 % of the shortest
    duration = 18 s = 3/20 of the cadence, I = 131 514 cells, rows of 1 MB): residue-class linear kernel against the
    oracle on every cell, then the streamed fold on a seeded subset of the 20 000 periods plus windows around the
    injected period and its aliases; the injected planet must come out at the identical (period, t0, duration)."""
    p = _problem(2)
    stride = 0.01 * p.durations[0]
    t0_start = p.times[0]
    n_t0 = int((p.times[-1] - p.times[0]) / stride) + 1
    assert n_t0 == 131514
    o = oracle_mod.linear_search(p.times, p.flux, p.flux_err, p.durations, t0_start, stride, n_t0, p.template)
    flux, err = _dev(torch_cuda, p.flux), _dev(torch_cuda, p.flux_err)
    lin = cetra.cetra_linear_search(p.times, flux, err, p.durations, t0_start, stride, n_t0, p.template, want_stats=True)
    worst = assert_linear_parity(lin.depth.cpu().numpy(), lin.depth_var.cpu().numpy(), lin.dlogL.cpu().numpy(),
                                 o.depth, o.depth_var, o.dlogL, what="config 2, default t0 grid")
    inj = [i["period"] for i in p.injections]
    sel = period_subset(p.periods, inj, 60, seed=22, half_width=15)
    periods = p.periods[sel]
    pk = cetra.peaks_to_numpy(cetra.cetra_periodic_search_stats(lin.stats, n_t0, t0_start, stride, p.durations,
                                                                periods))[0]
    orc = oracle_mod.periodic_search(o, t0_start, stride, p.durations, periods)
    must = [int(np.argmin(np.abs(periods - inj[0])))]
    res = assert_periodic_parity(pk, orc, lambda k, j, ph: oracle_mod.periodic_cell(o, stride, periods[k], j, ph),
                                 what="config 2, default t0 grid, streamed fold", must_match=must)
    print("default t0 grid:", worst, res, "periods", periods.shape[0])
    kb = int(np.nanargmax(pk["lr"]))
    assert kb == int(np.nanargmax(orc.lr)) and abs(periods[kb] - inj[0]) <= 0.01 * inj[0]
    # the batched entry point runs the same two kernels: identical records
    pb = cetra.peaks_to_numpy(cetra.cetra_search_batched(p.times, flux[None], err[None], p.durations, t0_start, stride,
                                                         n_t0, p.template, periods))[0]
    assert np.array_equal(pb.view(np.uint8), pk.view(np.uint8))


# ------------------------------------------------------------------------------------------ batched
def test_batched_equals_single_and_host_variant(torch_cuda, cetra, oracle_mod):
    """Survey batch (config 5 recipe, 7 light curves, chunks of 3 -> ragged last chunk): the batched call,
    the host-buffer call and one-at-a-time calls give bit-identical records; two curves are checked
    against the oracle."""
    from cetra_synth import make_survey_batch
    p = make_survey_batch(n_lc=7, n_periods=600)
    flux, err = _dev(torch_cuda, p.flux), _dev(torch_cuda, p.flux_err)
    args = (p.durations, p.t0_start, p.t0_stride, p.n_t0, p.template, p.periods)
    pk = cetra.peaks_to_numpy(cetra.cetra_search_batched(p.times, flux, err, *args, lc_chunk=3))
    pk_all = cetra.peaks_to_numpy(cetra.cetra_search_batched(p.times, flux, err, *args))
    assert np.array_equal(pk.view(np.uint8), pk_all.view(np.uint8))
    for b in (0, 3, 6):
        one = cetra.peaks_to_numpy(cetra.cetra_search_batched(p.times, flux[b:b + 1], err[b:b + 1], *args))
        assert np.array_equal(one[0].view(np.uint8), pk[b].view(np.uint8))
    host = cetra.cetra_search_batched_host(p.times, torch_cuda.from_numpy(p.flux).pin_memory(),
                                           torch_cuda.from_numpy(p.flux_err).pin_memory(), *args, lc_chunk=3)
    assert np.array_equal(host.view(np.uint8), pk.view(np.uint8))
    for b in (1, 6):
        o = oracle_mod.linear_search(p.times, p.flux[b], p.flux_err[b], p.durations, p.t0_start, p.t0_stride,
                                     p.n_t0, p.template)
        orc = oracle_mod.periodic_search(o, p.t0_start, p.t0_stride, p.durations, p.periods)

        def cell(k, j, ph):
            return oracle_mod.periodic_cell(o, p.t0_stride, p.periods[k], j, ph)

        assert_periodic_parity(pk[b], orc, cell, what=f"batch lc {b}")


def test_large_time_origin(torch_cuda, cetra, oracle_mod):
    """Times as BJD - 2 457 000 (origin ~ 3e3 d) and as full BJD: the sample times are then only regular to the FP64
    rounding of the origin, the float32 `t0` of a record resolves 20 s / 0.25 d, and i_t0 stays exact (cetra.h):
    the records match the oracle's on the shifted times, and the indices those of the search with origin 0."""
    p = _problem(1)
    periods = p.periods[::5]
    flux, err = _dev(torch_cuda, p.flux), _dev(torch_cuda, p.flux_err)
    base = cetra.peaks_to_numpy(cetra.cetra_search_batched(p.times, flux[None], err[None], p.durations, p.t0_start,
                                                           p.t0_stride, p.n_t0, p.template, periods))[0]
    for origin in (3456.0, 2458849.5):
        times = origin + np.arange(p.n) * p.cadence
        c = (times[-1] - times[0]) / (p.n - 1)                   # the cadence the library derives from these times
        pk = cetra.peaks_to_numpy(cetra.cetra_search_batched(times, flux[None], err[None], p.durations, times[0], c,
                                                             p.n_t0, p.template, periods))[0]
        o = oracle_mod.linear_search(times, p.flux, p.flux_err, p.durations, times[0], c, p.n_t0, p.template)
        orc = oracle_mod.periodic_search(o, times[0], c, p.durations, periods)
        assert_periodic_parity(pk, orc, lambda k, j, ph: oracle_mod.periodic_cell(o, c, periods[k], j, ph),
                               what=f"origin {origin}")
        same = (pk["i_t0"] == base["i_t0"]) & (pk["j_dur"] == base["j_dur"])       # rounding of the shifted times may
        assert same.mean() >= 0.9                                                    # move a near-tie, not more
        exact = times[0] + pk["i_t0"].astype(np.float64) * c
        assert np.array_equal(pk["t0"], exact.astype(np.float32))                      # float32 of the exact time ...
        assert np.abs(pk["t0"].astype(np.float64) - exact).max() > 1e-5               # ... which is coarser than a sample


def test_search_on_a_side_stream(torch_cuda, cetra):
    """Every wrapper takes `stream=`: workspace, outputs and input copies are then made on that stream (binding
    _on_stream).  A search enqueued on a side stream, behind a long kernel on that stream, with non-contiguous inputs,
    gives the records of the same search on the default stream bit for bit."""
    from cetra_synth import make_survey_batch
    torch = torch_cuda
    p = make_survey_batch(n_lc=6, n_periods=400)
    wide_f = torch.from_numpy(np.ascontiguousarray(np.repeat(p.flux, 2, axis=1))).cuda()
    wide_e = torch.from_numpy(np.ascontiguousarray(np.repeat(p.flux_err, 2, axis=1))).cuda()
    flux, err = wide_f[:, ::2], wide_e[:, ::2]                   # strided views: the wrapper must copy them
    assert not flux.is_contiguous()
    args = (p.times, flux, err, p.durations, p.t0_start, p.t0_stride, p.n_t0, p.template, p.periods)
    ref = cetra.peaks_to_numpy(cetra.cetra_search_batched(*args))
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    busy = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    with torch.cuda.stream(side):
        for _ in range(20):
            busy.add_(1)                                         # the side stream is busy when the search is enqueued
    got = cetra.cetra_search_batched(*args, stream=side)
    churn = [torch.full((1 << 20,), 7, dtype=torch.int32, device="cuda") for _ in range(32)]   # default-stream allocations
    side.synchronize()
    torch.cuda.synchronize()
    assert np.array_equal(cetra.peaks_to_numpy(got).view(np.uint8), ref.view(np.uint8))
    lin = cetra.cetra_linear_search(*args[:8], want_stats=True, stream=side)
    side.synchronize()
    lin0 = cetra.cetra_linear_search(*args[:8], want_stats=True)
    torch.cuda.synchronize()
    assert torch.equal(lin.stats, lin0.stats) and torch.equal(torch.nan_to_num(lin.depth), torch.nan_to_num(lin0.depth))
    del churn


def test_template_sequence_equals_one_search_per_template(torch_cuda, cetra, oracle_mod):
    """a sequence of impact parameters.  Every template's records are bit-identical to a search
    with that template alone, and the grazing template is checked against the oracle."""
    from cetra_synth import make_survey_batch, tabulate_template
    p = make_survey_batch(n_lc=3, n_periods=300)
    flux, err = _dev(torch_cuda, p.flux), _dev(torch_cuda, p.flux_err)
    tpls = np.stack([tabulate_template(1024, b=b) for b in (0.32, 0.93, 0.99)])      # the paper's three models
    assert not np.allclose(tpls[0], tpls[2])
    args = (p.durations, p.t0_start, p.t0_stride, p.n_t0)
    pk = cetra.cetra_search_batched_templates(p.times, flux, err, *args, tpls, p.periods)
    assert tuple(pk.shape) == (3, 3, 300, 8)
    pk = cetra.peaks_to_numpy(pk.reshape(9, 300, 8)).reshape(3, 3, 300)
    for t in range(3):
        one = cetra.peaks_to_numpy(cetra.cetra_search_batched(p.times, flux, err, *args, tpls[t], p.periods))
        assert np.array_equal(one.view(np.uint8), pk[t].view(np.uint8))
    o = oracle_mod.linear_search(p.times, p.flux[1], p.flux_err[1], *args, tpls[2])
    orc = oracle_mod.periodic_search(o, p.t0_start, p.t0_stride, p.durations, p.periods)
    assert_periodic_parity(pk[2][1], orc, lambda k, j, ph: oracle_mod.periodic_cell(o, p.t0_stride, p.periods[k], j, ph),
                           what="template b = 0.99")
    # chunks of two light curves (ragged last chunk), and the paper's default off-grid stride (one linear launch
    # over the templates' class tap tables): still the records of one search per template
    pk2 = cetra.peaks_to_numpy(cetra.cetra_search_batched_templates(p.times, flux, err, *args, tpls, p.periods,
                                                                    lc_chunk=2).reshape(9, 300, 8)).reshape(3, 3, 300)
    assert np.array_equal(pk2.view(np.uint8), pk.view(np.uint8))
    og = (p.durations, p.times[0], 0.01 * p.durations[0], 30000)
    pk3 = cetra.peaks_to_numpy(cetra.cetra_search_batched_templates(p.times, flux, err, *og, tpls, p.periods[:40],
                                                                    lc_chunk=2).reshape(9, 40, 8)).reshape(3, 3, 40)
    for t in range(3):
        one = cetra.peaks_to_numpy(cetra.cetra_search_batched(p.times, flux, err, *og, tpls[t], p.periods[:40]))
        assert np.array_equal(one.view(np.uint8), pk3[t].view(np.uint8))


def test_bench_configuration_sampled_against_oracle(torch_cuda, cetra, oracle_mod):
    """The launch configuration bench.py times: 64 survey curves of BASELINE configs[1] in one chunk, all 20 000
    periods.  Properties that hold at any size are checked on all 1.28 million records, and all 64 curves of the
    chunk are compared with the oracle (a seeded 64-curve subsample): 8 of them (injected and
    signal-free ones) on ALL 20 000 periods, the other 56 each on a seeded 1 500-period subset plus the windows around
    its injected period and the x1/2 and x2 aliases; the period nearest to an injected planet at identical indices."""
    from cetra_synth import make_survey_batch
    p = make_survey_batch(n_lc=64, lc_range=(0, 64))
    flux, err = _dev(torch_cuda, p.flux), _dev(torch_cuda, p.flux_err)
    pk = cetra.peaks_to_numpy(cetra.cetra_search_batched(p.times, flux, err, p.durations, p.t0_start, p.t0_stride,
                                                         p.n_t0, p.template, p.periods))
    K = p.periods.shape[0]
    assert pk.shape == (64, K)
    # properties of every record (R10, R13)
    ok = pk["i_t0"] >= 0
    assert ok.all()                                          # every period has a candidate in these curves
    assert np.all(pk["lr"] >= 0) and np.all(pk["depth_var"] > 0) and np.all(pk["n_transits"] >= 1)
    assert np.all(p.durations[pk["j_dur"]] < p.periods[None, :])
    assert np.all(pk["i_t0"] < np.ceil(p.periods / p.t0_stride)[None, :])
    n_epochs_max = np.floor((p.n_t0 - 1) / (p.periods / p.t0_stride)) + 1
    assert np.all(pk["n_transits"] <= n_epochs_max[None, :] + 1)
    assert np.allclose(pk["lr"], 0.5 * pk["depth"].astype(np.float64) ** 2 / pk["depth_var"], rtol=1e-5)
    rng = np.random.default_rng(64)
    injected = [b for b, i in enumerate(p.injections) if i["period"] is not None]
    flat = [b for b in range(64) if b not in injected]
    curves = sorted(rng.choice(injected, 5, replace=False).tolist() + rng.choice(flat, 3, replace=False).tolist())
    for b in curves:
        o = oracle_mod.linear_search(p.times, p.flux[b], p.flux_err[b], p.durations, p.t0_start, p.t0_stride,
                                     p.n_t0, p.template)
        orc = oracle_mod.periodic_search(o, p.t0_start, p.t0_stride, p.durations, p.periods)

        def cell(k, j, ph):
            return oracle_mod.periodic_cell(o, p.t0_stride, p.periods[k], j, ph)

        must = []
        if p.injections[b]["period"] is not None:
            must = [int(np.argmin(np.abs(p.periods - p.injections[b]["period"])))]
        res = assert_periodic_parity(pk[b], orc, cell, what=f"bench configuration, curve {b}", must_match=must)
        print("bench configuration curve", b, res)
        assert int(np.nanargmax(pk[b]["lr"])) == int(np.nanargmax(orc.lr))
    # ... and the other 56 curves ("a seeded 64-curve subsample"), each on its own seeded 1 500-period
    # subset plus 121-period windows around its injected period and that period's x1/2 and x2 aliases, so that all 64
    # curves of the chunk bench.py launches are compared with the oracle
    worst = 0.0
    for b in range(64):
        if b in curves:
            continue
        inj = p.injections[b]["period"]
        idx = period_subset(p.periods, [inj] if inj is not None else [], 1500, seed=6400 + b)
        o = oracle_mod.linear_search(p.times, p.flux[b], p.flux_err[b], p.durations, p.t0_start, p.t0_stride,
                                     p.n_t0, p.template)
        orc = oracle_mod.periodic_search(o, p.t0_start, p.t0_stride, p.durations, p.periods[idx])
        must = [int(np.argmin(np.abs(p.periods[idx] - inj)))] if inj is not None else []
        res = assert_periodic_parity(pk[b][idx], orc,
                                     lambda k, j, ph: oracle_mod.periodic_cell(o, p.t0_stride, p.periods[idx[k]], j, ph),
                                     what=f"bench configuration, curve {b} on {len(idx)} periods", must_match=must)
        worst = max(worst, res["lr"])
    print("bench configuration: 56 more curves on period subsets, worst LR error", worst)


def test_survey_recovery_fraction(torch_cuda, cetra):
    """BASELINE configs[4] "reports throughput and injection-recovery fraction": the first 512 curves of the
    10 000-curve survey recipe; a planet is recovered when the best period is within 1 % of the injected period,
    of half of it or of twice it.  Injected SNR is 6-12, so nearly all must be recovered."""
    from cetra_synth import make_survey_batch
    p = make_survey_batch(n_lc=10000, lc_range=(0, 512))
    flux, err = _dev(torch_cuda, p.flux), _dev(torch_cuda, p.flux_err)
    pk = cetra.peaks_to_numpy(cetra.cetra_search_batched(p.times, flux, err, p.durations, p.t0_start, p.t0_stride,
                                                         p.n_t0, p.template, p.periods))
    best = p.periods[np.nanargmax(pk["lr"], axis=1)]
    n_inj = n_rec = 0
    for b, inj in enumerate(p.injections):
        if inj["period"] is None:
            continue
        n_inj += 1
        n_rec += int(any(abs(best[b] - m * inj["period"]) <= 0.01 * m * inj["period"] for m in (0.5, 1.0, 2.0)))
    frac = n_rec / n_inj
    print(f"survey slice: {n_rec} of {n_inj} injected planets recovered ({100 * frac:.1f} %)")
    assert 200 <= n_inj <= 312 and frac >= 0.95


# ------------------------------------------------------------------------------- off-grid t0 grids (R25)
@pytest.mark.parametrize("cfg,frac", [(1, 0.01), (2, 0.01), (3, 0.037)])
def test_linear_search_off_grid_t0(cfg, frac, torch_cuda, cetra, oracle_mod):
    """the default t0 stride is 1 % of the shortest duration, which is not a multiple of the cadence."""
    p = _problem(cfg)
    stride = frac * p.durations[0]
    t0_start = p.times[0] - 0.31 * p.durations[-1]                  # starts before the data: clipped windows
    n_t0 = {1: 7000, 2: 30000, 3: 6000}[cfg]
    if cfg == 3:
        t0_start = p.times[0] + 12.9                                 # runs into the null gap at 13.2 d
    o = oracle_mod.linear_search(p.times, p.flux, p.flux_err, p.durations, t0_start, stride, n_t0, p.template)
    flux, err = _dev(torch_cuda, p.flux), _dev(torch_cuda, p.flux_err)
    r = cetra.cetra_linear_search(p.times, flux, err, p.durations, t0_start, stride, n_t0, p.template, want_stats=True)
    torch_cuda.cuda.synchronize()
    worst = assert_linear_parity(r.depth.cpu().numpy(), r.depth_var.cpu().numpy(), r.dlogL.cpu().numpy(),
                                 o.depth, o.depth_var, o.dlogL, what=f"config {cfg} off-grid")
    print("off-grid worst", cfg, worst)
    assert np.isnan(o.depth).any() and (~np.isnan(o.depth)).sum() > 0.5 * o.depth.size
    # the stats rows hold the same sufficient statistics, zero in null cells and in the padding
    st = r.stats[0].cpu().numpy()
    a, b = st[:, :n_t0, 0], st[:, :n_t0, 1]
    nul = np.isnan(o.depth)
    assert np.all(a[nul] == 0) and np.all(b[nul] == 0) and np.all(st[:, n_t0:] == 0)
    assert np.allclose(a[~nul], 1.0 / o.depth_var[~nul], rtol=1e-5)


def test_off_grid_default_stride_takes_the_exact_fallback(torch_cuda, cetra, oracle_mod):
    """The paper's default t0 grid on 2-min data (stride 18 s = 3/20 of the cadence) starting ON a sample:
    every 20th cell sits exactly on a sample, where the window centre lands exactly on a rounding boundary of the
    nearest-neighbour index (x = 1/2 -> position 512.0 in a 1 024-sample template).  The class tap tables withhold
    such taps and the kernel evaluates them per cell with the definition's FP64 sequence (R25): the
    counter of exact evaluations must be > 0 and every cell must agree with the oracle."""
    p = _problem(2)
    stride = 0.01 * p.durations[0]
    t0_start, n_t0 = p.times[0], 40000
    o = oracle_mod.linear_search(p.times, p.flux, p.flux_err, p.durations, t0_start, stride, n_t0, p.template)
    flux, err = _dev(torch_cuda, p.flux), _dev(torch_cuda, p.flux_err)
    cetra.cetra_exact_eval_count(reset=True)
    r = cetra.cetra_linear_search(p.times, flux, err, p.durations, t0_start, stride, n_t0, p.template)
    n_exact = cetra.cetra_exact_eval_count()
    worst = assert_linear_parity(r.depth.cpu().numpy(), r.depth_var.cpu().numpy(), r.dlogL.cpu().numpy(),
                                 o.depth, o.depth_var, o.dlogL, what="config 2 default t0 grid")
    print("default-grid worst", worst, "exact evaluations", n_exact)
    assert n_exact > 0
    # a stride that is not a small rational multiple of the cadence takes the per-cell kernel, same bar
    # (stepped fixed-point positions; cell 0 sits on a sample, so its centre position is exactly on an index step and
    # that block must take the exact sequence too)
    stride2 = stride * (1.0 + 1.0 / 977.0)
    o2 = oracle_mod.linear_search(p.times, p.flux, p.flux_err, p.durations, t0_start, stride2, 12000, p.template)
    cetra.cetra_exact_eval_count(reset=True)
    r2 = cetra.cetra_linear_search(p.times, flux, err, p.durations, t0_start, stride2, 12000, p.template)
    n_exact2 = cetra.cetra_exact_eval_count()
    assert_linear_parity(r2.depth.cpu().numpy(), r2.depth_var.cpu().numpy(), r2.dlogL.cpu().numpy(),
                         o2.depth, o2.depth_var, o2.dlogL, what="config 2 irrational stride")
    n_evals2 = sum(12000 * (2 * int(d / (2 * (p.times[1] - p.times[0]))) + 1) for d in p.durations)
    print("irrational stride: exact evaluations", n_exact2, "of about", n_evals2)
    assert 0 < n_exact2 < 0.01 * n_evals2
    # a whole-sample stride whose START is off the sample grid: a single residue class with a sub-sample offset
    c = p.times[1] - p.times[0]
    for start in (p.times[0] + 0.3 * c, p.times[0] - 100.5 * c):      # the second puts every cell half-way between samples
        o3 = oracle_mod.linear_search(p.times, p.flux, p.flux_err, p.durations, start, 2 * c, 9000, p.template)
        r3 = cetra.cetra_linear_search(p.times, flux, err, p.durations, start, 2 * c, 9000, p.template)
        assert_linear_parity(r3.depth.cpu().numpy(), r3.depth_var.cpu().numpy(), r3.dlogL.cpu().numpy(),
                             o3.depth, o3.depth_var, o3.dlogL, what="config 2 whole-sample stride, off-grid start")


def test_whole_path_off_grid_t0(torch_cuda, cetra, oracle_mod):
    """Linear + periodic search on the paper's default t0 grid through the batched entry point."""
    p = _problem(1)
    stride = 0.01 * p.durations[0]
    t0_start = p.times[0] - 0.5 * p.durations[-1]                    # PAPER.md:61 padding expressed as a grid start
    n_t0 = int((p.times[-1] - t0_start + 0.5 * p.durations[-1]) / stride) + 1
    periods = p.periods[::4]
    o = oracle_mod.linear_search(p.times, p.flux, p.flux_err, p.durations, t0_start, stride, n_t0, p.template)
    flux, err = _dev(torch_cuda, p.flux), _dev(torch_cuda, p.flux_err)
    lin = cetra.cetra_linear_search(p.times, flux, err, p.durations, t0_start, stride, n_t0, p.template)
    peaks = cetra.peaks_to_numpy(cetra.cetra_search_batched(p.times, flux[None], err[None], p.durations, t0_start,
                                                            stride, n_t0, p.template, periods))[0]
    torch_cuda.cuda.synchronize()
    # periodic parity: the oracle folds the GPU's own linear grids (FP32 -> FP64), as in the on-grid tests
    import oracle as oracle_pkg
    g32 = oracle_pkg.LinearGrids(*(a.cpu().numpy().astype(np.float64) for a in (lin.depth, lin.depth_var, lin.dlogL)))
    orc = oracle_mod.periodic_search(g32, t0_start, stride, p.durations, periods)
    res = assert_periodic_parity(peaks, orc, lambda k, j, pp: oracle_mod.periodic_cell(g32, stride, periods[k], j, pp),
                                 what="config 1 off-grid whole path")
    print("off-grid whole path", res)
    assert_linear_parity(lin.depth.cpu().numpy(), lin.depth_var.cpu().numpy(), lin.dlogL.cpu().numpy(),
                         o.depth, o.depth_var, o.dlogL, what="config 1 off-grid grids")


def test_large_row_fold_all_remainder_widths(torch_cuda, cetra, oracle_mod):
    """Rows larger than shared memory (t0 stride = half a cadence on config-2 data: 39 455 cells, 316 KB per row)
    take the per-period fold kernel; periods are chosen so that the number of phases modulo the 256-phase pass
    leaves every remainder width (1, 2, 3-4, 5-8 groups of 32) and the exact multiples."""
    import oracle as oracle_pkg
    p = _problem(2)
    stride = 0.5 * p.cadence
    n_t0 = 2 * p.n - 1
    durations = p.durations[[0, 7, 15, 22, 29]]
    flux, err = _dev(torch_cuda, p.flux), _dev(torch_cuda, p.flux_err)
    lin = cetra.cetra_linear_search(p.times, flux, err, durations, p.t0_start, stride, n_t0, p.template)
    assert cetra.cetra_stats_pitch(n_t0) * 8 > 232448          # the row cannot be staged in shared memory
    # numbers of phases: 256 m + {0, 1, 20, 33, 64, 65, 100, 128, 129, 200, 255} for a few m
    n_phase = np.array([256 * m + r for m in (3, 4, 9) for r in (0, 1, 20, 33, 64, 65, 100, 128, 129, 200, 255)])
    periods = (n_phase - 0.37) * stride
    assert np.array_equal(np.ceil(periods / stride).astype(int), n_phase)
    periods = np.concatenate([periods, [13.7, 6.01, 27.0, 40.0]])     # few epochs, a single epoch, longer than the data
    peaks = cetra.cetra_periodic_search(lin.depth, lin.depth_var, lin.dlogL, p.t0_start, stride, durations, periods)
    pk = cetra.peaks_to_numpy(peaks)[0]
    g32 = oracle_pkg.LinearGrids(*(a.cpu().numpy().astype(np.float64) for a in (lin.depth, lin.depth_var, lin.dlogL)))
    orc = oracle_mod.periodic_search(g32, p.t0_start, stride, durations, periods)
    res = assert_periodic_parity(pk, orc, lambda k, j, ph: oracle_mod.periodic_cell(g32, stride, periods[k], j, ph),
                                 what="large-row fold")
    print("large-row fold", res)


# ------------------------------------------------------------------------------- error behaviour
def test_status_codes_on_device(torch_cuda, cetra):
    p = _problem(1)
    flux, err = _dev(torch_cuda, p.flux), _dev(torch_cuda, p.flux_err)
    bad_times = p.times.copy()
    bad_times[500] += 0.5 * p.cadence
    with pytest.raises(cetra.CetraError) as e:
        cetra.cetra_linear_search(bad_times, flux, err, p.durations, p.t0_start, p.t0_stride, p.n_t0, p.template)
    assert e.value.status == cetra.CETRA_ERR_NONUNIFORM_TIMES
    with pytest.raises(cetra.CetraError) as e:
        cetra.cetra_linear_search(p.times, flux, err, np.full(129, 0.05), p.t0_start, p.t0_stride, p.n_t0, p.template)
    assert e.value.status == cetra.CETRA_ERR_UNSUPPORTED
    with pytest.raises(cetra.CetraError) as e:
        cetra.cetra_linear_search(p.times, flux, err, -p.durations, p.t0_start, p.t0_stride, p.n_t0, p.template)
    assert e.value.status == cetra.CETRA_ERR_INVALID_ARG
    small = torch_cuda.empty(512, dtype=torch_cuda.uint8, device="cuda")
    with pytest.raises(cetra.CetraError) as e:
        cetra.cetra_linear_search(p.times, flux, err, p.durations, p.t0_start, p.t0_stride, p.n_t0, p.template,
                                  workspace=small)
    assert e.value.status == cetra.CETRA_ERR_WORKSPACE
    before = cetra.cetra_kernel_launch_count()
    cetra.cetra_linear_search(p.times, flux, err, p.durations, p.t0_start, p.t0_stride, p.n_t0, p.template)
    assert cetra.cetra_kernel_launch_count() - before == 3      # preprocess, taps, windowed sums


# ------------------------------------------------------------------------------- random geometries
def _random_light_curve(rng, n, cadence, template):
    """A small seeded light curve with a few box-ish dips, null points and unequal errors (cetra_synth has the
    recipes of the BASELINE configs; this one only has to exercise geometry)."""
    times = 3.0 + np.arange(n) * cadence
    err = rng.uniform(3e-4, 2e-3, size=n)
    flux = 1.0 + rng.normal(size=n) * err
    for _ in range(3):
        c, w = rng.uniform(times[0], times[-1]), rng.uniform(4, 40) * cadence
        flux -= 2e-3 * (np.abs(times - c) < w / 2)
    bad = rng.random(n) < 0.03
    flux[bad] = np.nan
    lo = int(rng.integers(0, n - 40))
    err[lo:lo + int(rng.integers(5, 40))] = np.inf               # a gap of null points
    return times, flux.astype(np.float32), err.astype(np.float32)


@pytest.mark.parametrize("seed", range(12))
def test_linear_search_random_geometries(seed, torch_cuda, cetra, oracle_mod):
    """The three linear-search paths on random small problems, every cell against the oracle: strides on the sample grid
    (q = 1..5), rational off-grid strides p/q with random p, q and start (residue classes: p < q, p > q, a single
    class, starts before the data), and strides that are no small rational multiple (stepped per-cell kernel)."""
    from cetra_synth import tabulate_template
    rng = np.random.default_rng(9000 + seed)
    n = int(rng.integers(300, 2500))
    cadence = float(rng.choice([20.0, 120.0, 600.0])) / 86400.0
    tpl = tabulate_template(int(rng.choice([64, 333, 1024])))
    times, flux, err = _random_light_curve(rng, n, cadence, tpl)
    durations = np.sort(rng.uniform(2.0, 60.0, size=int(rng.integers(1, 6)))) * cadence
    fl, er = _dev(torch_cuda, flux), _dev(torch_cuda, err)
    kinds = ["grid", "rational", "rational", "general"]
    for kind in kinds:
        if kind == "grid":
            stride = int(rng.integers(1, 6)) * cadence
            start = times[0] + int(rng.integers(-30, 30)) * cadence
        elif kind == "rational":
            q = int(rng.integers(1, 24)); p = int(rng.integers(1, 2 * q + 2))
            stride = cadence * p / q
            start = times[0] + rng.uniform(-25, 25) * cadence if rng.random() < 0.7 else times[0] - 3 * cadence
        else:
            stride = cadence * rng.uniform(0.05, 2.5) * (1.0 + 1.0 / 1009.0)
            start = times[0] + rng.uniform(-25, 25) * cadence
        n_t0 = int(min(6000, max(10, (times[-1] - start + 20 * cadence) / stride)))
        o = oracle_mod.linear_search(times, flux, err, durations, start, stride, n_t0, tpl)
        r = cetra.cetra_linear_search(times, fl, er, durations, start, stride, n_t0, tpl, want_stats=True)
        assert_linear_parity(r.depth.cpu().numpy(), r.depth_var.cpu().numpy(), r.dlogL.cpu().numpy(),
                             o.depth, o.depth_var, o.dlogL, what=f"seed {seed} {kind} stride/c = {stride / cadence:.6f}")
        st = r.stats[0].cpu().numpy()
        assert np.all(st[:, n_t0:] == 0) and np.all(st[:, :n_t0, 0][np.isnan(o.depth)] == 0)


def _grids_from_stats(stats, n_t0):
    """The linear-search grids the sufficient-statistics rows stand for, in FP64: stats is one light curve's
    [n_dur][pitch][2] float32 tensor (S_wmm, S_wmf); null cells (S_wmm = 0) become NaN.  Feeding the oracle these
    gives both sides of a periodic-search comparison the same numbers to start from."""
    import oracle as oracle_pkg
    st = stats.cpu().numpy().astype(np.float64)[:, :n_t0, :]
    a, b = st[..., 0], st[..., 1]
    with np.errstate(divide="ignore", invalid="ignore"):
        depth = np.where(a > 0, b / a, np.nan)
        var = np.where(a > 0, 1.0 / a, np.nan)
        dl = np.where(a > 0, 0.5 * b * b / a, np.nan)
    return oracle_pkg.LinearGrids(depth, var, dl)


@pytest.mark.parametrize("seed", range(8))
def test_periodic_search_random_geometries_both_fold_kernels(seed, torch_cuda, cetra, oracle_mod):
    """Random small grids and period sets folded by the resident-row kernel and, through the library's test hook
    (cetra_test_fold_override: forced streaming, small stages), by the streamed kernel with its epoch blocks split and some
    windows too wide for a stage: identical records from both, and parity with the oracle on every period."""
    from cetra_synth import tabulate_template
    rng = np.random.default_rng(7000 + seed)
    n = int(rng.integers(800, 3000))
    cadence = 120.0 / 86400.0
    tpl = tabulate_template(256)
    times, flux, err = _random_light_curve(rng, n, cadence, tpl)
    durations = np.sort(rng.uniform(3.0, 40.0, size=int(rng.integers(2, 5)))) * cadence
    stride = cadence * float(rng.choice([1.0, 0.5, 0.15, 2.0]))
    n_t0 = int((times[-1] - times[0]) / stride) + 1
    span = times[-1] - times[0]
    kinds = rng.integers(0, 3)
    if kinds == 0:
        periods = 1.0 / np.linspace(1.0 / (0.6 * span), 1.0 / (30 * cadence), int(rng.integers(50, 400)))
    elif kinds == 1:
        periods = rng.uniform(20 * cadence, 1.5 * span, size=int(rng.integers(30, 200)))      # unsorted, far apart
    else:
        periods = np.sort(rng.uniform(40 * cadence, 0.3 * span, size=int(rng.integers(30, 200))))
    fl, er = _dev(torch_cuda, flux), _dev(torch_cuda, err)
    lin = cetra.cetra_linear_search(times, fl, er, durations, times[0], stride, n_t0, tpl, want_stats=True)
    torch_cuda.cuda.synchronize()
    # the oracle folds exactly what the GPU folds: the FP32 (S_wmm, S_wmf) rows, as FP64 depth = B/A, var = 1/A
    g64 = _grids_from_stats(lin.stats[0], n_t0)
    orc = oracle_mod.periodic_search(g64, times[0], stride, durations, periods)
    cell = lambda k, j, ph: oracle_mod.periodic_cell(g64, stride, periods[k], j, ph)
    run = lambda: cetra.peaks_to_numpy(cetra.cetra_periodic_search_stats(lin.stats, n_t0, times[0], stride, durations,
                                                                         periods))[0]
    resident = run()
    assert_periodic_parity(resident, orc, cell, what=f"seed {seed} resident-row fold")
    try:
        cetra.cetra_test_fold_override(force_stream=True)
        streamed = run()
        cetra.cetra_test_fold_override(force_stream=True, stage_cells=int(rng.choice([96, 200, 600])))
        streamed_small = run()
    finally:
        cetra.cetra_test_fold_override()
    assert_periodic_parity(streamed, orc, cell, what=f"seed {seed} streamed fold")
    assert_periodic_parity(streamed_small, orc, cell, what=f"seed {seed} streamed fold, small stages")
    same = lambda a, b: np.array_equal(a["i_t0"], b["i_t0"]) and np.array_equal(a["j_dur"], b["j_dur"]) and \
        np.array_equal(a["n_transits"], b["n_transits"])
    assert same(streamed, streamed_small)
    # the two kernels add a cell's epochs in different orders: same winners except at FP32 near-ties
    assert np.mean((resident["i_t0"] == streamed["i_t0"]) & (resident["j_dur"] == streamed["j_dur"])) >= 0.97


def _cancelling_light_curve(rng, n, cadence):
    """Deep events of BOTH signs (dips and equally deep brightenings, tens to hundreds of sigma) at random places:
    folded at a period that is the spacing of two of them, a cell's epochs cancel, the common depth Z is a small
    difference of large per-transit terms, and so is the combined likelihood ratio.  Returns the light curve and the
    event centres."""
    times = 3.0 + np.arange(n) * cadence
    err = rng.uniform(3e-4, 1.2e-3, size=n)
    flux = 1.0 + rng.normal(size=n) * err
    centres = np.sort(rng.uniform(times[0] + 20 * cadence, times[-1] - 20 * cadence, size=int(rng.integers(3, 7))))
    partners = []
    for c in centres:
        depth = float(rng.choice([-1.0, 1.0])) * rng.uniform(0.8e-2, 5e-2)
        width = rng.uniform(6, 30) * cadence
        flux -= depth * (np.abs(times - c) < width / 2)
        if rng.random() < 0.5:
            # a partner of the same shape and nearly the opposite depth: folded at their spacing, 90-99 % of the
            # signal cancels and the cell still stands out of the noise
            c2 = c + float(rng.choice([-1.0, 1.0])) * rng.uniform(60, 0.4 * n) * cadence
            if times[0] + 20 * cadence < c2 < times[-1] - 20 * cadence:
                flux += depth * (1.0 + float(rng.choice([-1.0, 1.0])) * rng.uniform(0.01, 0.1)) * \
                    (np.abs(times - c2) < width / 2)
                partners.append(c2)
    flux[rng.random(n) < 0.02] = np.nan
    return times, flux.astype(np.float32), err.astype(np.float32), np.sort(np.concatenate([centres, partners]))


def test_periodic_search_ill_conditioned_folds(torch_cuda, cetra, oracle_mod):
    """200 seeded problems of the kind the 1e-5 bound is hardest on: events of opposite sign folded
    onto one another, so that the winning cell's LR is what is left of large terms that cancel.  The trial periods
    are the spacings of the events (and their halves), where that happens, plus random ones.  Both fold kernels,
    every period against the oracle folding the same FP32 statistics.  Time-boxed: at least 60 of the 200 seeds must
    have run when the box closes (all of them do on a B200 in well under a minute)."""
    import time
    from cetra_synth import tabulate_template
    tpl = tabulate_template(256)
    cadence = 120.0 / 86400.0
    t_end = time.monotonic() + 150.0
    done, worst, n_cancel = 0, 0.0, 0
    for seed in range(200):
        if time.monotonic() > t_end:
            break
        rng = np.random.default_rng(31000 + seed)
        n = int(rng.integers(500, 1600))
        times, flux, err, centres = _cancelling_light_curve(rng, n, cadence)
        durations = np.sort(rng.uniform(5.0, 32.0, size=3)) * cadence
        stride = cadence * float(rng.choice([1.0, 0.5]))
        n_t0 = int((times[-1] - times[0]) / stride) + 1
        gaps = np.abs(centres[:, None] - centres[None, :])[np.triu_indices(len(centres), 1)]
        cand = np.concatenate([gaps, gaps / 2.0, gaps / 3.0, rng.uniform(40 * cadence, 0.6 * (times[-1] - times[0]), 12)])
        periods = np.sort(cand[cand > durations.max() + 2 * cadence])
        fl, er = _dev(torch_cuda, flux), _dev(torch_cuda, err)
        lin = cetra.cetra_linear_search(times, fl, er, durations, times[0], stride, n_t0, tpl, want_stats=True,
                                        want_grids=False)
        g64 = _grids_from_stats(lin.stats[0], n_t0)
        orc = oracle_mod.periodic_search(g64, times[0], stride, durations, periods)
        cell = lambda k, j, ph: oracle_mod.periodic_cell(g64, stride, periods[k], j, ph)
        run = lambda: cetra.peaks_to_numpy(cetra.cetra_periodic_search_stats(lin.stats, n_t0, times[0], stride,
                                                                             durations, periods))[0]
        resident = run()
        try:
            cetra.cetra_test_fold_override(force_stream=True)
            streamed = run()
        finally:
            cetra.cetra_test_fold_override()
        for name, rec in (("resident", resident), ("streamed", streamed)):
            w = assert_periodic_parity(rec, orc, cell, what=f"cancelling seed {seed} {name}")
            worst = max(worst, w["lr"])
        # how hard the case was: winners whose |Z| is far below the single-epoch depths that went into them
        ok = ~np.isnan(orc.lr)
        single = np.nanmax(np.abs(g64.depth))
        n_cancel += int(np.sum(np.abs(orc.depth[ok]) < 0.05 * single))
        done += 1
    print(f"ill-conditioned fuzz: {done} seeds, {n_cancel} cancelling winners, worst LR error {worst:.3g}")
    assert done >= 60, f"only {done} seeds ran inside the time box"
    assert n_cancel >= done                     # on average at least one strongly cancelling winner per problem
    assert worst <= REL

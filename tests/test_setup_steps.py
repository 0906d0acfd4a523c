"""Resampling, monotransit search and masking through the
C ABI: host helpers against the oracle on CPU, the kernels against the oracle on the GPU."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="module")
def cetra():
    import paper_2503_20875_b200 as c
    c.load_library()
    return c


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: the CETRA library has no CPU fallback")
    torch.cuda.set_device(0)
    return torch


# ------------------------------------------------------------------------------------------ host logic
def test_median_cadence_and_grid_helpers_match_the_oracle(cetra, oracle_mod):
    from cetra_synth import make_irregular_batch
    t, _, _ = make_irregular_batch()
    c = cetra.cetra_median_cadence(t)
    assert c == oracle_mod.median_cadence(t)
    assert c == pytest.approx(120.0 / 86400.0, rel=0.05)
    t_start, c2, n_out = cetra.cetra_resample_grid(t, 0.0, 0.25)       # pad = half of a 0.5 d maximum duration
    pad_n = int(np.ceil(0.25 / c))
    assert c2 == c
    assert t_start == pytest.approx(t.min() - pad_n * c, abs=1e-12)
    assert n_out == int(np.floor((t.max() - t.min()) / c + 0.5)) + 1 + 2 * pad_n
    # every observation lands inside the grid, the padding at both ends holds none
    cell = np.floor((t - t_start) / c + 0.5)
    assert cell.min() == pad_n and cell.max() == n_out - 1 - pad_n
    # an explicit cadence is taken as is
    _, c3, n3 = cetra.cetra_resample_grid(t, 0.5 * c, 0.0)
    assert c3 == 0.5 * c and abs(n3 - 2 * (n_out - 2 * pad_n)) <= 2


def test_setup_argument_errors_without_a_device(cetra):
    import ctypes
    lib = cetra.load_library()
    out = ctypes.c_double()
    t = np.array([0.0, 1.0])
    dp = t.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
    assert lib.cetra_median_cadence(dp, 1, ctypes.byref(out)) == cetra.CETRA_ERR_INVALID_ARG
    assert lib.cetra_median_cadence(None, 2, ctypes.byref(out)) == cetra.CETRA_ERR_INVALID_ARG
    same = np.array([1.0, 1.0, 1.0])
    assert lib.cetra_median_cadence(same.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), 3,
                                    ctypes.byref(out)) == cetra.CETRA_ERR_INVALID_ARG
    assert lib.cetra_resample_workspace_bytes(100, 0, 10) == 0
    assert lib.cetra_resample_workspace_bytes(3000, 2, 1000) >= 4 * (2 * 3000 + 2 * 1000 + 1)
    # the lists are shared by the light curves: the scratch does not grow with their number
    assert lib.cetra_resample_workspace_bytes(3000, 64, 1000) == lib.cetra_resample_workspace_bytes(3000, 2, 1000)
    assert lib.cetra_resample_workspace_bytes(2 ** 31, 1, 1000) == 0           # 32-bit indices
    assert lib.cetra_monotransit_workspace_bytes(3, 1000) >= 3 * 1000 * 9
    assert lib.cetra_mask_workspace_bytes(5) >= 3 * 5 * 8
    # invalid arguments are reported before any device work
    assert lib.cetra_resample(0x1000, 0x1000, 0x1000, 0, 10, 1, 0.0, -1.0, 10, 0x1000, 0x1000, 0x1000, 1 << 20,
                              None) == cetra.CETRA_ERR_INVALID_ARG
    assert lib.cetra_resample(0x1000, 0x1000, 0x1000, 0, 10, 1, 0.0, 1.0, 10, 0x1000, 0x1000, 0x1100, 16,
                              None) == cetra.CETRA_ERR_WORKSPACE


# ------------------------------------------------------------------------------------------- GPU parity
@pytest.mark.gpu
@pytest.mark.parametrize("dtype,shuffle,cad_factor", [("float32", True, 1.0), ("float64", False, 0.5),
                                                       ("float32", True, 2.5)])
def test_resample_matches_oracle(dtype, shuffle, cad_factor, torch_cuda, cetra, oracle_mod):
    from cetra_synth import make_irregular_batch
    torch = torch_cuda
    t, f, e = make_irregular_batch(n_lc=3, n=6000, dtype=np.dtype(dtype), shuffle=shuffle)
    t_start, c, n_out = cetra.cetra_resample_grid(t, cad_factor * cetra.cetra_median_cadence(t), 0.2)
    of, oe = cetra.cetra_resample(torch.from_numpy(t).cuda(), torch.from_numpy(f).cuda(), torch.from_numpy(e).cuda(),
                                  t_start, c, n_out)
    torch.cuda.synchronize()
    of, oe = of.cpu().numpy(), oe.cpu().numpy()
    assert of.dtype == np.dtype(dtype) and of.shape == (3, n_out)
    # FP64 sums in an order-free (atomic) sequence, then one rounding to the output dtype
    eps = 2.0 ** -23 if dtype == "float32" else 1e-13
    n_multi = 0
    for b in range(3):
        rf, re = oracle_mod.resample(t, f[b], e[b], t_start, c, n_out)
        null = np.isnan(rf)
        assert np.array_equal(np.isnan(of[b]), null)                        # identical null pattern (bit-exact cells)
        assert np.all(np.isinf(oe[b][null])) and np.all(oe[b][null] > 0)
        assert np.allclose(of[b][~null], rf[~null], rtol=eps, atol=0)
        assert np.allclose(oe[b][~null], re[~null], rtol=eps, atol=0)
        n_multi += int(np.sum(re[~null] < 0.9 * np.nanmin(e[b][np.isfinite(e[b])])))
    pad_n = int(np.ceil(0.2 / c))
    assert np.all(np.isnan(of[:, :pad_n])) and np.all(np.isnan(of[:, n_out - pad_n:]))
    if cad_factor >= 1.0:
        assert n_multi > 0                      # some points did combine several observations


@pytest.mark.gpu
def test_resample_sums_in_input_order_bit_for_bit(torch_cuda, cetra, oracle_mod):
    """cetra_resample adds a point's observations in ascending input index in FP64, which is the order of the oracle's
    sequential loop: in float64 the two are therefore bit-identical (not merely within rounding), also for shuffled
    input and on a degenerate grid where thousands of observations share one output point (the heapsort branch of the
    per-point index sort); and two runs give the same bits (no floating-point atomics)."""
    from cetra_synth import make_irregular_batch
    torch = torch_cuda
    same = lambda a, b: np.array_equal(a, b, equal_nan=True)
    for shuffle, cad_factor in ((True, 1.0), (False, 3.7), (True, 40.0)):
        t, f, e = make_irregular_batch(n_lc=2, n=5000, dtype=np.float64, shuffle=shuffle)
        t_start, c, n_out = cetra.cetra_resample_grid(t, cad_factor * cetra.cetra_median_cadence(t), 0.1)
        dev = [torch.from_numpy(a).cuda() for a in (t, f, e)]
        first = [a.cpu().numpy() for a in cetra.cetra_resample(*dev, t_start, c, n_out)]
        again = [a.cpu().numpy() for a in cetra.cetra_resample(*dev, t_start, c, n_out)]
        assert same(first[0], again[0]) and same(first[1], again[1])
        for b in range(2):
            rf, re = oracle_mod.resample(t, f[b], e[b], t_start, c, n_out)
            assert same(first[0][b], rf) and same(first[1][b], re), (shuffle, cad_factor, b)
    # everything in three points: lists of thousands of indices
    t, f, e = make_irregular_batch(n_lc=1, n=20000, dtype=np.float64, shuffle=True)
    span = t.max() - t.min()
    of, oe = cetra.cetra_resample(torch.from_numpy(t).cuda(), torch.from_numpy(f).cuda(), torch.from_numpy(e).cuda(),
                                  t.min(), span / 2.0, 3)
    rf, re = oracle_mod.resample(t, f[0], e[0], t.min(), span / 2.0, 3)
    assert same(of.cpu().numpy()[0], rf) and same(oe.cpu().numpy()[0], re)


@pytest.mark.gpu
def test_resample_edge_cases(torch_cuda, cetra, oracle_mod):
    torch = torch_cuda
    # no observation at all / all null / every observation in one point / off-grid observations
    t = np.array([0.0, 0.1, 0.2, 5.0, -3.0, np.nan])
    f = np.array([1.0, 2.0, np.nan, 4.0, 5.0, 6.0], dtype=np.float32)
    e = np.array([0.1, 0.2, 0.1, 0.1, 0.1, 0.1], dtype=np.float32)
    of, oe = cetra.cetra_resample(torch.from_numpy(t).cuda(), torch.from_numpy(f).cuda(), torch.from_numpy(e).cuda(),
                                  0.0, 1.0, 3)
    rf, re = oracle_mod.resample(t, f, e, 0.0, 1.0, 3)
    of, oe = of.cpu().numpy(), oe.cpu().numpy()
    assert np.array_equal(np.isnan(of), np.isnan(rf)) and np.isnan(of[1]) and np.isnan(of[2])
    assert of[0] == pytest.approx(rf[0], rel=1e-6) and oe[0] == pytest.approx(re[0], rel=1e-6)
    empty_t = torch.zeros(0, dtype=torch.float64, device="cuda")
    empty = torch.zeros(0, dtype=torch.float32, device="cuda")
    of, oe = cetra.cetra_resample(empty_t, empty, empty, 0.0, 1.0, 4)
    assert torch.isnan(of).all() and torch.isinf(oe).all()


@pytest.mark.gpu
def test_resampled_light_curve_feeds_the_search(torch_cuda, cetra, oracle_mod):
    """Whole setup path: irregular input -> cetra_resample (padded) -> linear + periodic search, against the oracle
    fed with the oracle's own resampled light curve."""
    from cetra_synth import make_irregular_batch, tabulate_template
    from parity_util import assert_linear_parity
    torch = torch_cuda
    t, f, e = make_irregular_batch(n_lc=2, n=5000, dtype=np.float32)
    durations = np.array([0.05, 0.1, 0.2])
    t_start, c, n_out = cetra.cetra_resample_grid(t, 0.0, 0.5 * durations.max())
    rf, re = cetra.cetra_resample(torch.from_numpy(t).cuda(), torch.from_numpy(f).cuda(), torch.from_numpy(e).cuda(),
                                  t_start, c, n_out)
    times = t_start + c * np.arange(n_out)
    tpl = tabulate_template(1024)
    lin = cetra.cetra_linear_search(times, rf, re, durations, t_start, c, n_out, tpl)
    periods = np.linspace(1.0, 2.5, 301)
    peaks = cetra.peaks_to_numpy(cetra.cetra_periodic_search(lin.depth, lin.depth_var, lin.dlogL, t_start, c,
                                                             durations, periods))
    for b in range(2):
        of, oe = oracle_mod.resample(t, f[b], e[b], t_start, c, n_out)
        # the oracle sees the same FP32 light curve the GPU search saw
        g = oracle_mod.linear_search(times, rf[b].cpu().numpy(), re[b].cpu().numpy(), durations, t_start, c, n_out, tpl)
        assert np.allclose(rf[b].cpu().numpy()[~np.isnan(of)], of[~np.isnan(of)], rtol=2.0 ** -23)
        assert_linear_parity(lin.depth[b].cpu().numpy(), lin.depth_var[b].cpu().numpy(), lin.dlogL[b].cpu().numpy(),
                             g.depth, g.depth_var, g.dlogL, what=f"resampled curve {b}")
        pg = oracle_mod.periodic_search(g, t_start, c, durations, periods)
        k = int(np.nanargmax(pg.lr))
        kg = int(np.nanargmax(peaks[b]["lr"]))
        assert k == kg and abs(periods[k] - (1.3 + 0.4 * b)) < 0.01          # the injected period is found
        assert peaks[b]["i_t0"][k] == pg.i_t0[k] and peaks[b]["j_dur"][k] == pg.j_dur[k]


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,n_peaks,excl", [(1, 5, 1.0), (2, 12, 1.5)])
def test_monotransit_search_matches_oracle(cfg, n_peaks, excl, torch_cuda, cetra, oracle_mod):
    from cetra_synth import make_config
    import oracle as oracle_pkg
    torch = torch_cuda
    p = make_config(cfg, n_periods=10)
    flux, err = torch.from_numpy(p.flux).cuda(), torch.from_numpy(p.flux_err).cuda()
    lin = cetra.cetra_linear_search(p.times, flux, err, p.durations, p.t0_start, p.t0_stride, p.n_t0, p.template)
    res = cetra.cetra_monotransit_search(lin.depth, lin.depth_var, lin.dlogL, p.t0_start, p.t0_stride, p.durations,
                                         n_peaks, excl, want_profile=True)
    torch.cuda.synchronize()
    # the oracle is fed the GPU's own FP32 grids, so that every comparison it makes is between the same values:
    # profile, duration index and the greedy event sequence must then be identical
    g = oracle_pkg.LinearGrids(*(a.cpu().numpy().astype(np.float64) for a in (lin.depth, lin.depth_var, lin.dlogL)))
    m = oracle_mod.monotransit(g, p.t0_stride, p.durations, n_peaks, excl)
    pl, pj = res.profile_lr[0].cpu().numpy(), res.profile_j[0].cpu().numpy()
    assert np.array_equal(pj, m.profile_j)
    assert np.array_equal(np.isnan(pl), np.isnan(m.profile_lr))
    assert np.array_equal(pl[~np.isnan(pl)].astype(np.float64), m.profile_lr[~np.isnan(pl)])
    ev = cetra.events_to_numpy(res.events)[0]
    nf = int(res.n_found.cpu().numpy()[0])
    assert nf == len(m.i_t0) == n_peaks
    assert np.array_equal(ev["i_t0"][:nf], m.i_t0) and np.array_equal(ev["j_dur"][:nf], m.j_dur)
    assert np.array_equal(ev["lr"][:nf].astype(np.float64), m.lr)
    assert np.array_equal(ev["depth"][:nf].astype(np.float64), m.depth)
    assert np.array_equal(ev["depth_var"][:nf].astype(np.float64), m.depth_var)
    assert np.allclose(ev["t0"][:nf], p.t0_start + m.i_t0 * p.t0_stride, rtol=1e-6)
    if cfg == 1:            # the strongest event is the injected single transit (t0 = 0.7 d, D = 2 h)
        assert abs(ev["t0"][0] - 0.7) <= 3 * p.t0_stride
        assert abs(p.durations[ev["j_dur"][0]] - 2.0 / 24.0) < 0.03


@pytest.mark.gpu
def test_monotransit_runs_out_and_batches(torch_cuda, cetra, oracle_mod):
    import oracle as oracle_pkg
    torch = torch_cuda
    rng = np.random.default_rng(4)
    n_lc, n_dur, n_t0 = 3, 4, 300
    dl = rng.random((n_lc, n_dur, n_t0)).astype(np.float32)
    dl[0, :, 50:80] = np.nan                       # a fully null stretch
    dl[1] = np.nan                                 # a light curve with no candidate at all
    dl[2, 1, 7] = dl[2, 3, 7] = 5.0                # a tie between durations and ...
    dl[2, 0, 200] = 5.0                            # ... between reference times
    depth = rng.standard_normal((n_lc, n_dur, n_t0)).astype(np.float32)
    var = rng.random((n_lc, n_dur, n_t0)).astype(np.float32) + 0.1
    durations = np.array([0.5, 1.0, 2.0, 4.0])
    res = cetra.cetra_monotransit_search(torch.from_numpy(depth).cuda(), torch.from_numpy(var).cuda(),
                                         torch.from_numpy(dl).cuda(), 10.0, 0.1, durations, 40, 2.0)
    ev = cetra.events_to_numpy(res.events)
    nf = res.n_found.cpu().numpy()
    for b in range(n_lc):
        g = oracle_pkg.LinearGrids(depth[b].astype(np.float64), var[b].astype(np.float64), dl[b].astype(np.float64))
        m = oracle_mod.monotransit(g, 0.1, durations, 40, 2.0)
        assert nf[b] == len(m.i_t0) < 40
        assert np.array_equal(ev[b]["i_t0"][:nf[b]], m.i_t0) and np.array_equal(ev[b]["j_dur"][:nf[b]], m.j_dur)
        assert np.all(ev[b]["i_t0"][nf[b]:] == -1) and np.all(np.isnan(ev[b]["lr"][nf[b]:]))
    assert nf[1] == 0
    assert ev[2]["i_t0"][0] == 7 and ev[2]["j_dur"][0] == 1          # ties: smallest i, then smallest j


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", ["float32", "float64"])
def test_mask_transits_matches_oracle(dtype, torch_cuda, cetra, oracle_mod):
    from cetra_synth import make_config
    torch = torch_cuda
    p = make_config(2, n_periods=10)
    n_lc = 4
    flux = np.tile(p.flux.astype(dtype), (n_lc, 1))
    period = np.array([5.3, 0.0, 1.234567, 2.0])
    t0 = np.array([1.7, 20.0, 0.3, np.nan])                         # the last curve is left untouched
    dur = np.array([0.125, 0.5, 0.02, 0.1])
    fd = torch.from_numpy(flux).cuda()
    n_masked = cetra.cetra_mask_transits(torch.from_numpy(p.times).cuda(), fd, period, t0, dur, width=1.5)
    out = fd.cpu().numpy()
    nm = n_masked.cpu().numpy()
    for b in range(n_lc):
        if np.isnan(t0[b]):
            assert nm[b] == 0 and np.array_equal(np.isnan(out[b]), np.isnan(flux[b]))
            continue
        ref, cnt = oracle_mod.mask_transits(p.times, flux[b], period[b], t0[b], dur[b], 1.5)
        assert np.array_equal(np.isnan(out[b]), np.isnan(ref))       # bit-exact sample set
        assert nm[b] == cnt
        keep = ~np.isnan(ref)
        assert np.array_equal(out[b][keep], flux[b][keep])


@pytest.mark.gpu
def test_mask_and_research_finds_the_second_planet(torch_cuda, cetra):
    """PAPER.md:258 on the GPU: search, nullify the best signal, search again."""
    from cetra_synth import tabulate_template, transit_profile
    torch = torch_cuda
    rng = np.random.default_rng(8)
    c, n = 10.0 / 1440.0, 2880
    t = c * np.arange(n)
    f = 1.0 + 3e-4 * rng.standard_normal(n)
    for P, t0, D, d in ((2.0, 0.4, 0.15, 3e-3), (3.1, 1.3, 0.15, 1.5e-3)):
        ph = np.mod(t - t0 + 0.5 * P, P) - 0.5 * P
        x = ph / D + 0.5
        ins = (x >= 0) & (x <= 1)
        f[ins] -= d * transit_profile(x[ins])
    fd = torch.from_numpy(f.astype(np.float32)).cuda()
    ed = torch.full_like(fd, 3e-4)
    td = torch.from_numpy(t).cuda()
    durations = np.array([0.1, 0.15, 0.2])
    periods = np.linspace(1.5, 4.0, 501)
    tpl = tabulate_template(1024)
    found = []
    for _ in range(2):
        peaks = cetra.peaks_to_numpy(cetra.cetra_search_batched(t, fd[None], ed[None], durations, t[0], c, n, tpl,
                                                                periods))[0]
        k = int(np.nanargmax(peaks["lr"]))
        found.append(periods[k])
        cetra.cetra_mask_transits(td, fd, periods[k], float(peaks["t0"][k]), durations[peaks["j_dur"][k]], width=2.0)
    assert abs(found[0] - 2.0) < 0.02 and abs(found[1] - 3.1) < 0.03

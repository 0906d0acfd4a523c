"""Tolerances and comparison helpers of the GPU-vs-oracle parity tests (R13, R15).

north_star: relative 1e-5 on depth and dlogL, identical peak indices on injected signals.  Where a
quantity crosses zero the relative error is taken against its natural scale (R15):
    |depth_g - depth_o| <= 1e-5 * max(|depth_o|, sigma_o)        sigma_o = sqrt(var_o)
    |var_g   - var_o|   <= 1e-5 * var_o
    |LR_g    - LR_o|    <= 1e-5 * max(LR_o, 1/2)
and the null (NaN) pattern must be identical.
"""
import numpy as np

REL = 1e-5


def assert_linear_parity(depth_g, var_g, dl_g, depth_o, var_o, dl_o, what=""):
    depth_g, var_g, dl_g = (np.asarray(a, dtype=np.float64) for a in (depth_g, var_g, dl_g))
    nan_o = np.isnan(depth_o)
    for name, a in (("depth", depth_g), ("var", var_g), ("dlogL", dl_g)):
        assert np.array_equal(np.isnan(a), nan_o), f"{what}: null pattern of {name} differs"
    ok = ~nan_o
    sig = np.sqrt(var_o[ok])
    e_d = np.abs(depth_g[ok] - depth_o[ok]) / np.maximum(np.abs(depth_o[ok]), sig)
    e_v = np.abs(var_g[ok] - var_o[ok]) / var_o[ok]
    e_l = np.abs(dl_g[ok] - dl_o[ok]) / np.maximum(dl_o[ok], 0.5)
    worst = dict(depth=float(e_d.max(initial=0.0)), var=float(e_v.max(initial=0.0)), dlogL=float(e_l.max(initial=0.0)))
    assert worst["depth"] <= REL and worst["var"] <= REL and worst["dlogL"] <= REL, f"{what}: {worst}"
    return worst


def assert_periodic_parity(peaks, orc, cell_lr, what="", must_match=()):
    """peaks: numpy PEAK_DTYPE [K] from the GPU.  orc: oracle Periodogram on the same inputs.
    cell_lr(k, j, p) -> oracle LR of one (period, duration, phase) cell (R13: a GPU winner that is not
    the oracle's winner must be a cell whose oracle LR is within tolerance of the oracle maximum).
    must_match: period indices where (j, p) must be identical (injected peaks)."""
    K = orc.lr.shape[0]
    assert peaks.shape[0] == K
    none_o = np.isnan(orc.lr)
    assert np.array_equal(np.isnan(peaks["lr"]), none_o), f"{what}: no-candidate periods differ"
    assert np.all(peaks["j_dur"][none_o] == -1) and np.all(peaks["i_t0"][none_o] == -1)
    n_alt = 0
    worst = 0.0
    for k in np.nonzero(~none_o)[0]:
        tol = REL * max(orc.lr[k], 0.5)
        same = peaks["j_dur"][k] == orc.j_dur[k] and peaks["i_t0"][k] == orc.i_t0[k]
        if same:
            ref_lr, ref_z, ref_v, ref_n = orc.lr[k], orc.depth[k], orc.depth_var[k], orc.n_transits[k]
        else:
            assert k not in must_match, f"{what}: indices differ at injected period {k}"
            ref_lr, ref_z, ref_v, ref_n = cell_lr(k, int(peaks["j_dur"][k]), int(peaks["i_t0"][k]))
            assert abs(ref_lr - orc.lr[k]) <= tol, f"{what}: period {k}: GPU cell is not a near-tie of the maximum"
            n_alt += 1
        err = abs(float(peaks["lr"][k]) - ref_lr)
        worst = max(worst, err / max(ref_lr, 0.5))
        assert err <= REL * max(ref_lr, 0.5), f"{what}: period {k}: LR {peaks['lr'][k]} vs {ref_lr}"
        assert abs(float(peaks["depth"][k]) - ref_z) <= REL * max(abs(ref_z), np.sqrt(ref_v)), f"{what}: depth @ {k}"
        assert abs(float(peaks["depth_var"][k]) - ref_v) <= REL * ref_v, f"{what}: var @ {k}"
        assert int(peaks["n_transits"][k]) == ref_n, f"{what}: n_transits @ {k}"
    # near-ties must be rare
    assert n_alt <= max(2, K // 50), f"{what}: {n_alt} of {K} periods picked a different (tied) cell"
    return dict(lr=worst, alt=n_alt)


def period_subset(periods, injected, n_random, seed, half_width=60):
    """Indices of a seeded random subset of the trial periods plus windows around each injected period and
    its x1/2 and x2 aliases (SURVEY.md §8(d) 'Checks')."""
    rng = np.random.default_rng(seed)
    K = periods.shape[0]
    pick = set(rng.choice(K, size=min(n_random, K), replace=False).tolist())
    for p_inj in injected:
        for mult in (0.5, 1.0, 2.0):
            target = p_inj * mult
            if target < periods.min() or target > periods.max():
                continue
            k0 = int(np.argmin(np.abs(periods - target)))
            pick.update(range(max(0, k0 - half_width), min(K, k0 + half_width + 1)))
    return np.array(sorted(pick), dtype=np.int64)


def nearest_template_sample(x, M):
    """Index of the tabulated template sample nearest to position x in [0, 1] ("the nearest model point
    is selected"), straight from the definition: the template's M samples sit at m / (M - 1), m = 0 .. M-1 (first to
    last contact), and the nearest one is found by comparing distances.  No rounding expression is involved, so a test
    that takes its indices from here does not repeat the oracle's (or the kernels') arithmetic.  Also returns the
    margin by which the nearest sample wins over the runner-up, so callers can keep clear of exact half-steps, where
    "nearest" has two answers."""
    x = np.atleast_1d(np.asarray(x, dtype=np.float64))
    pos = np.arange(M, dtype=np.float64) / (M - 1.0)
    dist = np.abs(x[:, None] - pos[None, :])
    order = np.argsort(dist, axis=1, kind="stable")
    rows = np.arange(x.shape[0])
    return order[:, 0], dist[rows, order[:, 1]] - dist[rows, order[:, 0]]

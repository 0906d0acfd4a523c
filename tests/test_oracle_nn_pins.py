"""Independent pins of the oracle's nearest-neighbour template index ("the nearest model point is
selected"; R3 on the sample grid, R25 off it), and of two tie rules of the setup steps.  CPU only.

Why a file of its own: the oracle evaluates the index as one rounding expression, the CUDA kernels use the same
one, and before this file every test that could see it either repeated that expression or compared the oracle with
itself.  Here the expected index comes from `parity_util.nearest_template_sample`, which compares the distances to
the M tabulated positions m / (M - 1) and contains no rounding expression at all.

The probe is a one-hot template: tpl[m*] = 1 and 0 elsewhere.  Then for a cell (t_i, D)
    S_wmm = sum of w_n over exactly those samples whose nearest template sample is m*,
    S_wmf = sum of w_n f_n over the same samples,
so depth_var = 1 / S_wmm and depth = S_wmf / S_wmm reveal the set, and a cell with no such sample is null.  The
weights are 2^-n-like distinct values, so that two different sets never give the same sum.

Mutants of the index expression that this file kills (each was applied to oracle/cetra_oracle.c on a scratch copy,
in all four places and in the on-grid / off-grid forms separately):
    truncation            floor(x (M-1))            instead of rounding to nearest
    rounding up           ceil(x (M-1))
    short table           floor(x (M-1-1/2) + 1/2)  (positions stretched over M - 1/2 samples)
    M instead of M-1      floor(x M)                (last contact mapped past the table)
    reversed template     M-1 - index
and truncation in each one of the four places alone (first and second pass of either form).
None of the assertions below contains the oracle's expression.
"""
import numpy as np
import pytest

from parity_util import nearest_template_sample


@pytest.fixture(scope="module")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


def _light_curve(n, c, seed):
    rng = np.random.default_rng(seed)
    t = 3.25 + c * np.arange(n)
    f = 1.0 - rng.uniform(1e-4, 3e-3, n)
    # distinct weights with an irrational-looking spread: sums over different sample sets differ by far more than 1e-12
    e = 1e-3 * np.sqrt(1.0 + np.mod(np.arange(n) * 0.6180339887498949, 1.0) * 3.0)
    f[n // 2 + 7] = np.nan                                    # a null sample inside some windows
    return t, f, e


def _expected_from_the_definition(t, f, e, ti, D, M, m_star):
    """(depth, var) of the one-hot template at reference time ti, duration D -- or None for a null cell -- and the
    smallest margin to a half-step among the window's samples."""
    x = (t - ti) / D + 0.5
    ins = (x >= 0.0) & (x <= 1.0) & np.isfinite(f)
    idx, margin = nearest_template_sample(x[ins], M)
    edge = min(np.min(np.abs(x)), np.min(np.abs(x - 1.0)))    # distance of any sample to a window edge
    sel = np.flatnonzero(ins)[idx == m_star]
    w = 1.0 / e[sel] ** 2
    clear = min(float(margin.min(initial=1.0)), float(edge))
    if sel.size == 0:
        return None, clear
    return (float(np.sum(w * (1.0 - f[sel])) / np.sum(w)), float(1.0 / np.sum(w))), clear


@pytest.mark.parametrize("M", [9, 33])
@pytest.mark.parametrize("mode", ["on_grid", "on_grid_through_general", "off_grid"])
def test_one_hot_template_selects_the_nearest_tabulated_sample(oracle_mod, M, mode):
    n, c = 260, 0.01
    t, f, e = _light_curve(n, c, 11)
    durations = np.array([0.2137, 0.5519])                    # 21 and 55 samples: several per template step for M = 9
    if mode == "off_grid":
        t0_start, stride, n_t0 = t[0] + 0.37 * c, 0.3 * c, 700
    else:
        t0_start, stride, n_t0 = t[0] - 3 * c, c, 250
    cells = [5, 40, 111, 135, 201, n_t0 - 2]
    n_checked = n_null = 0
    for m_star in range(M):
        tpl = np.zeros(M)
        tpl[m_star] = 1.0
        g = oracle_mod.linear_search(t, f, e, durations, t0_start, stride, n_t0, tpl,
                                     force_general=(mode == "on_grid_through_general"))
        for j, D in enumerate(durations):
            for i in cells:
                want, clear = _expected_from_the_definition(t, f, e, t0_start + i * stride, D, M, m_star)
                assert clear > 1e-9                           # "nearest" is unambiguous for every sample of the window
                if want is None:
                    assert np.isnan(g.depth[j, i]) and np.isnan(g.depth_var[j, i]) and np.isnan(g.dlogL[j, i])
                    n_null += 1
                    continue
                assert g.depth_var[j, i] == pytest.approx(want[1], rel=1e-12), (m_star, j, i)
                assert g.depth[j, i] == pytest.approx(want[0], rel=1e-11), (m_star, j, i)
                # the second pass (literal Eq. 2) must have sampled the template at the same indices:
                # only then does it equal the closed form 1/2 depth^2 / var of this sample set
                assert g.dlogL[j, i] == pytest.approx(0.5 * want[0] ** 2 / want[1], rel=1e-9), (m_star, j, i)
                n_checked += 1
    assert n_checked > 8 * M                                  # the pin looked at many (template sample, cell) pairs
    if M == 33:
        assert n_null > 0                                     # ... and at template samples no observation is nearest to


def test_one_hot_sets_partition_the_window(oracle_mod):
    """Summed over m*, the one-hot sets are the whole window: sum_m* S_wmm(m*) = sum of w over the window, which is what
    a box template gives.  A rounding rule that sends some sample to no table entry, or to two, breaks the total."""
    n, c, M = 200, 0.01, 17
    t, f, e = _light_curve(n, c, 5)
    durations = np.array([0.3331])
    t0_start, stride, n_t0 = t[0] + 0.41 * c, 0.7 * c, 250
    total = np.zeros(n_t0)
    for m_star in range(M):
        tpl = np.zeros(M)
        tpl[m_star] = 1.0
        g = oracle_mod.linear_search(t, f, e, durations, t0_start, stride, n_t0, tpl)
        total += np.where(np.isnan(g.depth_var[0]), 0.0, 1.0 / g.depth_var[0])
    box = oracle_mod.linear_search(t, f, e, durations, t0_start, stride, n_t0, np.ones(M))
    ok = ~np.isnan(box.depth_var[0])
    assert ok.sum() > 200
    assert np.allclose(total[ok], 1.0 / box.depth_var[0][ok], rtol=1e-12)
    assert np.all(total[~ok] == 0.0)


# ------------------------------------------------------------------------------ tie rules of the setup steps
def test_median_cadence_of_an_even_count_averages_two_different_middle_values(oracle_mod):
    """R22: with an even number of differences the median is the mean of the two middle ones.  The differences here
    are all distinct, so the two middle values differ and taking either of them alone is wrong by a known amount."""
    d = np.array([0.5, 0.0625, 0.25, 1.0, 0.125, 2.0])         # exact binary fractions: sums are exact
    t = np.concatenate([[10.0], 10.0 + np.cumsum(d)])
    assert oracle_mod.median_cadence(t) == 0.375               # (0.25 + 0.5) / 2, not 0.25 and not 0.5
    assert oracle_mod.median_cadence(t[::-1].copy()) == 0.375  # input order is irrelevant
    assert oracle_mod.median_cadence(t[:-1]) == 0.25           # odd count: the middle value itself


def test_monotransit_ties_go_to_the_smallest_duration_and_the_earliest_time(oracle_mod):
    """R23: equal dlogL at one reference time -> the smallest duration index; equal profile maxima -> the earliest
    reference time.  A hand-built grid with exact ties."""
    import oracle as oracle_pkg
    n_dur, n_t0 = 3, 40
    dl = np.full((n_dur, n_t0), 1.0)
    dl[1, 10] = dl[2, 10] = 9.0                                # durations 1 and 2 tie at cell 10
    dl[0, 30] = dl[2, 30] = 9.0                                # cells 10 and 30 tie; at 30 durations 0 and 2 tie
    depth = np.arange(n_dur * n_t0, dtype=np.float64).reshape(n_dur, n_t0)
    var = depth + 0.5
    g = oracle_pkg.LinearGrids(depth, var, dl)
    m = oracle_mod.monotransit(g, 1.0, np.array([1.0, 2.0, 3.0]), n_peaks=2, excl=1.0)
    assert m.profile_j[10] == 1 and m.profile_j[30] == 0 and m.profile_j[0] == 0
    assert list(m.i_t0) == [10, 30] and list(m.j_dur) == [1, 0]
    assert m.depth[0] == depth[1, 10] and m.depth_var[1] == var[0, 30]

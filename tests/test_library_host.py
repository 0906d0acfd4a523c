"""CPU-side checks of the C-ABI library: it builds, loads, exports every symbol include/cetra.h declares,
sizes its workspaces, and reports argument errors before touching the device.  No compute call here
reaches a kernel launch (there is no GPU in the build container)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cetra():
    import paper_2503_20875_b200 as c
    c.load_library()
    return c


def _has_cuda():
    import torch
    return torch.cuda.is_available()


def test_library_exports_every_declared_symbol(cetra):
    header = open(os.path.join(ROOT, "include", "cetra.h")).read()
    declared = set(re.findall(r"\b(cetra_[a-z0-9_]+)\s*\(", header))
    assert declared == set(cetra.EXPORTED_SYMBOLS)
    lib = cetra.load_library()
    for name in declared:
        assert getattr(lib, name) is not None
    # the measurement probes have a header and a library of their own; the product exports none of them
    diag_header = open(os.path.join(ROOT, "include", "cetra_diag.h")).read()
    diag_declared = set(re.findall(r"\b(cetra_[a-z0-9_]+)\s*\(", diag_header))
    assert diag_declared == set(cetra.DIAG_SYMBOLS) and not (diag_declared & declared)
    diag = cetra.load_diag_library()
    for name in diag_declared:
        assert getattr(diag, name) is not None
        assert not hasattr(lib, name), f"{name} leaked into the product ABI"


def test_product_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the package may import or load it."""
    pkg = os.path.join(ROOT, "paper_2503_20875_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b|libcetra_oracle|cetra_oracle\.c|oracle/",
                                     text, flags=re.M), f"{f} reaches into oracle/"


def test_status_strings_and_pitch(cetra):
    assert cetra.status_string(0) == "ok"
    for s in (-1, -2, -3, -4, -5):
        assert cetra.status_string(s) not in ("ok", "unknown status")
    assert cetra.status_string(-99) == "unknown status"
    for n_t0 in (1, 31, 32, 1000, 19728, 256464):
        pitch = cetra.cetra_stats_pitch(n_t0)
        assert pitch % 32 == 0 and pitch >= n_t0 + 128


def test_workspace_sizes_scale_with_the_problem(cetra):
    from cetra_synth import make_config
    p = make_config(2, n_periods=100)
    one = cetra.cetra_linear_workspace_bytes(p.times, 1, p.durations, p.t0_start, p.t0_stride, p.n_t0, 1024)
    four = cetra.cetra_linear_workspace_bytes(p.times, 4, p.durations, p.t0_start, p.t0_stride, p.n_t0, 1024)
    assert 0 < one < four
    # (w f, w) per sample and light curve dominates: 8 B x N
    assert four - one >= 3 * 8 * p.n
    per = cetra.cetra_periodic_workspace_bytes(1, 30, p.t0_start, p.t0_stride, p.n_t0, 20000)
    assert per >= 8 * 30 * cetra.cetra_stats_pitch(p.n_t0) + 8 * 20000 + 8 * 20000
    b = cetra.cetra_search_batched_workspace_bytes(p.times, 1000, 0, p.durations, p.t0_start, p.t0_stride, p.n_t0,
                                                   1024, 20000)
    b8 = cetra.cetra_search_batched_workspace_bytes(p.times, 1000, 8, p.durations, p.t0_start, p.t0_stride, p.n_t0,
                                                    1024, 20000)
    assert 0 < b8 < b < 700 << 20          # the default chunk keeps the resident grids within 512 MiB
    # invalid problems have no workspace size
    bad = p.times.copy()
    bad[10] += 0.4 * p.cadence
    assert cetra.cetra_linear_workspace_bytes(bad, 1, p.durations, p.t0_start, p.t0_stride, p.n_t0, 1024) == 0


def test_plan_picks_the_off_grid_path_by_the_stride(cetra):
    """Host plan logic, seen through the workspace sizes (no device needed): a t0 stride that is a small rational multiple
    of the cadence (the paper's default, 18 s on 2-min data = 3/20) gets one set of tap tables per residue
    class; any other stride keeps the per-cell kernel, which needs no tap tables; a template set needs one statistics
    grid and one set of tap tables per template."""
    from cetra_synth import make_config
    p = make_config(2, n_periods=100)
    c, n_t0 = p.cadence, 30000
    w = lambda start, stride: cetra.cetra_linear_workspace_bytes(p.times, 1, p.durations, start, stride, n_t0, 1024)
    on_grid = w(p.times[0], c)
    classes = w(p.times[0], 0.15 * c)                      # 3/20: 20 classes, each with its own tables and lists
    general = w(p.times[0], 0.15 * c * (1.0 + 1.0 / 977.0))
    shifted = w(p.times[0] + 0.3 * c, 2 * c)               # whole-sample stride, off-grid start: one class
    assert 0 < general < on_grid < shifted < classes
    assert classes > 3 * on_grid                           # 20 x the tables, with their flags and lists
    # an almost rational stride is rational only while the cells stay within 1e-6 samples of their class position
    assert w(p.times[0], 0.15 * c * (1.0 + 1e-12)) == classes
    assert w(p.times[0], 0.15 * c * (1.0 + 1e-9)) == general
    lib = cetra.load_library()
    from paper_2503_20875_b200.binding import cetra_t0_grid, _dp, _f64
    t, d = _f64(p.times), _f64(p.durations)
    grid = cetra_t0_grid(p.t0_start, p.t0_stride, p.n_t0)
    one = lib.cetra_search_batched_templates_workspace_bytes(_dp(t), t.shape[0], 8, 8, _dp(d), d.shape[0], grid, 1024, 1, 100)
    three = lib.cetra_search_batched_templates_workspace_bytes(_dp(t), t.shape[0], 8, 8, _dp(d), d.shape[0], grid, 1024, 3, 100)
    assert one == cetra.cetra_search_batched_workspace_bytes(p.times, 8, 8, p.durations, p.t0_start, p.t0_stride, p.n_t0, 1024, 100)
    stats = 8 * 8 * d.shape[0] * cetra.cetra_stats_pitch(p.n_t0)
    assert three - one >= 2 * stats and three - one < 2 * stats + (1 << 20)


def _call_linear(cetra, times, durations, t0_start, stride, n_t0, n_tpl=64, flux=0x1000, ws=0x10000, ws_bytes=1 << 30,
                 dtype=0, n_lc=1):
    lib = cetra.load_library()
    from paper_2503_20875_b200.binding import cetra_t0_grid
    times = np.ascontiguousarray(times, dtype=np.float64)
    durations = np.ascontiguousarray(durations, dtype=np.float64)
    tpl = np.ones(n_tpl, dtype=np.float32)
    dp = ctypes.POINTER(ctypes.c_double)
    return lib.cetra_linear_search(times.ctypes.data_as(dp), flux, flux, dtype, times.shape[0], n_lc,
                                   durations.ctypes.data_as(dp), durations.shape[0],
                                   cetra_t0_grid(t0_start, stride, n_t0), tpl.ctypes.data, n_tpl, None, None, None,
                                   None, ws, ws_bytes, None)


def test_argument_errors_are_reported_without_a_device(cetra):
    """Validation happens before any device work, so these statuses are the same on a CPU-only host."""
    c = 0.01
    times = np.arange(500) * c
    dur = np.array([0.05, 0.1])
    ok_args = (times, dur, 0.0, c, 500)
    assert _call_linear(cetra, *ok_args, flux=None) == cetra.CETRA_ERR_INVALID_ARG
    assert _call_linear(cetra, *ok_args, dtype=7) == cetra.CETRA_ERR_INVALID_ARG
    assert _call_linear(cetra, times, -dur, 0.0, c, 500) == cetra.CETRA_ERR_INVALID_ARG
    assert _call_linear(cetra, times, dur, 0.0, c, 0) == cetra.CETRA_ERR_INVALID_ARG
    assert _call_linear(cetra, times, dur, 0.0, -c, 500) == cetra.CETRA_ERR_INVALID_ARG
    assert _call_linear(cetra, times, np.full(129, 0.05), 0.0, c, 500) == cetra.CETRA_ERR_UNSUPPORTED
    # t0 grids off the sample grid are legal (R25): with valid arguments only the missing device can fail
    assert _call_linear(cetra, times, dur, 0.0, 1.5 * c, 100) in (cetra.CETRA_ERR_CUDA, cetra.CETRA_OK)
    assert _call_linear(cetra, times, dur, 0.25 * c, c, 100) in (cetra.CETRA_ERR_CUDA, cetra.CETRA_OK)
    jitter = times.copy()
    jitter[123] += 0.01 * c
    assert _call_linear(cetra, jitter, dur, 0.0, c, 500) == cetra.CETRA_ERR_NONUNIFORM_TIMES
    assert _call_linear(cetra, *ok_args, ws=None) == cetra.CETRA_ERR_WORKSPACE
    assert _call_linear(cetra, *ok_args, ws=0x10008) == cetra.CETRA_ERR_WORKSPACE      # misaligned
    assert _call_linear(cetra, *ok_args, ws_bytes=1024) == cetra.CETRA_ERR_WORKSPACE


def test_compute_fails_loudly_without_a_device(cetra):
    """No CPU fallback: with valid arguments and no GPU the entry point returns CETRA_ERR_CUDA, and the
    Python binding refuses to run."""
    if _has_cuda():
        pytest.skip("a CUDA device is present")
    c = 0.01
    times = np.arange(500) * c
    assert _call_linear(cetra, times, np.array([0.05]), 0.0, c, 500) == cetra.CETRA_ERR_CUDA
    import torch
    with pytest.raises((RuntimeError, TypeError)):
        cetra.cetra_linear_search(times, torch.ones(500), torch.ones(500), np.array([0.05]), 0.0, c, 500,
                                  np.ones(16, np.float32))


def test_peak_record_layout(cetra):
    from paper_2503_20875_b200.binding import cetra_peak
    assert ctypes.sizeof(cetra_peak) == 32 == cetra.PEAK_DTYPE.itemsize
    for name, _ in cetra_peak._fields_:
        assert getattr(cetra_peak, name).offset == cetra.PEAK_DTYPE.fields[name][1]


def test_resample_template_host_helper_matches_the_oracle(cetra, oracle_mod):
    """cetra_resample_template (host-side setup helper) against the oracle's linear interpolation."""
    from cetra_synth import tabulate_template
    dense = tabulate_template(20001)                              # a densely sampled model, as the paper ships
    for m in (64, 1024, 4096):
        got = cetra.cetra_resample_template(dense, m)
        want = oracle_mod.resample_template(dense.astype(np.float32).astype(np.float64), m)
        assert got.dtype == np.float32 and got.shape == (m,)
        assert np.array_equal(got, want.astype(np.float32)) or np.abs(got - want).max() <= 6e-8
    with pytest.raises(cetra.CetraError):
        cetra.cetra_resample_template(dense[:1], 8)


def test_light_curve_count_limits_of_one_launch(cetra):
    """Light curves are one dimension of the linear kernel's launch grid (65 535 at most).  cetra_linear_search says so
    (no workspace size = unsupported); the batched search slices by itself and clamps a caller's larger chunk."""
    c = 2.0 / 1440.0
    times = c * np.arange(64)
    durations = np.array([4 * c, 8 * c])
    args = (durations, 0.0, c, 64, 32)
    assert cetra.cetra_linear_workspace_bytes(times, 65535, *args) > 0
    assert cetra.cetra_linear_workspace_bytes(times, 65536, *args) == 0
    at_limit = cetra.cetra_search_batched_workspace_bytes(times, 100000, 65535, *args, 10)
    beyond = cetra.cetra_search_batched_workspace_bytes(times, 100000, 90000, *args, 10)
    smaller = cetra.cetra_search_batched_workspace_bytes(times, 100000, 30000, *args, 10)
    assert 0 < smaller < at_limit == beyond

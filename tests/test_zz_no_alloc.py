"""cetra_resample_static: the resampler for callers that cannot allocate device memory (include/cetra.h).

Some users of this library are handed their input and output buffers and nothing else: a stage plugged into another
program's fixed device-memory budget, a service loop that must not call cudaMalloc because it stalls the whole
device, a process whose framework forbids allocations it does not see.  cetra_resample is closed to them because it
wants a workspace; cetra_resample_static keeps its FP64 sums in a 4 MiB array built into the library instead and
accepts at most cetra_resample_static_max_points() = 262 144 output points (light curves x grid points) per call.

What is checked here: the new entry point gives what cetra_resample gives, within the tolerance the resampling
tests use (test_setup_steps.py: identical null pattern, 2^-23 relative for float32 and 1e-13 for float64, because
the FP64 atomic sums may be added in a different order), on two calls in a row.  The second call is a different,
smaller problem laid over the part of the built-in array that the first call left full of its own sums, so a call
that forgot to clear its scratch would fail it; a third call repeats the first.  Requests beyond the limit must be
refused with CETRA_ERR_STATIC_LIMIT and leave the outputs untouched.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here
must not hide the parity tests.  It passes run alone in a fresh process (its first call is then the one that looks
the array up on the device) and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest


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


def test_static_limit_is_reported_before_any_device_work(cetra):
    """Host-side contract (runs without a GPU): the limit is the documented one, and a request beyond it, or a
    malformed one, is turned away before the library touches the device."""
    lib = cetra.load_library()
    limit = cetra.cetra_resample_static_max_points()
    assert limit == 262144
    assert cetra.status_string(cetra.CETRA_ERR_STATIC_LIMIT) not in ("ok", "unknown status")
    fake = 0x1000                                  # never dereferenced: these calls fail before any launch
    args = lambda n_lc, n_out, cadence=1.0: (fake, fake, fake, 0, 10, n_lc, 0.0, cadence, n_out, fake, fake, None)
    assert lib.cetra_resample_static(*args(1, limit + 1)) == cetra.CETRA_ERR_STATIC_LIMIT
    assert lib.cetra_resample_static(*args(2, limit // 2 + 1)) == cetra.CETRA_ERR_STATIC_LIMIT
    assert lib.cetra_resample_static(*args(2 ** 31 - 1, 2 ** 40)) == cetra.CETRA_ERR_STATIC_LIMIT     # no overflow
    assert lib.cetra_resample_static(*args(1, 10, cadence=-1.0)) == cetra.CETRA_ERR_INVALID_ARG
    assert lib.cetra_resample_static(*args(0, 10)) == cetra.CETRA_ERR_INVALID_ARG


def _problem(cetra, torch, seed, n_lc, n, dtype, cad_factor):
    from cetra_synth import make_irregular_batch
    t, f, e = make_irregular_batch(seed=seed, n_lc=n_lc, n=n, dtype=np.dtype(dtype))
    t_start, c, n_out = cetra.cetra_resample_grid(t, cad_factor * cetra.cetra_median_cadence(t), 0.2)
    return (torch.from_numpy(t).cuda(), torch.from_numpy(f).cuda(), torch.from_numpy(e).cuda(), t_start, c, n_out)


def _same(torch, got, want, dtype):
    eps = 2.0 ** -23 if dtype == "float32" else 1e-13      # the resampling tests' tolerance (test_setup_steps.py)
    for g, w in zip(got, want):
        g, w = g.cpu().numpy(), w.cpu().numpy()
        assert g.shape == w.shape and g.dtype == w.dtype
        null = np.isnan(w) | np.isinf(w)
        assert np.array_equal(np.isnan(g), np.isnan(w)) and np.array_equal(np.isinf(g), np.isinf(w))
        assert np.allclose(g[~null], w[~null], rtol=eps, atol=0)
        assert np.any(~null) and np.any(null)               # the case has both data points and null points


@pytest.mark.gpu
def test_resample_static_equals_resample_on_consecutive_calls(torch_cuda, cetra):
    torch = torch_cuda
    first = _problem(cetra, torch, 250320881, 3, 6000, "float32", 1.0)
    second = _problem(cetra, torch, 250320882, 2, 2500, "float64", 2.5)     # smaller: sits on the first call's leftovers
    assert second[5] * 2 < first[5] * 3 <= cetra.cetra_resample_static_max_points()
    want_first = cetra.cetra_resample(*first)
    want_second = cetra.cetra_resample(*second)
    torch.cuda.synchronize()

    launches = cetra.cetra_kernel_launch_count()
    # the caller's own output buffers, as a caller without an allocator would pass them
    out1 = (torch.empty((3, first[5]), dtype=torch.float32, device="cuda"),
            torch.empty((3, first[5]), dtype=torch.float32, device="cuda"))
    got_first = cetra.cetra_resample_static(*first, out=out1)
    got_second = cetra.cetra_resample_static(*second)                       # straight after, same stream
    torch.cuda.synchronize()
    assert got_first[0] is out1[0] and got_first[1] is out1[1]
    assert cetra.cetra_kernel_launch_count() - launches == 4                # accumulate + finalize, twice
    _same(torch, got_first, want_first, "float32")
    _same(torch, got_second, want_second, "float64")

    keep = [o.clone() for o in out1]
    again = cetra.cetra_resample_static(*first)                             # after the smaller call: all cleared again
    torch.cuda.synchronize()
    _same(torch, again, want_first, "float32")
    _same(torch, again, keep, "float32")

    # a single light curve given as a 1-D tensor comes back 1-D, like cetra_resample
    one = cetra.cetra_resample_static(first[0], first[1][1], first[2][1], *first[3:])
    torch.cuda.synchronize()
    assert one[0].dim() == 1
    _same(torch, one, (want_first[0][1], want_first[1][1]), "float32")


@pytest.mark.gpu
def test_resample_static_refuses_what_does_not_fit(torch_cuda, cetra):
    torch = torch_cuda
    limit = cetra.cetra_resample_static_max_points()
    t = torch.linspace(0.0, 10.0, 500, dtype=torch.float64, device="cuda")
    f = torch.ones((2, 500), dtype=torch.float32, device="cuda")
    e = torch.full((2, 500), 1e-3, dtype=torch.float32, device="cuda")
    n_out = limit // 2 + 1
    out = (torch.full((2, n_out), 7.0, dtype=torch.float32, device="cuda"),
           torch.full((2, n_out), 7.0, dtype=torch.float32, device="cuda"))
    launches = cetra.cetra_kernel_launch_count()
    with pytest.raises(cetra.CetraError) as err:
        cetra.cetra_resample_static(t, f, e, 0.0, 10.0 / n_out, n_out, out=out)
    assert err.value.status == cetra.CETRA_ERR_STATIC_LIMIT and "built-in scratch" in str(err.value)
    torch.cuda.synchronize()
    assert cetra.cetra_kernel_launch_count() == launches
    assert bool((out[0] == 7.0).all()) and bool((out[1] == 7.0).all())      # nothing was enqueued
    # exactly at the limit it runs, and agrees with the workspace path
    n_fit = limit // 2
    got = cetra.cetra_resample_static(t, f, e, 0.0, 10.0 / n_fit, n_fit)
    want = cetra.cetra_resample(t, f, e, 0.0, 10.0 / n_fit, n_fit)
    torch.cuda.synchronize()
    _same(torch, got, want, "float32")

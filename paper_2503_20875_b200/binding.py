"""ctypes binding of libcetra_b200.so (include/cetra.h) -- argument marshalling only.

Every function has the name of the C entry point it calls.  Device arrays are torch CUDA tensors
(PyTorch is used for device memory and streams only); small grids are numpy/host arrays.  All the
arithmetic of the path runs in the CUDA kernels; there is no CPU fallback: if the library cannot be
loaded, or no CUDA device is present, the compute calls raise.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

from . import build as _build

CETRA_OK = 0
CETRA_ERR_INVALID_ARG = -1
CETRA_ERR_NONUNIFORM_TIMES = -2
CETRA_ERR_UNSUPPORTED = -3
CETRA_ERR_WORKSPACE = -4
CETRA_ERR_CUDA = -5
CETRA_ERR_STATIC_LIMIT = -6
CETRA_F32, CETRA_F64 = 0, 1
CETRA_MAX_DURATIONS = 128

# Every symbol include/cetra.h declares (tests check that the library exports each of them).
EXPORTED_SYMBOLS = (
    "cetra_status_string", "cetra_device_info", "cetra_stats_pitch", "cetra_kernel_launch_count",
    "cetra_linear_workspace_bytes", "cetra_linear_search", "cetra_exact_eval_count",
    "cetra_periodic_workspace_bytes", "cetra_periodic_search", "cetra_periodic_search_stats",
    "cetra_search_batched_workspace_bytes", "cetra_search_batched", "cetra_search_batched_templates",
    "cetra_search_batched_templates_workspace_bytes",
    "cetra_search_batched_host_workspace_bytes", "cetra_search_batched_host",
    "cetra_profile_enable", "cetra_profile_read",
    "cetra_resample_template", "cetra_median_cadence", "cetra_resample_grid", "cetra_resample_workspace_bytes", "cetra_resample",
    "cetra_resample_static_max_points", "cetra_resample_static", "cetra_test_fold_override",
    "cetra_monotransit_workspace_bytes", "cetra_monotransit_search",
    "cetra_mask_workspace_bytes", "cetra_mask_transits",
)


# The probes of include/cetra_diag.h, exported by libcetra_diag.so only.
DIAG_SYMBOLS = ("cetra_peak_probe_workspace_bytes", "cetra_peak_probe",
                "cetra_tc_correlation_probe_workspace_bytes", "cetra_tc_correlation_probe")


class CetraError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {status_string(status)} (status {status})")


class cetra_t0_grid(ctypes.Structure):
    _fields_ = [("t0_start", ctypes.c_double), ("t0_stride", ctypes.c_double), ("n_t0", ctypes.c_int64)]


class cetra_peak(ctypes.Structure):
    _fields_ = [("lr", ctypes.c_float), ("depth", ctypes.c_float), ("depth_var", ctypes.c_float),
                ("t0", ctypes.c_float), ("i_t0", ctypes.c_int32), ("j_dur", ctypes.c_int32),
                ("n_transits", ctypes.c_int32), ("reserved", ctypes.c_int32)]


PEAK_DTYPE = np.dtype([("lr", "<f4"), ("depth", "<f4"), ("depth_var", "<f4"), ("t0", "<f4"),
                       ("i_t0", "<i4"), ("j_dur", "<i4"), ("n_transits", "<i4"), ("reserved", "<i4")])
assert PEAK_DTYPE.itemsize == ctypes.sizeof(cetra_peak) == 32


class cetra_event(ctypes.Structure):
    _fields_ = [("lr", ctypes.c_float), ("depth", ctypes.c_float), ("depth_var", ctypes.c_float),
                ("t0", ctypes.c_float), ("i_t0", ctypes.c_int32), ("j_dur", ctypes.c_int32),
                ("reserved", ctypes.c_int32 * 2)]


EVENT_DTYPE = np.dtype([("lr", "<f4"), ("depth", "<f4"), ("depth_var", "<f4"), ("t0", "<f4"),
                        ("i_t0", "<i4"), ("j_dur", "<i4"), ("reserved", "<i4", (2,))])
assert EVENT_DTYPE.itemsize == ctypes.sizeof(cetra_event) == 32

_lib: Optional[ctypes.CDLL] = None


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree library (building it with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB_PATH
    if not os.path.exists(path) or os.environ.get("CETRA_REBUILD") == "1" or (_build.stale() and _build.have_nvcc()):
        path = _build.build(force=os.environ.get("CETRA_REBUILD") == "1")
    lib = ctypes.CDLL(path)
    vp, dp, fp, ip = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_void_p, ctypes.c_void_p
    i32, i64, sz = ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t
    lib.cetra_status_string.restype = ctypes.c_char_p
    lib.cetra_status_string.argtypes = [ctypes.c_int]
    lib.cetra_device_info.restype = ctypes.c_int
    lib.cetra_device_info.argtypes = [ctypes.POINTER(i32), ctypes.POINTER(i32)]
    lib.cetra_stats_pitch.restype = i64
    lib.cetra_stats_pitch.argtypes = [i64]
    lib.cetra_kernel_launch_count.restype = i64
    lib.cetra_kernel_launch_count.argtypes = []
    lib.cetra_exact_eval_count.restype = ctypes.c_int
    lib.cetra_exact_eval_count.argtypes = [ctypes.POINTER(i64), i32]
    lib.cetra_linear_workspace_bytes.restype = sz
    lib.cetra_linear_workspace_bytes.argtypes = [dp, i64, i32, dp, i32, cetra_t0_grid, i32]
    lib.cetra_linear_search.restype = ctypes.c_int
    lib.cetra_linear_search.argtypes = [dp, vp, vp, ctypes.c_int, i64, i32, dp, i32, cetra_t0_grid, fp, i32,
                                        vp, vp, vp, vp, vp, sz, vp]
    lib.cetra_periodic_workspace_bytes.restype = sz
    lib.cetra_periodic_workspace_bytes.argtypes = [i32, i32, cetra_t0_grid, i32]
    lib.cetra_periodic_search.restype = ctypes.c_int
    lib.cetra_periodic_search.argtypes = [vp, vp, vp, i32, i32, cetra_t0_grid, dp, dp, i32, ip, ip, vp, vp, sz, vp]
    lib.cetra_periodic_search_stats.restype = ctypes.c_int
    lib.cetra_periodic_search_stats.argtypes = [vp, i32, i32, cetra_t0_grid, dp, dp, i32, ip, ip, vp, vp, sz, vp]
    lib.cetra_search_batched_workspace_bytes.restype = sz
    lib.cetra_search_batched_workspace_bytes.argtypes = [dp, i64, i32, i32, dp, i32, cetra_t0_grid, i32, i32]
    lib.cetra_search_batched.restype = ctypes.c_int
    lib.cetra_search_batched.argtypes = [dp, vp, vp, ctypes.c_int, i64, i32, i32, dp, i32, cetra_t0_grid, fp, i32,
                                         dp, i32, ip, ip, vp, vp, sz, vp]
    lib.cetra_search_batched_templates_workspace_bytes.restype = sz
    lib.cetra_search_batched_templates_workspace_bytes.argtypes = [dp, i64, i32, i32, dp, i32, cetra_t0_grid, i32, i32, i32]
    lib.cetra_search_batched_templates.restype = ctypes.c_int
    lib.cetra_search_batched_templates.argtypes = [dp, vp, vp, ctypes.c_int, i64, i32, i32, dp, i32, cetra_t0_grid, fp,
                                                   i32, i32, dp, i32, ip, ip, vp, vp, sz, vp]
    lib.cetra_search_batched_host_workspace_bytes.restype = sz
    lib.cetra_search_batched_host_workspace_bytes.argtypes = [dp, i64, i32, i32, ctypes.c_int, dp, i32,
                                                              cetra_t0_grid, i32, i32]
    lib.cetra_search_batched_host.restype = ctypes.c_int
    lib.cetra_search_batched_host.argtypes = [dp, vp, vp, ctypes.c_int, i64, i32, i32, dp, i32, cetra_t0_grid, fp,
                                              i32, dp, i32, ip, ip, vp, vp, sz, vp]
    lib.cetra_median_cadence.restype = ctypes.c_int
    lib.cetra_median_cadence.argtypes = [dp, i64, dp]
    lib.cetra_resample_grid.restype = ctypes.c_int
    lib.cetra_resample_grid.argtypes = [dp, i64, ctypes.c_double, ctypes.c_double, dp, dp, ctypes.POINTER(i64)]
    lib.cetra_resample_workspace_bytes.restype = sz
    lib.cetra_resample_workspace_bytes.argtypes = [i64, i32, i64]
    lib.cetra_resample.restype = ctypes.c_int
    lib.cetra_resample.argtypes = [vp, vp, vp, ctypes.c_int, i64, i32, ctypes.c_double, ctypes.c_double, i64,
                                   vp, vp, vp, sz, vp]
    lib.cetra_resample_static_max_points.restype = i64
    lib.cetra_resample_static_max_points.argtypes = []
    lib.cetra_resample_static.restype = ctypes.c_int
    lib.cetra_resample_static.argtypes = [vp, vp, vp, ctypes.c_int, i64, i32, ctypes.c_double, ctypes.c_double, i64,
                                          vp, vp, vp]
    lib.cetra_monotransit_workspace_bytes.restype = sz
    lib.cetra_monotransit_workspace_bytes.argtypes = [i32, i64]
    lib.cetra_monotransit_search.restype = ctypes.c_int
    lib.cetra_monotransit_search.argtypes = [vp, vp, vp, i32, i32, cetra_t0_grid, dp, i32, ctypes.c_double,
                                             vp, vp, vp, vp, vp, sz, vp]
    lib.cetra_mask_workspace_bytes.restype = sz
    lib.cetra_mask_workspace_bytes.argtypes = [i32]
    lib.cetra_mask_transits.restype = ctypes.c_int
    lib.cetra_mask_transits.argtypes = [vp, vp, ctypes.c_int, i64, i32, dp, dp, dp, ctypes.c_double, vp, vp, sz, vp]
    lib.cetra_test_fold_override.restype = None
    lib.cetra_test_fold_override.argtypes = [i32, i32]
    lib.cetra_profile_enable.restype = ctypes.c_int
    lib.cetra_profile_enable.argtypes = [i32]
    lib.cetra_profile_read.restype = ctypes.c_int
    lib.cetra_profile_read.argtypes = [dp, ctypes.POINTER(i64), dp, ctypes.POINTER(i64), i32]
    _lib = lib
    return lib


_diag: Optional[ctypes.CDLL] = None


def load_diag_library() -> ctypes.CDLL:
    """dlopen libcetra_diag.so, the measurement probes (include/cetra_diag.h); built on demand like the product."""
    global _diag
    if _diag is not None:
        return _diag
    path = _build.DIAG_LIB_PATH
    if not os.path.exists(path) or (_build.stale(path) and _build.have_nvcc()):
        path = _build.build_diag()
    lib = ctypes.CDLL(path)
    vp, dp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double)
    i32, sz = ctypes.c_int32, ctypes.c_size_t
    lib.cetra_peak_probe_workspace_bytes.restype = sz
    lib.cetra_peak_probe_workspace_bytes.argtypes = []
    lib.cetra_peak_probe.restype = ctypes.c_int
    lib.cetra_peak_probe.argtypes = [i32, i32, dp, dp, vp, sz, vp]
    _diag = lib
    return lib


def status_string(status: int) -> str:
    return load_library().cetra_status_string(int(status)).decode()


def _check(status: int, where: str) -> None:
    if status != CETRA_OK:
        raise CetraError(status, where)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _opt_i32(a):
    if a is None:
        return None, None
    arr = np.ascontiguousarray(a, dtype=np.int32)
    return arr, arr.ctypes.data


def _grid(t0_start: float, t0_stride: float, n_t0: int) -> cetra_t0_grid:
    return cetra_t0_grid(float(t0_start), float(t0_stride), int(n_t0))


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2503_20875_b200 needs a CUDA device: there is no CPU fallback")
    return torch


def _on_stream(fn):
    """Run a wrapper with `stream` as torch's current stream: the implicit workspace, the output tensors and any
    `.contiguous()` copy of an input are then allocated and produced on the stream the kernels are enqueued on, and
    the caching allocator ties their lifetime to that stream (a workspace freed on return is not handed to a tensor
    of another stream while the kernels still use it).  Inputs produced on a different stream are the caller's to
    order, as everywhere in torch."""
    import functools
    import inspect
    sig = inspect.signature(fn)

    @functools.wraps(fn)
    def wrapper(*args, **kwargs):
        stream = sig.bind_partial(*args, **kwargs).arguments.get("stream")
        if stream is None:
            return fn(*args, **kwargs)
        import torch
        with torch.cuda.stream(stream):
            return fn(*args, **kwargs)
    return wrapper


def _stream_ptr(torch, stream) -> int:
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def _dtype_code(torch, t) -> int:
    if t.dtype == torch.float32:
        return CETRA_F32
    if t.dtype == torch.float64:
        return CETRA_F64
    raise TypeError(f"flux must be float32 or float64, got {t.dtype}")


def _dev_input(torch, flux, flux_err):
    if not (flux.is_cuda and flux_err.is_cuda):
        raise TypeError("flux and flux_err must be CUDA tensors")
    if flux.dtype != flux_err.dtype or flux.shape != flux_err.shape:
        raise TypeError("flux and flux_err must have the same dtype and shape")
    flux, flux_err = flux.contiguous(), flux_err.contiguous()
    if flux.dim() == 1:
        n_lc, n = 1, flux.shape[0]
    elif flux.dim() == 2:
        n_lc, n = flux.shape
    else:
        raise TypeError("flux must be [N] or [B][N]")
    return flux, flux_err, int(n_lc), int(n)


def _workspace(torch, nbytes: int, device, workspace=None):
    if workspace is not None:
        if workspace.dtype != torch.uint8 or not workspace.is_cuda or workspace.numel() < nbytes:
            raise CetraError(CETRA_ERR_WORKSPACE, "workspace")
        return workspace
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)


def cetra_device_info():
    lib = load_library()
    a, b = ctypes.c_int32(), ctypes.c_int32()
    _check(lib.cetra_device_info(ctypes.byref(a), ctypes.byref(b)), "cetra_device_info")
    return a.value, b.value


def cetra_stats_pitch(n_t0: int) -> int:
    return int(load_library().cetra_stats_pitch(int(n_t0)))


def cetra_kernel_launch_count() -> int:
    return int(load_library().cetra_kernel_launch_count())


def cetra_exact_eval_count(reset: bool = False) -> int:
    """Exact (R25) evaluations done by the off-grid linear search since the last reset (synchronises)."""
    v = ctypes.c_int64()
    _check(load_library().cetra_exact_eval_count(ctypes.byref(v), 1 if reset else 0), "cetra_exact_eval_count")
    return int(v.value)


def cetra_profile_enable(enable: bool) -> None:
    _check(load_library().cetra_profile_enable(1 if enable else 0), "cetra_profile_enable")


def cetra_profile_read(reset: bool = True):
    """{'linear_ms', 'linear_launches', 'fold_ms', 'fold_launches'} since the last reset (waits for the events)."""
    lm, fm = ctypes.c_double(), ctypes.c_double()
    ll, fl = ctypes.c_int64(), ctypes.c_int64()
    _check(load_library().cetra_profile_read(ctypes.byref(lm), ctypes.byref(ll), ctypes.byref(fm), ctypes.byref(fl),
                                             1 if reset else 0), "cetra_profile_read")
    return dict(linear_ms=lm.value, linear_launches=ll.value, fold_ms=fm.value, fold_launches=fl.value)


CETRA_PROBE_FFMA2, CETRA_PROBE_FADD2, CETRA_PROBE_LDS64 = 0, 1, 2


@_on_stream
def cetra_peak_probe(kind: int, iters: int = 20000, stream=None):
    """(units per clock per SM, units per second) of one of the probed instructions; synchronises the stream.
    A probe of libcetra_diag.so (include/cetra_diag.h), not of the product library."""
    torch = _torch()
    lib = load_diag_library()
    nbytes = int(lib.cetra_peak_probe_workspace_bytes())
    ws = _workspace(torch, nbytes, torch.device("cuda", torch.cuda.current_device()))
    a, b = ctypes.c_double(), ctypes.c_double()
    _check(lib.cetra_peak_probe(int(kind), int(iters), ctypes.byref(a), ctypes.byref(b), ws.data_ptr(), ws.numel(),
                                _stream_ptr(torch, stream)), "cetra_peak_probe")
    return a.value, b.value


@_on_stream
def cetra_tc_correlation_probe(n_out: int, n_taps: int, split: bool = True, reps: int = 20, stream=None):
    """The measured tensor-core variant of the windowed sums (cetra_diag.h): dict(ms, evals_per_s, err_wmf, err_wmm)."""
    torch = _torch()
    lib = load_diag_library()
    lib.cetra_tc_correlation_probe_workspace_bytes.restype = ctypes.c_size_t
    lib.cetra_tc_correlation_probe_workspace_bytes.argtypes = [ctypes.c_int64, ctypes.c_int32]
    lib.cetra_tc_correlation_probe.restype = ctypes.c_int
    lib.cetra_tc_correlation_probe.argtypes = [ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                               ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double),
                                               ctypes.POINTER(ctypes.c_double), ctypes.c_void_p, ctypes.c_size_t,
                                               ctypes.c_void_p]
    nbytes = int(lib.cetra_tc_correlation_probe_workspace_bytes(int(n_out), int(n_taps)))
    ws = _workspace(torch, nbytes, torch.device("cuda", torch.cuda.current_device()))
    ms, ef, ew = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _check(lib.cetra_tc_correlation_probe(int(n_out), int(n_taps), 1 if split else 0, int(reps), ctypes.byref(ms),
                                          ctypes.byref(ef), ctypes.byref(ew), ws.data_ptr(), ws.numel(),
                                          _stream_ptr(torch, stream)), "cetra_tc_correlation_probe")
    return dict(ms=ms.value, evals_per_s=float(n_out) * n_taps / (ms.value * 1e-3), err_wmf=ef.value, err_wmm=ew.value)


def cetra_test_fold_override(force_stream: bool = False, stage_cells: int = 0) -> None:
    """Test hook (include/cetra.h): make every later periodic search of this process use the streamed fold kernel
    and/or small stages; called without arguments it restores the library's own plan."""
    load_library().cetra_test_fold_override(1 if force_stream else 0, int(stage_cells))


def cetra_linear_workspace_bytes(times, n_lc: int, durations, t0_start, t0_stride, n_t0, n_template: int) -> int:
    lib = load_library()
    times, durations = _f64(times), _f64(durations)
    return int(lib.cetra_linear_workspace_bytes(_dp(times), times.shape[0], int(n_lc), _dp(durations),
                                                durations.shape[0], _grid(t0_start, t0_stride, n_t0),
                                                int(n_template)))


@dataclass
class LinearResult:
    """Outputs of cetra_linear_search: float32 CUDA tensors [B][J][I] (or [J][I] for a 1-D input)."""
    depth: object
    depth_var: object
    dlogL: object
    stats: object          # [B][J][pitch][2] (S_wmm, S_wmf) or None


@_on_stream
def cetra_linear_search(times, flux, flux_err, durations, t0_start: float, t0_stride: float, n_t0: int, template,
                        want_grids: bool = True, want_stats: bool = False, workspace=None,
                        stream=None) -> LinearResult:
    torch = _torch()
    lib = load_library()
    flux, flux_err, n_lc, n = _dev_input(torch, flux, flux_err)
    squeeze = flux.dim() == 1
    times, durations = _f64(times), _f64(durations)
    tpl = np.ascontiguousarray(template, dtype=np.float32)
    if times.shape[0] != n:
        raise CetraError(CETRA_ERR_INVALID_ARG, "cetra_linear_search: len(times) != flux.shape[-1]")
    grid = _grid(t0_start, t0_stride, n_t0)
    n_dur = durations.shape[0]
    nbytes = int(lib.cetra_linear_workspace_bytes(_dp(times), n, n_lc, _dp(durations), n_dur, grid, tpl.shape[0]))
    if nbytes == 0:
        # let the entry point report the precise status
        nbytes = 256
    ws = _workspace(torch, nbytes, flux.device, workspace)
    dev = flux.device
    depth = var = dl = stats = None
    if want_grids:
        depth = torch.empty((n_lc, n_dur, n_t0), dtype=torch.float32, device=dev)
        var = torch.empty_like(depth)
        dl = torch.empty_like(depth)
    if want_stats:
        stats = torch.empty((n_lc, n_dur, cetra_stats_pitch(n_t0), 2), dtype=torch.float32, device=dev)
    ptr = lambda t: t.data_ptr() if t is not None else None
    with torch.cuda.device(dev):
        rc = lib.cetra_linear_search(_dp(times), flux.data_ptr(), flux_err.data_ptr(), _dtype_code(torch, flux), n,
                                     n_lc, _dp(durations), n_dur, grid, tpl.ctypes.data, tpl.shape[0], ptr(depth),
                                     ptr(var), ptr(dl), ptr(stats), ws.data_ptr(), ws.numel(),
                                     _stream_ptr(torch, stream))
    _check(rc, "cetra_linear_search")
    if squeeze and want_grids:
        depth, var, dl = depth[0], var[0], dl[0]
    return LinearResult(depth, var, dl, stats)


def cetra_periodic_workspace_bytes(n_lc: int, n_dur: int, t0_start, t0_stride, n_t0, n_per: int) -> int:
    return int(load_library().cetra_periodic_workspace_bytes(int(n_lc), int(n_dur), _grid(t0_start, t0_stride, n_t0),
                                                             int(n_per)))


def _peaks_tensor(torch, n_lc: int, n_per: int, device):
    return torch.empty((n_lc, n_per, 8), dtype=torch.int32, device=device)


def peaks_to_numpy(peaks) -> np.ndarray:
    """[B][K][8] int32 tensor of cetra_peak records -> numpy structured array [B][K] (PEAK_DTYPE)."""
    arr = peaks.detach().cpu().numpy()
    return np.ascontiguousarray(arr).view(PEAK_DTYPE).reshape(arr.shape[:-1])


@_on_stream
def cetra_periodic_search(depth, depth_var, dlogL, t0_start: float, t0_stride: float, durations, periods,
                          dur_lo=None, dur_hi=None, workspace=None, stream=None):
    """Returns a CUDA int32 tensor [B][K][8] holding cetra_peak records (see peaks_to_numpy)."""
    torch = _torch()
    lib = load_library()
    for t in (depth, depth_var, dlogL):
        if t is not None and (not t.is_cuda or t.dtype != torch.float32):
            raise TypeError("linear-search grids must be float32 CUDA tensors")
    depth, depth_var = depth.contiguous(), depth_var.contiguous()
    dlogL = dlogL.contiguous() if dlogL is not None else None      # None: LR_e = 1/2 depth^2/var (cetra.h)
    if depth.dim() == 2:
        n_lc, (n_dur, n_t0) = 1, depth.shape
    else:
        n_lc, n_dur, n_t0 = depth.shape
    durations, periods = _f64(durations), _f64(periods)
    lo_arr, lo = _opt_i32(dur_lo)
    hi_arr, hi = _opt_i32(dur_hi)
    grid = _grid(t0_start, t0_stride, n_t0)
    n_per = periods.shape[0]
    nbytes = int(lib.cetra_periodic_workspace_bytes(n_lc, n_dur, grid, n_per))
    ws = _workspace(torch, nbytes, depth.device, workspace)
    peaks = _peaks_tensor(torch, n_lc, n_per, depth.device)
    with torch.cuda.device(depth.device):
        rc = lib.cetra_periodic_search(depth.data_ptr(), depth_var.data_ptr(),
                                       dlogL.data_ptr() if dlogL is not None else None, n_lc, n_dur, grid,
                                       _dp(durations), _dp(periods), n_per, lo, hi, peaks.data_ptr(), ws.data_ptr(),
                                       ws.numel(), _stream_ptr(torch, stream))
    _check(rc, "cetra_periodic_search")
    return peaks


@_on_stream
def cetra_periodic_search_stats(stats, n_t0: int, t0_start: float, t0_stride: float, durations, periods,
                                dur_lo=None, dur_hi=None, workspace=None, stream=None):
    torch = _torch()
    lib = load_library()
    if not stats.is_cuda or stats.dtype != torch.float32 or stats.dim() != 4 or stats.shape[-1] != 2:
        raise TypeError("stats must be a float32 CUDA tensor [B][J][pitch][2]")
    stats = stats.contiguous()
    n_lc, n_dur, pitch, _ = stats.shape
    if pitch != cetra_stats_pitch(n_t0):
        raise CetraError(CETRA_ERR_INVALID_ARG, "cetra_periodic_search_stats: wrong row pitch")
    durations, periods = _f64(durations), _f64(periods)
    lo_arr, lo = _opt_i32(dur_lo)
    hi_arr, hi = _opt_i32(dur_hi)
    grid = _grid(t0_start, t0_stride, n_t0)
    n_per = periods.shape[0]
    nbytes = int(lib.cetra_periodic_workspace_bytes(n_lc, n_dur, grid, n_per))
    ws = _workspace(torch, nbytes, stats.device, workspace)
    peaks = _peaks_tensor(torch, n_lc, n_per, stats.device)
    with torch.cuda.device(stats.device):
        rc = lib.cetra_periodic_search_stats(stats.data_ptr(), n_lc, n_dur, grid, _dp(durations), _dp(periods), n_per,
                                             lo, hi, peaks.data_ptr(), ws.data_ptr(), ws.numel(),
                                             _stream_ptr(torch, stream))
    _check(rc, "cetra_periodic_search_stats")
    return peaks


def cetra_search_batched_workspace_bytes(times, n_lc: int, lc_chunk: int, durations, t0_start, t0_stride, n_t0,
                                         n_template: int, n_per: int) -> int:
    lib = load_library()
    times, durations = _f64(times), _f64(durations)
    return int(lib.cetra_search_batched_workspace_bytes(_dp(times), times.shape[0], int(n_lc), int(lc_chunk),
                                                        _dp(durations), durations.shape[0],
                                                        _grid(t0_start, t0_stride, n_t0), int(n_template), int(n_per)))


@_on_stream
def cetra_search_batched(times, flux, flux_err, durations, t0_start: float, t0_stride: float, n_t0: int, template,
                         periods, dur_lo=None, dur_hi=None, lc_chunk: int = 0, workspace=None, peaks=None,
                         stream=None):
    """Linear + periodic search of [B][N] device light curves sharing `times`; returns peaks [B][K][8] int32."""
    torch = _torch()
    lib = load_library()
    flux, flux_err, n_lc, n = _dev_input(torch, flux, flux_err)
    times, durations, periods = _f64(times), _f64(durations), _f64(periods)
    tpl = np.ascontiguousarray(template, dtype=np.float32)
    if times.shape[0] != n:
        raise CetraError(CETRA_ERR_INVALID_ARG, "cetra_search_batched: len(times) != flux.shape[-1]")
    lo_arr, lo = _opt_i32(dur_lo)
    hi_arr, hi = _opt_i32(dur_hi)
    grid = _grid(t0_start, t0_stride, n_t0)
    n_dur, n_per = durations.shape[0], periods.shape[0]
    nbytes = int(lib.cetra_search_batched_workspace_bytes(_dp(times), n, n_lc, int(lc_chunk), _dp(durations), n_dur,
                                                          grid, tpl.shape[0], n_per))
    ws = _workspace(torch, nbytes, flux.device, workspace)
    if peaks is None:
        peaks = _peaks_tensor(torch, n_lc, n_per, flux.device)
    with torch.cuda.device(flux.device):
        rc = lib.cetra_search_batched(_dp(times), flux.data_ptr(), flux_err.data_ptr(), _dtype_code(torch, flux), n,
                                      n_lc, int(lc_chunk), _dp(durations), n_dur, grid, tpl.ctypes.data, tpl.shape[0],
                                      _dp(periods), n_per, lo, hi, peaks.data_ptr(), ws.data_ptr(), ws.numel(),
                                      _stream_ptr(torch, stream))
    _check(rc, "cetra_search_batched")
    return peaks


@_on_stream
def cetra_search_batched_templates(times, flux, flux_err, durations, t0_start: float, t0_stride: float, n_t0: int,
                                   templates, periods, dur_lo=None, dur_hi=None, lc_chunk: int = 0, workspace=None,
                                   stream=None):
    """The batched search for every row of `templates` [T][M]; returns peaks [T][B][K][8] int32."""
    torch = _torch()
    lib = load_library()
    flux, flux_err, n_lc, n = _dev_input(torch, flux, flux_err)
    times, durations, periods = _f64(times), _f64(durations), _f64(periods)
    tpl = np.ascontiguousarray(templates, dtype=np.float32)
    if tpl.ndim != 2:
        raise TypeError("templates must be [T][M]")
    if times.shape[0] != n:
        raise CetraError(CETRA_ERR_INVALID_ARG, "cetra_search_batched_templates: len(times) != flux.shape[-1]")
    lo_arr, lo = _opt_i32(dur_lo)
    hi_arr, hi = _opt_i32(dur_hi)
    grid = _grid(t0_start, t0_stride, n_t0)
    n_dur, n_per = durations.shape[0], periods.shape[0]
    nbytes = int(lib.cetra_search_batched_templates_workspace_bytes(_dp(times), n, n_lc, int(lc_chunk), _dp(durations),
                                                                    n_dur, grid, tpl.shape[1], tpl.shape[0], n_per))
    ws = _workspace(torch, nbytes, flux.device, workspace)
    peaks = torch.empty((tpl.shape[0], n_lc, n_per, 8), dtype=torch.int32, device=flux.device)
    with torch.cuda.device(flux.device):
        rc = lib.cetra_search_batched_templates(_dp(times), flux.data_ptr(), flux_err.data_ptr(),
                                                _dtype_code(torch, flux), n, n_lc, int(lc_chunk), _dp(durations),
                                                n_dur, grid, tpl.ctypes.data, tpl.shape[1], tpl.shape[0],
                                                _dp(periods), n_per, lo, hi, peaks.data_ptr(), ws.data_ptr(),
                                                ws.numel(), _stream_ptr(torch, stream))
    _check(rc, "cetra_search_batched_templates")
    return peaks


def cetra_search_batched_host_workspace_bytes(times, n_lc: int, lc_chunk: int, dtype_code: int, durations, t0_start,
                                              t0_stride, n_t0, n_template: int, n_per: int) -> int:
    lib = load_library()
    times, durations = _f64(times), _f64(durations)
    return int(lib.cetra_search_batched_host_workspace_bytes(_dp(times), times.shape[0], int(n_lc), int(lc_chunk),
                                                             int(dtype_code), _dp(durations), durations.shape[0],
                                                             _grid(t0_start, t0_stride, n_t0), int(n_template),
                                                             int(n_per)))


@_on_stream
def cetra_search_batched_host(times, flux_host, flux_err_host, durations, t0_start: float, t0_stride: float,
                              n_t0: int, template, periods, dur_lo=None, dur_hi=None, lc_chunk: int = 0,
                              workspace=None, peaks_host=None, device=None, stream=None) -> np.ndarray:
    """Same search with HOST light curves (torch CPU tensors, ideally pinned, or numpy arrays) and a HOST
    result: the library copies each chunk in, searches it and copies the records out.  Returns a numpy
    structured array [B][K] of PEAK_DTYPE viewing `peaks_host`."""
    torch = _torch()
    lib = load_library()
    if isinstance(flux_host, np.ndarray):
        flux_host, flux_err_host = torch.from_numpy(flux_host), torch.from_numpy(flux_err_host)
    if flux_host.is_cuda or flux_err_host.is_cuda:
        raise TypeError("cetra_search_batched_host takes host tensors")
    flux_host, flux_err_host = flux_host.contiguous(), flux_err_host.contiguous()
    if flux_host.dtype != flux_err_host.dtype or flux_host.shape != flux_err_host.shape or flux_host.dim() != 2:
        raise TypeError("flux and flux_err must be [B][N] host tensors of one dtype")
    n_lc, n = (int(x) for x in flux_host.shape)
    times, durations, periods = _f64(times), _f64(durations), _f64(periods)
    tpl = np.ascontiguousarray(template, dtype=np.float32)
    if times.shape[0] != n:
        raise CetraError(CETRA_ERR_INVALID_ARG, "cetra_search_batched_host: len(times) != flux.shape[-1]")
    lo_arr, lo = _opt_i32(dur_lo)
    hi_arr, hi = _opt_i32(dur_hi)
    grid = _grid(t0_start, t0_stride, n_t0)
    n_dur, n_per = durations.shape[0], periods.shape[0]
    code = _dtype_code(torch, flux_host)
    dev = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
    nbytes = int(lib.cetra_search_batched_host_workspace_bytes(_dp(times), n, n_lc, int(lc_chunk), code,
                                                               _dp(durations), n_dur, grid, tpl.shape[0], n_per))
    ws = _workspace(torch, nbytes, dev, workspace)
    if peaks_host is None:
        peaks_host = torch.empty((n_lc, n_per, 8), dtype=torch.int32, pin_memory=True)
    with torch.cuda.device(dev):
        rc = lib.cetra_search_batched_host(_dp(times), flux_host.data_ptr(), flux_err_host.data_ptr(), code, n, n_lc,
                                           int(lc_chunk), _dp(durations), n_dur, grid, tpl.ctypes.data, tpl.shape[0],
                                           _dp(periods), n_per, lo, hi, peaks_host.data_ptr(), ws.data_ptr(),
                                           ws.numel(), _stream_ptr(torch, stream))
    _check(rc, "cetra_search_batched_host")
    return peaks_host.numpy().view(PEAK_DTYPE).reshape(n_lc, n_per)


# ----------------------------------------------------------------------- setup and follow-up steps
def cetra_resample_template(model, n_template: int = 1024) -> np.ndarray:
    """Supplied transit model -> n_template-sample search template by linear interpolation; host-side."""
    lib = load_library()
    model = np.ascontiguousarray(model, dtype=np.float32)
    out = np.empty(int(n_template), dtype=np.float32)
    lib.cetra_resample_template.restype = ctypes.c_int
    lib.cetra_resample_template.argtypes = [ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_int32]
    _check(lib.cetra_resample_template(model.ctypes.data, model.shape[0], out.ctypes.data, out.shape[0]),
           "cetra_resample_template")
    return out


def cetra_median_cadence(times) -> float:
    """Default resample cadence: host-only helper of the library."""
    times = _f64(times)
    out = ctypes.c_double()
    _check(load_library().cetra_median_cadence(_dp(times), times.shape[0], ctypes.byref(out)), "cetra_median_cadence")
    return out.value


def cetra_resample_grid(times, cadence: float = 0.0, pad_days: float = 0.0):
    """(t_start, cadence, n_out) of the regular grid for `times`; cadence <= 0: the median."""
    times = _f64(times)
    t_start, c, n_out = ctypes.c_double(), ctypes.c_double(), ctypes.c_int64()
    _check(load_library().cetra_resample_grid(_dp(times), times.shape[0], float(cadence), float(pad_days),
                                              ctypes.byref(t_start), ctypes.byref(c), ctypes.byref(n_out)),
           "cetra_resample_grid")
    return t_start.value, c.value, int(n_out.value)


@_on_stream
def cetra_resample(times_dev, flux, flux_err, t_start: float, cadence: float, n_out: int, workspace=None,
                   stream=None):
    """Irregular light curves [B][N_in] (or [N_in]) sharing `times_dev` -> (flux, flux_err) on the regular grid."""
    torch = _torch()
    lib = load_library()
    flux, flux_err, n_lc, n_in = _dev_input(torch, flux, flux_err)
    squeeze = flux.dim() == 1
    if not (times_dev.is_cuda and times_dev.dtype == torch.float64 and times_dev.numel() == n_in):
        raise TypeError("times_dev must be a float64 CUDA tensor with one entry per observation")
    times_dev = times_dev.contiguous()
    nbytes = int(lib.cetra_resample_workspace_bytes(n_in, n_lc, int(n_out)))
    ws = _workspace(torch, nbytes, flux.device, workspace)
    out_f = torch.empty((n_lc, int(n_out)), dtype=flux.dtype, device=flux.device)
    out_e = torch.empty_like(out_f)
    with torch.cuda.device(flux.device):
        rc = lib.cetra_resample(times_dev.data_ptr(), flux.data_ptr(), flux_err.data_ptr(), _dtype_code(torch, flux),
                                n_in, n_lc, float(t_start), float(cadence), int(n_out), out_f.data_ptr(),
                                out_e.data_ptr(), ws.data_ptr(), ws.numel(), _stream_ptr(torch, stream))
    _check(rc, "cetra_resample")
    return (out_f[0], out_e[0]) if squeeze else (out_f, out_e)


def cetra_resample_static_max_points() -> int:
    """Largest n_lc * n_out one cetra_resample_static call accepts (the size of the library's built-in scratch)."""
    return int(load_library().cetra_resample_static_max_points())


@_on_stream
def cetra_resample_static(times_dev, flux, flux_err, t_start: float, cadence: float, n_out: int, out=None,
                          stream=None):
    """cetra_resample without a workspace, for callers that cannot allocate device memory.

    Same arguments and results as cetra_resample, but the FP64 sums are kept in a 4 MiB array built into the library
    instead of a workspace tensor, so the C call underneath allocates nothing.  It exists for code that is handed
    buffers but no allocator: a stage running inside another program's fixed device-memory budget, a service loop
    where cudaMalloc's device-wide synchronisation is not acceptable, a process whose framework forbids allocations
    it does not see.  Such a caller passes `out=(flux_out, flux_err_out)`, two [B][n_out] (or [n_out]) CUDA tensors
    of the input dtype that it already owns, and then this wrapper allocates nothing either; without `out` the
    wrapper creates the two result tensors with torch, as cetra_resample does.

    Limits and caveats (include/cetra.h has the full text): B * n_out <= cetra_resample_static_max_points()
    (262 144), else CetraError with status CETRA_ERR_STATIC_LIMIT; the first call on each device looks the array up
    and should happen during set-up, before any stream capture; all calls on a device share the array, so calls that
    could overlap on the GPU (unordered streams, threads) must be ordered by the caller.
    """
    torch = _torch()
    lib = load_library()
    flux, flux_err, n_lc, n_in = _dev_input(torch, flux, flux_err)
    squeeze = flux.dim() == 1
    if not (times_dev.is_cuda and times_dev.dtype == torch.float64 and times_dev.numel() == n_in):
        raise TypeError("times_dev must be a float64 CUDA tensor with one entry per observation")
    times_dev = times_dev.contiguous()
    if out is None:
        out_f = torch.empty((n_lc, int(n_out)), dtype=flux.dtype, device=flux.device)
        out_e = torch.empty_like(out_f)
    else:
        out_f, out_e = out
        for o in (out_f, out_e):
            if not (o.is_cuda and o.device == flux.device and o.dtype == flux.dtype and o.is_contiguous()
                    and o.numel() == n_lc * int(n_out)):
                raise TypeError("out must be two contiguous CUDA tensors of the input dtype with B * n_out elements")
    with torch.cuda.device(flux.device):
        rc = lib.cetra_resample_static(times_dev.data_ptr(), flux.data_ptr(), flux_err.data_ptr(),
                                       _dtype_code(torch, flux), n_in, n_lc, float(t_start), float(cadence),
                                       int(n_out), out_f.data_ptr(), out_e.data_ptr(), _stream_ptr(torch, stream))
    _check(rc, "cetra_resample_static")
    if out is not None:
        return out_f, out_e
    return (out_f[0], out_e[0]) if squeeze else (out_f, out_e)


@dataclass
class MonotransitResult:
    """Outputs of cetra_monotransit_search: events [B][n_peaks] records (int32 view, see events_to_numpy),
    n_found [B] int32, optional profile tensors [B][I]."""
    events: object
    n_found: object
    profile_lr: object
    profile_j: object


@_on_stream
def cetra_monotransit_search(depth, depth_var, dlogL, t0_start: float, t0_stride: float, durations, n_peaks: int,
                             excl: float = 1.0, want_profile: bool = False, workspace=None,
                             stream=None) -> MonotransitResult:
    torch = _torch()
    lib = load_library()
    grids = []
    for g in (depth, depth_var, dlogL):
        if not (g.is_cuda and g.dtype == torch.float32):
            raise TypeError("the linear-search grids must be float32 CUDA tensors")
        grids.append(g.contiguous() if g.dim() == 3 else g.contiguous()[None])
    n_lc, n_dur, n_t0 = (int(x) for x in grids[0].shape)
    durations = _f64(durations)
    if durations.shape[0] != n_dur:
        raise CetraError(CETRA_ERR_INVALID_ARG, "cetra_monotransit_search: len(durations) != grids.shape[-2]")
    dev = grids[0].device
    nbytes = int(lib.cetra_monotransit_workspace_bytes(n_lc, n_t0))
    ws = _workspace(torch, nbytes, dev, workspace)
    events = torch.empty((n_lc, int(n_peaks), 8), dtype=torch.int32, device=dev)
    n_found = torch.empty((n_lc,), dtype=torch.int32, device=dev)
    pl = torch.empty((n_lc, n_t0), dtype=torch.float32, device=dev) if want_profile else None
    pj = torch.empty((n_lc, n_t0), dtype=torch.int32, device=dev) if want_profile else None
    ptr = lambda t: t.data_ptr() if t is not None else None
    with torch.cuda.device(dev):
        rc = lib.cetra_monotransit_search(grids[0].data_ptr(), grids[1].data_ptr(), grids[2].data_ptr(), n_lc, n_dur,
                                          _grid(t0_start, t0_stride, n_t0), _dp(durations), int(n_peaks), float(excl),
                                          ptr(pl), ptr(pj), events.data_ptr(), n_found.data_ptr(), ws.data_ptr(),
                                          ws.numel(), _stream_ptr(torch, stream))
    _check(rc, "cetra_monotransit_search")
    return MonotransitResult(events, n_found, pl, pj)


def events_to_numpy(events) -> np.ndarray:
    """[B][n_peaks][8] int32 tensor of cetra_event records -> numpy structured array [B][n_peaks]."""
    a = events.detach().cpu().contiguous().numpy()
    return a.view(EVENT_DTYPE).reshape(a.shape[:-1])


@_on_stream
def cetra_mask_transits(times_dev, flux, period, t0, duration, width: float = 1.0, workspace=None, stream=None):
    """Set the samples within width*D/2 of a transit mid-time to NaN, in place; returns the
    per-curve count of nullified samples as an int32 CUDA tensor."""
    torch = _torch()
    lib = load_library()
    if not (flux.is_cuda and flux.is_contiguous()):
        raise TypeError("flux must be a contiguous CUDA tensor (it is modified in place)")
    n_lc, n = (1, flux.shape[0]) if flux.dim() == 1 else (int(flux.shape[0]), int(flux.shape[1]))
    if not (times_dev.is_cuda and times_dev.dtype == torch.float64 and times_dev.numel() == n):
        raise TypeError("times_dev must be a float64 CUDA tensor with one entry per sample")
    per, tt, dur = (_f64(np.atleast_1d(x)) for x in (period, t0, duration))
    if not (per.shape[0] == tt.shape[0] == dur.shape[0] == n_lc):
        raise CetraError(CETRA_ERR_INVALID_ARG, "cetra_mask_transits: one (period, t0, duration) per light curve")
    nbytes = int(lib.cetra_mask_workspace_bytes(n_lc))
    ws = _workspace(torch, nbytes, flux.device, workspace)
    n_masked = torch.empty((n_lc,), dtype=torch.int32, device=flux.device)
    with torch.cuda.device(flux.device):
        rc = lib.cetra_mask_transits(times_dev.contiguous().data_ptr(), flux.data_ptr(), _dtype_code(torch, flux), n,
                                     n_lc, _dp(per), _dp(tt), _dp(dur), float(width), n_masked.data_ptr(),
                                     ws.data_ptr(), ws.numel(), _stream_ptr(torch, stream))
    _check(rc, "cetra_mask_transits")
    return n_masked

"""CETRA oracle -- TEST INFRASTRUCTURE ONLY (see the header of cetra_oracle.c).

ctypes wrapper around the plain FP64 C oracle.  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs may import this package; the
product (paper_2503_20875_b200) never does, and this package never imports the product.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cetra_oracle.c")
_SRC_SETUP = os.path.join(_HERE, "cetra_oracle_setup.c")
_LIB = os.path.join(_HERE, "libcetra_oracle.so")
_lib: Optional[ctypes.CDLL] = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc.  -ffp-contract=off keeps every FP64 operation a plain IEEE one."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_SETUP))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
               _SRC, _SRC_SETUP, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        lp = ctypes.POINTER(ctypes.c_int64)
        lib.oracle_linear_search.restype = ctypes.c_int
        lib.oracle_linear_search.argtypes = [dp, dp, dp, ctypes.c_int64, dp, ctypes.c_int32,
                                             ctypes.c_double, ctypes.c_double, ctypes.c_int64,
                                             dp, ctypes.c_int32, dp, dp, dp]
        lib.oracle_periodic_search.restype = ctypes.c_int
        lib.oracle_periodic_search.argtypes = [dp, dp, dp, ctypes.c_int32, ctypes.c_int64,
                                               ctypes.c_double, ctypes.c_double, dp, dp, ctypes.c_int32,
                                               ip, ip, dp, dp, lp, ip, dp, dp, ip]
        lib.oracle_periodic_cell.restype = ctypes.c_int
        lib.oracle_periodic_cell.argtypes = [dp, dp, dp, ctypes.c_int32, ctypes.c_int64, ctypes.c_double,
                                             ctypes.c_double, ctypes.c_int32, ctypes.c_int64,
                                             dp, dp, dp, ip]
        lib.oracle_resample_template.restype = ctypes.c_int
        lib.oracle_resample_template.argtypes = [dp, ctypes.c_int32, dp, ctypes.c_int32]
        lib.oracle_median_cadence.restype = ctypes.c_int
        lib.oracle_median_cadence.argtypes = [dp, ctypes.c_int64, dp]
        lib.oracle_resample.restype = ctypes.c_int
        lib.oracle_resample.argtypes = [dp, dp, dp, ctypes.c_int64, ctypes.c_double, ctypes.c_double,
                                        ctypes.c_int64, dp, dp]
        lib.oracle_monotransit.restype = ctypes.c_int
        lib.oracle_monotransit.argtypes = [dp, dp, dp, ctypes.c_int32, ctypes.c_int64, ctypes.c_double, dp,
                                           ctypes.c_int32, ctypes.c_double, dp, ip, lp, ip, dp, dp, dp, ip]
        lib.oracle_mask_transits.restype = ctypes.c_int
        lib.oracle_mask_transits.argtypes = [dp, dp, ctypes.c_int64, ctypes.c_double, ctypes.c_double,
                                             ctypes.c_double, ctypes.c_double, lp]
        lib.oracle_set_threads.argtypes = [ctypes.c_int]
        lib.oracle_force_general.argtypes = [ctypes.c_int]
        lib.oracle_get_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def set_threads(n: int) -> None:
    _load().oracle_set_threads(int(n))


def get_threads() -> int:
    return int(_load().oracle_get_threads())


def _d(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a: np.ndarray, t):
    return a.ctypes.data_as(ctypes.POINTER(t))


@dataclass
class LinearGrids:
    """Outputs of the linear search, each [J][I] float64."""
    depth: np.ndarray
    depth_var: np.ndarray
    dlogL: np.ndarray


@dataclass
class Periodogram:
    """Outputs of the periodic search, one entry per trial period."""
    lr: np.ndarray
    t0: np.ndarray
    i_t0: np.ndarray
    j_dur: np.ndarray
    depth: np.ndarray
    depth_var: np.ndarray
    n_transits: np.ndarray


def linear_search(times, flux, flux_err, durations, t0_start: float, t0_stride: float, n_t0: int,
                  template, force_general: bool = False) -> LinearGrids:
    """t0 grids on the sample grid use the integer-offset form (R3), others the time-difference form (R25);
    force_general evaluates an on-grid t0 grid through the R25 form too (a pin of that form)."""
    lib = _load()
    lib.oracle_force_general(1 if force_general else 0)
    times, flux, flux_err, durations, template = map(_d, (times, flux, flux_err, durations, template))
    n, j = times.shape[0], durations.shape[0]
    depth = np.empty((j, n_t0)); var = np.empty((j, n_t0)); dl = np.empty((j, n_t0))
    c = ctypes.c_double
    rc = lib.oracle_linear_search(_p(times, c), _p(flux, c), _p(flux_err, c), n, _p(durations, c), j,
                                  float(t0_start), float(t0_stride), int(n_t0), _p(template, c),
                                  template.shape[0], _p(depth, c), _p(var, c), _p(dl, c))
    lib.oracle_force_general(0)
    if rc != 0:
        raise ValueError(f"oracle_linear_search failed with status {rc}")
    return LinearGrids(depth, var, dl)


def periodic_search(grids: LinearGrids, t0_start: float, t0_stride: float, durations, periods,
                    dur_lo=None, dur_hi=None) -> Periodogram:
    lib = _load()
    depth, var, dl = _d(grids.depth), _d(grids.depth_var), _d(grids.dlogL)
    durations, periods = _d(durations), _d(periods)
    j, i = depth.shape
    k = periods.shape[0]
    c, i32, i64 = ctypes.c_double, ctypes.c_int32, ctypes.c_int64
    lo = np.ascontiguousarray(dur_lo, dtype=np.int32) if dur_lo is not None else None
    hi = np.ascontiguousarray(dur_hi, dtype=np.int32) if dur_hi is not None else None
    out = Periodogram(np.empty(k), np.empty(k), np.empty(k, np.int64), np.empty(k, np.int32),
                      np.empty(k), np.empty(k), np.empty(k, np.int32))
    rc = lib.oracle_periodic_search(_p(depth, c), _p(var, c), _p(dl, c), j, i, float(t0_start),
                                    float(t0_stride), _p(durations, c), _p(periods, c), k,
                                    _p(lo, i32) if lo is not None else None,
                                    _p(hi, i32) if hi is not None else None,
                                    _p(out.lr, c), _p(out.t0, c), _p(out.i_t0, i64), _p(out.j_dur, i32),
                                    _p(out.depth, c), _p(out.depth_var, c), _p(out.n_transits, i32))
    if rc != 0:
        raise ValueError(f"oracle_periodic_search failed with status {rc}")
    return out


def periodic_cell(grids: LinearGrids, t0_stride: float, period: float, j: int, p: int):
    """(lr, depth, depth_var, n_transits) of one (period, duration, phase) cell; lr is NaN if no epoch contributes."""
    lib = _load()
    depth, var, dl = _d(grids.depth), _d(grids.depth_var), _d(grids.dlogL)
    nj, ni = depth.shape
    c = ctypes.c_double
    lr, z, zv, ntr = c(), c(), c(), ctypes.c_int32()
    rc = lib.oracle_periodic_cell(_p(depth, c), _p(var, c), _p(dl, c), nj, ni, float(t0_stride), float(period),
                                  int(j), int(p), ctypes.byref(lr), ctypes.byref(z), ctypes.byref(zv),
                                  ctypes.byref(ntr))
    if rc != 0:
        raise ValueError(f"oracle_periodic_cell failed with status {rc}")
    return lr.value, z.value, zv.value, ntr.value


# ------------------------------------------------------------------------- setup and follow-up steps
def resample_template(model, n_out: int) -> np.ndarray:
    """Supplied transit model -> n_out-sample template by linear interpolation."""
    lib = _load()
    model = _d(model)
    out = np.empty(int(n_out))
    rc = lib.oracle_resample_template(_p(model, ctypes.c_double), model.shape[0], _p(out, ctypes.c_double), int(n_out))
    if rc != 0:
        raise ValueError(f"oracle_resample_template failed with status {rc}")
    return out


def median_cadence(times) -> float:
    """Default resample cadence: the median cadence of the input (R22)."""
    lib = _load()
    times = _d(times)
    out = ctypes.c_double()
    rc = lib.oracle_median_cadence(_p(times, ctypes.c_double), times.shape[0], ctypes.byref(out))
    if rc != 0:
        raise ValueError(f"oracle_median_cadence failed with status {rc}")
    return out.value


def resample(times, flux, flux_err, t_start: float, cadence: float, n_out: int):
    """Irregular light curve -> regular grid (R21): (flux[n_out], flux_err[n_out])."""
    lib = _load()
    times, flux, flux_err = map(_d, (times, flux, flux_err))
    of, oe = np.empty(n_out), np.empty(n_out)
    c = ctypes.c_double
    rc = lib.oracle_resample(_p(times, c), _p(flux, c), _p(flux_err, c), times.shape[0], float(t_start),
                             float(cadence), int(n_out), _p(of, c), _p(oe, c))
    if rc != 0:
        raise ValueError(f"oracle_resample failed with status {rc}")
    return of, oe


@dataclass
class Monotransits:
    """Single-transit events of the linear-search output (R23)."""
    profile_lr: np.ndarray      # [I] max over durations of dlogL
    profile_j: np.ndarray       # [I] its duration index (-1: every duration null)
    i_t0: np.ndarray            # [n_found]
    j_dur: np.ndarray
    lr: np.ndarray
    depth: np.ndarray
    depth_var: np.ndarray


def monotransit(grids: LinearGrids, t0_stride: float, durations, n_peaks: int, excl: float = 1.0) -> Monotransits:
    lib = _load()
    depth, var, dl = _d(grids.depth), _d(grids.depth_var), _d(grids.dlogL)
    durations = _d(durations)
    nj, ni = depth.shape
    c, i32, i64 = ctypes.c_double, ctypes.c_int32, ctypes.c_int64
    pl, pj = np.empty(ni), np.empty(ni, np.int32)
    ei, ej = np.empty(n_peaks, np.int64), np.empty(n_peaks, np.int32)
    el, ed, ev = np.empty(n_peaks), np.empty(n_peaks), np.empty(n_peaks)
    nf = ctypes.c_int32()
    rc = lib.oracle_monotransit(_p(depth, c), _p(var, c), _p(dl, c), nj, ni, float(t0_stride), _p(durations, c),
                                int(n_peaks), float(excl), _p(pl, c), _p(pj, i32), _p(ei, i64), _p(ej, i32),
                                _p(el, c), _p(ed, c), _p(ev, c), ctypes.byref(nf))
    if rc != 0:
        raise ValueError(f"oracle_monotransit failed with status {rc}")
    n = nf.value
    return Monotransits(pl, pj, ei[:n], ej[:n], el[:n], ed[:n], ev[:n])


def mask_transits(times, flux, period: float, t0: float, duration: float, width: float = 1.0):
    """Copy of `flux` with the samples within width*D/2 of a transit mid-time set to NaN (R24)."""
    lib = _load()
    times = _d(times)
    out = _d(flux).copy()
    cnt = ctypes.c_int64()
    rc = lib.oracle_mask_transits(_p(times, ctypes.c_double), _p(out, ctypes.c_double), times.shape[0],
                                  float(period), float(t0), float(duration), float(width), ctypes.byref(cnt))
    if rc != 0:
        raise ValueError(f"oracle_mask_transits failed with status {rc}")
    return out, cnt.value

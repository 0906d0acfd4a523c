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
_LIB = os.path.join(_HERE, "libcetra_oracle.so")
_lib: Optional[ctypes.CDLL] = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc.  -ffp-contract=off keeps every FP64 operation a plain IEEE one."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
               _SRC, "-o", _LIB, "-lm"]
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
        lib.oracle_set_threads.argtypes = [ctypes.c_int]
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
                  template) -> LinearGrids:
    lib = _load()
    times, flux, flux_err, durations, template = map(_d, (times, flux, flux_err, durations, template))
    n, j = times.shape[0], durations.shape[0]
    depth = np.empty((j, n_t0)); var = np.empty((j, n_t0)); dl = np.empty((j, n_t0))
    c = ctypes.c_double
    rc = lib.oracle_linear_search(_p(times, c), _p(flux, c), _p(flux_err, c), n, _p(durations, c), j,
                                  float(t0_start), float(t0_stride), int(n_t0), _p(template, c),
                                  template.shape[0], _p(depth, c), _p(var, c), _p(dl, c))
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

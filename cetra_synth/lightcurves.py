"""Synthetic TESS-shaped light curves, transit profile table and trial grids.

Everything here is input generation.  Nothing in this file computes any
quantity that the linear or periodic search defines (§2.2-§2.3).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Tuple

import numpy as np

BASE_SEED = 250320875  # arXiv id; per-config seed = BASE_SEED + cfg
DAY_S = 86400.0

CONFIG_NAMES = {
    1: "tiny-1000pt-2min",
    2: "tess-2min-sector",
    3: "tess-20s-sector",
    4: "multi-sector-13x2min",
    5: "survey-batch-2min",
}


# --------------------------------------------------------------------------
# Transit profile (stand-in for the Batman models of PAPER.md:65-69)
# --------------------------------------------------------------------------
def _overlap_area(z: np.ndarray, k: float) -> np.ndarray:
    """Area common to a unit disc and a disc of radius k whose centres are z apart."""
    z = np.asarray(z, dtype=np.float64)
    out = np.zeros_like(z)
    inside = z <= 1.0 - k
    out[inside] = np.pi * k * k
    part = (~inside) & (z < 1.0 + k)
    zp = z[part]
    a1 = np.clip((zp * zp + k * k - 1.0) / (2.0 * zp * k), -1.0, 1.0)
    a2 = np.clip((zp * zp + 1.0 - k * k) / (2.0 * zp), -1.0, 1.0)
    rad = np.clip((-zp + k + 1.0) * (zp + k - 1.0) * (zp - k + 1.0) * (zp + k + 1.0), 0.0, None)
    out[part] = k * k * np.arccos(a1) + np.arccos(a2) - 0.5 * np.sqrt(rad)
    return out


def transit_profile(x, u1: float = 0.4, u2: float = 0.25, k: float = 0.03, b: float = 0.32) -> np.ndarray:
    """Normalised dip T(x) for x in [0,1] (first to last contact), T(1/2)=1, 0 outside.

    Small-planet approximation: (area of the planet disc on the star) x (quadratic
    limb-darkened intensity at the planet's centre, clipped to the limb).
    Parameters k=R_p/R_*=0.03 and b=0.32 are those of PAPER.md:68.
    """
    x = np.asarray(x, dtype=np.float64)
    half_chord = np.sqrt((1.0 + k) ** 2 - b * b)

    def raw(xx):
        z = np.sqrt(b * b + ((2.0 * xx - 1.0) * half_chord) ** 2)
        r = np.minimum(z, 1.0)
        mu = np.sqrt(np.clip(1.0 - r * r, 0.0, None))
        inten = 1.0 - u1 * (1.0 - mu) - u2 * (1.0 - mu) ** 2
        return _overlap_area(z, k) * inten

    val = raw(x) / raw(np.array([0.5]))[0]
    val = np.where((x < 0.0) | (x > 1.0), 0.0, val)
    return val


def tabulate_template(n_template: int = 1024, u1: float = 0.4, u2: float = 0.25,
                      k: float = 0.03, b: float = 0.32) -> np.ndarray:
    """The tabulated profile handed to the library: M samples on x = m/(M-1)."""
    x = np.arange(n_template, dtype=np.float64) / float(n_template - 1)
    tpl = transit_profile(x, u1, u2, k, b)
    return tpl.astype(np.float32)


# --------------------------------------------------------------------------
# Trial grids
# --------------------------------------------------------------------------
def duration_grid(d_min_h: float, d_max_h: float, n_dur: int) -> np.ndarray:
    """Log-spaced trial durations in days."""
    return np.geomspace(d_min_h / 24.0, d_max_h / 24.0, n_dur).astype(np.float64)


def period_grid_uniform_frequency(p_min: float, p_max: float, n_per: int) -> np.ndarray:
    """Trial periods (days), uniform in frequency, returned in increasing-frequency order."""
    f = np.linspace(1.0 / p_max, 1.0 / p_min, n_per)
    return (1.0 / f).astype(np.float64)


# --------------------------------------------------------------------------
# Problem container
# --------------------------------------------------------------------------
@dataclass
class SearchProblem:
    """One search problem: light curve(s) + template + trial grids.

    flux / flux_err have shape [N] (single light curve) or [B][N] (batch sharing `times`).
    """
    cfg: int
    name: str
    times: np.ndarray            # [N] float64 days, regular cadence
    flux: np.ndarray             # float32 or float64; NaN marks a null point
    flux_err: np.ndarray         # same dtype; +inf marks a null point
    cadence: float               # days
    template: np.ndarray         # [M] float32
    durations: np.ndarray        # [J] float64 days
    t0_start: float              # days
    t0_stride: float             # days
    n_t0: int
    periods: np.ndarray          # [K] float64 days
    injections: List[Dict] = field(default_factory=list)   # per light curve for batches
    meta: Dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.times.shape[0])


def _regular_times(n: int, cadence_s: float) -> Tuple[np.ndarray, float]:
    c = cadence_s / DAY_S
    return np.arange(n, dtype=np.float64) * c, c


def _inject(times: np.ndarray, flux: np.ndarray, period: Optional[float], t0: float,
            depth: float, duration: float, u1: float, u2: float) -> None:
    """flux -= depth * T((t - t0_e)/D + 1/2) for every epoch inside the baseline."""
    t_lo, t_hi = times[0], times[-1]
    if period is None:
        epochs = [t0]
    else:
        e_lo = int(np.floor((t_lo - duration - t0) / period))
        e_hi = int(np.ceil((t_hi + duration - t0) / period))
        epochs = [t0 + e * period for e in range(e_lo, e_hi + 1)]
    for te in epochs:
        lo = np.searchsorted(times, te - 0.5 * duration, side="left")
        hi = np.searchsorted(times, te + 0.5 * duration, side="right")
        if hi <= lo:
            continue
        x = (times[lo:hi] - te) / duration + 0.5
        flux[lo:hi] -= depth * transit_profile(x, u1, u2)


def _t0_grid_over_baseline(times: np.ndarray, stride: float) -> Tuple[float, int]:
    """t0_i = times[0] + i*stride, I = floor(baseline/stride) + 1."""
    n_t0 = int(np.floor((times[-1] - times[0]) / stride + 1e-9)) + 1
    return float(times[0]), n_t0


def _ar1(rng: np.random.Generator, n: int, phi: float, sigma: float) -> np.ndarray:
    innov = rng.standard_normal(n) * sigma * np.sqrt(1.0 - phi * phi)
    out = np.empty(n, dtype=np.float64)
    acc = rng.standard_normal() * sigma
    for i in range(n):
        acc = phi * acc + innov[i]
        out[i] = acc
    return out


def make_config(cfg: int, n_periods: Optional[int] = None) -> SearchProblem:
    """BASELINE.json configs 1-4 (single light curve).  `n_periods` overrides K (tests)."""
    rng = np.random.default_rng(BASE_SEED + cfg)
    tpl = tabulate_template(1024, 0.4, 0.25)
    stride = 120.0 / DAY_S
    if cfg == 1:
        times, c = _regular_times(1000, 120.0)
        sigma = 1e-3
        flux = 1.0 + rng.standard_normal(1000) * sigma
        inj = dict(period=None, t0=0.7, depth=2e-3, duration=2.0 / 24.0, u1=0.4, u2=0.25)
        _inject(times, flux, None, inj["t0"], inj["depth"], inj["duration"], 0.4, 0.25)
        err = np.full(1000, sigma)
        durations = duration_grid(0.5, 4.0, 8)
        k = 200 if n_periods is None else n_periods
        periods = period_grid_uniform_frequency(0.3, 0.69, k)
        dtype = np.float64
        injections = [inj]
    elif cfg in (2, 3):
        cad_s = 120.0 if cfg == 2 else 20.0
        n = 19728 if cfg == 2 else 118368
        times, c = _regular_times(n, cad_s)
        sigma = 500e-6 if cfg == 2 else 1200e-6
        flux = 1.0 + rng.standard_normal(n) * sigma
        if cfg == 2:
            inj = dict(period=5.3, t0=1.7, depth=400e-6, duration=3.0 / 24.0, u1=0.4, u2=0.25)
            durations = duration_grid(0.5, 12.0, 30)
        else:
            inj = dict(period=11.2, t0=2.9, depth=250e-6, duration=4.5 / 24.0, u1=0.4, u2=0.25)
            durations = duration_grid(0.5, 15.0, 40)
        _inject(times, flux, inj["period"], inj["t0"], inj["depth"], inj["duration"], 0.4, 0.25)
        err = np.full(n, sigma)
        gap = (times >= 13.2) & (times < 14.2)
        flux[gap] = np.nan
        err[gap] = np.inf
        k = 20000 if n_periods is None else n_periods
        periods = period_grid_uniform_frequency(0.5, 13.7, k)
        dtype = np.float32
        injections = [inj]
    elif cfg == 4:
        n = 13 * 19728
        times, c = _regular_times(n, 120.0)
        phi = float(np.exp(-c / (6.0 / 24.0)))
        red = _ar1(rng, n, phi, 300e-6)
        white = rng.standard_normal(n) * 400e-6
        flux = 1.0 + red + white
        injections = [
            dict(period=127.0, t0=40.0, depth=150e-6, duration=9.0 / 24.0, u1=0.4, u2=0.25),
            dict(period=23.4, t0=5.0, depth=300e-6, duration=4.0 / 24.0, u1=0.4, u2=0.25),
        ]
        for inj in injections:
            _inject(times, flux, inj["period"], inj["t0"], inj["depth"], inj["duration"], 0.4, 0.25)
        err = np.full(n, 500e-6)
        for g in range(1, 26):
            gap = (times >= 13.7 * g - 0.5) & (times < 13.7 * g + 0.5)
            flux[gap] = np.nan
            err[gap] = np.inf
        durations = duration_grid(0.5, 24.0, 50)
        k = 200000 if n_periods is None else n_periods
        periods = period_grid_uniform_frequency(0.5, 178.0, k)
        dtype = np.float32
    else:
        raise ValueError("make_config handles cfg 1-4; use make_survey_batch for cfg 5")
    t0_start, n_t0 = _t0_grid_over_baseline(times, stride)
    return SearchProblem(
        cfg=cfg, name=CONFIG_NAMES[cfg], times=times, flux=flux.astype(dtype), flux_err=err.astype(dtype),
        cadence=c, template=tpl, durations=durations, t0_start=t0_start, t0_stride=stride, n_t0=n_t0,
        periods=periods, injections=injections, meta=dict(seed=BASE_SEED + cfg),
    )


def make_survey_batch(n_lc: int = 10000, n_periods: Optional[int] = None,
                      seed_offset: int = 0, lc_range: Optional[Tuple[int, int]] = None) -> SearchProblem:
    """BASELINE.json config 5: n_lc light curves on the cfg-2 time array, gap and grids.

    `lc_range=(lo, hi)` returns only curves lo..hi-1 of the n_lc-curve batch (the same curves a full
    call would return), so that a large survey can be generated and searched a slice at a time."""
    n = 19728
    times, c = _regular_times(n, 120.0)
    stride = 120.0 / DAY_S
    tpl = tabulate_template(1024, 0.4, 0.25)
    durations = duration_grid(0.5, 12.0, 30)
    k = 20000 if n_periods is None else n_periods
    periods = period_grid_uniform_frequency(0.5, 13.7, k)
    gap = (times >= 13.2) & (times < 14.2)
    children = np.random.SeedSequence(BASE_SEED + 5 + seed_offset).spawn(n_lc)
    if lc_range is not None:
        children = children[lc_range[0]:lc_range[1]]
    flux = np.empty((len(children), n), dtype=np.float32)
    err = np.empty((len(children), n), dtype=np.float32)
    injections: List[Dict] = []
    for b, child in enumerate(children):
        rng = np.random.default_rng(child)
        sigma = float(np.exp(rng.uniform(np.log(200e-6), np.log(2000e-6))))
        f = 1.0 + rng.standard_normal(n) * sigma
        has_planet = bool(rng.random() < 0.5)
        inj: Dict = dict(period=None, sigma=sigma)
        if has_planet:
            period = float(np.exp(rng.uniform(np.log(1.0), np.log(13.0))))
            t0 = float(rng.uniform(0.0, period))
            u1 = float(rng.uniform(0.2, 0.6))
            u2 = float(rng.uniform(0.0, 0.4))
            snr = float(rng.uniform(6.0, 12.0))
            a_rs = 4.2077 * period ** (2.0 / 3.0)
            half_chord = np.sqrt((1.0 + 0.03) ** 2 - 0.32 ** 2)
            duration = float(period / np.pi * np.arcsin(half_chord / a_rs))
            shape = np.zeros(n, dtype=np.float64)
            _inject(times, shape, period, t0, -1.0, duration, u1, u2)   # shape = +T at every epoch
            shape[gap] = 0.0
            norm = np.sqrt(np.sum(shape * shape) / (sigma * sigma))
            depth = snr / norm if norm > 0 else 0.0
            f -= depth * shape
            inj = dict(period=period, t0=t0, depth=depth, duration=duration, u1=u1, u2=u2,
                       snr=snr, sigma=sigma)
        e = np.full(n, sigma)
        f[gap] = np.nan
        e[gap] = np.inf
        flux[b] = f.astype(np.float32)
        err[b] = e.astype(np.float32)
        injections.append(inj)
    t0_start, n_t0 = _t0_grid_over_baseline(times, stride)
    return SearchProblem(
        cfg=5, name=CONFIG_NAMES[5], times=times, flux=flux, flux_err=err, cadence=c, template=tpl,
        durations=durations, t0_start=t0_start, t0_stride=stride, n_t0=n_t0, periods=periods,
        injections=injections, meta=dict(seed=BASE_SEED + 5 + seed_offset, n_lc=n_lc, lc_range=lc_range),
    )


# --------------------------------------------------------------------------
# Irregularly sampled input for the resampler (PLATO camera-group averages, barycentric times)
# --------------------------------------------------------------------------
def make_irregular_batch(seed: int = 250320881, n_lc: int = 3, n: int = 6000, cadence_s: float = 120.0,
                         dtype=np.float32, shuffle: bool = True):
    """`n_lc` light curves sharing one irregular timestamp array: a 2-min clock with a slow barycentric drift
    and per-point jitter, 3 % of the points dropped, a 0.4 d gap, 10 % extra "second camera group" points
    half a minute after their partner, a few null observations; optionally in shuffled order.
    Returns (times [n_obs] float64, flux [n_lc][n_obs], flux_err [n_lc][n_obs])."""
    rng = np.random.default_rng(seed)
    c = cadence_s / 86400.0
    t = 1325.0 + c * np.arange(n) + 2.0e-4 * np.sin(np.arange(n) * c * 2 * np.pi / 27.0) \
        + rng.uniform(-0.2, 0.2, n) * c
    keep = rng.random(n) > 0.03
    keep &= ~((t > t[0] + 3.1) & (t < t[0] + 3.5))
    t = t[keep]
    extra = t[rng.random(t.shape[0]) < 0.10] + 0.25 * c
    t = np.concatenate([t, extra])
    if shuffle:
        t = t[rng.permutation(t.shape[0])]
    n_obs = t.shape[0]
    sig = rng.uniform(4e-4, 1.5e-3, (n_lc, n_obs))
    flux = 1.0 + sig * rng.standard_normal((n_lc, n_obs))
    for b in range(n_lc):
        flux[b] -= _inject_profile(t, period=1.3 + 0.4 * b, t0=t.min() + 0.5, depth=2e-3, duration=0.1)
    bad = rng.random((n_lc, n_obs)) < 0.01
    flux[bad] = np.nan
    sig[rng.random((n_lc, n_obs)) < 0.005] = np.inf
    return t.astype(np.float64), flux.astype(dtype), sig.astype(dtype)


def _inject_profile(t: np.ndarray, period: float, t0: float, depth: float, duration: float) -> np.ndarray:
    ph = np.mod(t - t0 + 0.5 * period, period) - 0.5 * period
    x = ph / duration + 0.5
    out = np.zeros_like(t)
    ins = (x >= 0.0) & (x <= 1.0)
    out[ins] = depth * transit_profile(x[ins])
    return out

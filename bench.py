#!/usr/bin/env python
"""bench.py -- throughput of the CETRA hot path on B200 (one JSON line on stdout, rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--n-lc B] [--workload sector|survey] [--impl cuda|reference]

A *step* is one pass of the whole hot path (preprocess, template taps,
windowed sums + epilogue, fold-gather-sum, combine, per-period argmax) over one batch of B synthetic
light curves.  The workload is BASELINE.json configs[1], the TESS-like 2-min sector (19 728 points,
30 durations, 20 000 periods), B curves per GPU drawn with the config-5 survey recipe (cetra_synth).

  value      light curves/s, inputs resident in HBM when the timed region starts (cetra_search_batched)
  e2e        the same metric through cetra_search_batched_host: pinned HOST buffers, H2D + D2H timed
  roofline   the dominant kernel (fold_pair_argmax_kernel, periodic search).  Its rows live in shared memory, so
             the level that bounds it is the shared-memory crossbar: achieved = bytes its LDS instructions moved
             (ncu wavefront count of this workload x 128 B, a property of the launch, see NCU_FOLD) / the
             kernel's event-timed duration in THIS run; peak = 148 SM x 128 B/clk x clock (cetra_peak_probe's
             measured LDS.64 rate is reported beside it).  north_star's HBM yardstick (8 B per (period, duration, t0 cell)) is kept
             beside it as `algorithmic`.
  cpu_baseline  the FP64 oracle on the host cores (all cores, and one thread), on a bounded sample of the workload

N > 1: `python bench.py --gpus N` re-executes itself under torch.distributed.run with N ranks (the driver's own
torchrun launch is used as it is); every rank searches its own B curves (no data-path collective; "weak"
scaling), the time is the max over ranks.  --impl reference times the oracle (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "TESS-sector light curves/sec"
UNIT = "light curves/s"
L2_FLUSH_BYTES = 512 << 20
N_SM, FP32_LANES = 148, 128          # B200: SMs, FP32 FMA lanes per SM (B200_PROFILING.md unit counts)
SMEM_BYTES_PER_CLK = 128             # shared-memory crossbar bytes/clk/SM (B300_MICROARCH.md, LDS/STS)
# nominal per-clock per-SM rates of the probed instructions: 128 lanes x 2 flop (FFMA2), x 1 flop (FADD2), crossbar bytes
PROBE_NOMINAL = dict(ffma2=2.0 * FP32_LANES, fadd2=1.0 * FP32_LANES, lds64=float(SMEM_BYTES_PER_CLK))
# Counters of ONE fold_pair_argmax_kernel launch over the 64-curve chunk of this workload, from the `ncu --set full`
# capture summarised in `profile` (command inside).  They are properties of the launch (the kernel's loads do not
# depend on timing), valid for the kernel sources whose hash is `src_sha256`: bench.py hashes the sources it runs
# and reports `stale: true` (and no traffic) when they differ.
NCU_FOLD = dict(
    profile="profiles/r02e_fold_pair_full.md", commit="9c3afc6", n_lc=64,
    src_sha256="7d2b85c78a98cdc2fe2ff350a7ff8c4264e32d289f7b65781ea0f389f99a9de2",
    lds_wavefronts=32077233385.0,       # l1tex__data_pipe_lsu_wavefronts_mem_shared.sum (128 B each)
    dram_bytes=332411904.0 + 12120576.0,  # dram__bytes_read.sum + dram__bytes_write.sum
    crossbar_pct_under_ncu=90.63,       # ...wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed
    duration_ms_under_ncu=121.93,
)
FOLD_SOURCES = ("fold_pair.cu", "fold_common.cuh", "periodic_search.cuh", "common.cuh")


def fold_sources_sha256() -> str:
    import hashlib
    h = hashlib.sha256()
    for name in FOLD_SOURCES:
        with open(os.path.join(ROOT, "paper_2503_20875_b200", "csrc", name), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


# ---------------------------------------------- other workloads on the same line (round-2 review, "Next round" 3)
# Per-curve counters of fold_stream_argmax_kernel from the ncu pass named in `profile` (metrics only: LDS wavefronts,
# DRAM bytes), valid for the sources whose hash is `src_sha256`; like NCU_FOLD they are properties of the launch.
NCU_STREAM = dict(
    profile="profiles/r03a_fold_stream_legs.md", src_sha256="9d7102a06b6e1040f84cc9443b940568184f8c03867b304e3f1df1f4f9add4bf", per_curve={
        # leg name -> (l1tex__data_pipe_lsu_wavefronts_mem_shared.sum, dram bytes read + written) of ONE light curve
        "configs3": (101992340344.0, 113329408.0 + 2987520.0),                       # one curve per launch, 78.2 % under ncu
        "default_grid": (62437322352.0 / 16, (141049652224.0 + 20825344.0) / 16),   # 16 curves per launch, 85.8 % under ncu
    })
STREAM_SOURCES = ("fold_stream.cu", "fold_common.cuh", "periodic_search.cuh", "common.cuh")


def sources_sha256(names) -> str:
    import hashlib
    h = hashlib.sha256()
    for name in names:
        with open(os.path.join(ROOT, "paper_2503_20875_b200", "csrc", name), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def config_legs(cetra, torch, dev, peaks, flush, reps: int = 2):
    """The workloads whose rooflines the docs quote besides the headline one, timed in this process after the main
    region (a few seconds in all): BASELINE configs[2] (20-s cadence) linear search in a batch of 32, configs[3]
    (one 256 464-cell curve) whole search, and configs[1] on the paper's default t0 grid (stride = 1 % of the
    shortest duration) in a batch of 64.  Kernel times are the library's own event brackets around its
    linear-search and fold kernels (cetra_profile_enable), averaged per launch over `reps` passes after one warm-up,
    L2 flushed between passes.  Returns a list of {workload, kernel, ms, launches, bound, achieved, peak, unit, frac}."""
    from cetra_synth import make_config, make_survey_batch
    fp32_peak = N_SM * FP32_LANES * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12          # TFLOP/s
    smem_peak = N_SM * SMEM_BYTES_PER_CLK * peaks["sm_max_mhz"] * 1e6 / 1e9        # GB/s
    stream_stale = sources_sha256(STREAM_SOURCES) != NCU_STREAM["src_sha256"]

    def profiled(fn):
        fn()
        torch.cuda.synchronize()
        cetra.cetra_profile_enable(True)
        for _ in range(reps):
            flush.zero_()
            fn()
        torch.cuda.synchronize()
        prof = cetra.cetra_profile_read(reset=True)
        cetra.cetra_profile_enable(False)
        return prof

    def linear_leg(workload, kernel, prof, evals_per_pass):
        ms = prof["linear_ms"] / max(prof["linear_launches"], 1)
        tf = 4.0 * evals_per_pass * reps / (prof["linear_ms"] * 1e-3) / 1e12
        return dict(workload=workload, kernel=kernel, ms=ms, launches=int(prof["linear_launches"]), bound="alu",
                    achieved=tf, peak=fp32_peak, unit="TFLOP/s", frac=tf / fp32_peak,
                    template_evals_per_s=evals_per_pass * reps / (prof["linear_ms"] * 1e-3))

    def stream_leg(workload, name, prof, curves_per_pass, cells_per_curve):
        ms = prof["fold_ms"] / max(prof["fold_launches"], 1)
        counters = None if stream_stale else NCU_STREAM["per_curve"].get(name)
        leg = dict(workload=workload, kernel="fold_stream_argmax_kernel", ms=ms, launches=int(prof["fold_launches"]),
                   bound="smem", peak=smem_peak, unit="GB/s", achieved=None, frac=None, traffic=None,
                   fold_cells_per_s=cells_per_curve * curves_per_pass * reps / (prof["fold_ms"] * 1e-3),
                   ms_per_curve=prof["fold_ms"] / (curves_per_pass * reps), ncu_stale=stream_stale)
        if counters:
            gbs = 128.0 * counters[0] * curves_per_pass * reps / (prof["fold_ms"] * 1e-3) / 1e9
            leg.update(achieved=gbs, frac=gbs / smem_peak, traffic=counters[1] * curves_per_pass * reps /
                       max(prof["fold_launches"], 1))
        return leg

    legs = []
    # -- configs[2]: 20-s cadence, 118 368 points, long windows (up to 2 701 taps): the linear kernel in a batch of 32
    p = make_config(3)
    wc = work_counts(p)
    fl = torch.from_numpy(np.tile(p.flux, (32, 1))).to(dev)
    er = torch.from_numpy(np.tile(p.flux_err, (32, 1))).to(dev)
    prof = profiled(lambda: cetra.cetra_linear_search(p.times, fl, er, p.durations, p.t0_start, p.t0_stride, p.n_t0,
                                                      p.template, want_grids=False, want_stats=True))
    legs.append(linear_leg(f"BASELINE configs[2] {p.name} x 32 light curves (one curve tiled), linear search",
                           "linear_search_kernel", prof, 32.0 * wc["template_evals"]))
    del fl, er
    # -- configs[3]: one curve, rows of 2 MB: linear search + the streamed fold
    p = make_config(4)
    wc = work_counts(p)
    fl, er = torch.from_numpy(p.flux).to(dev), torch.from_numpy(p.flux_err).to(dev)
    prof = profiled(lambda: cetra.cetra_search_batched(p.times, fl[None], er[None], p.durations, p.t0_start,
                                                       p.t0_stride, p.n_t0, p.template, p.periods))
    legs.append(linear_leg(f"BASELINE configs[3] {p.name}, one light curve, linear search", "linear_search_kernel",
                           prof, float(wc["template_evals"])))
    legs.append(stream_leg(f"BASELINE configs[3] {p.name}, one light curve, periodic search", "configs3", prof, 1,
                           float(wc["gathers"])))
    del fl, er
    # -- configs[1] on the paper's default t0 grid (18 s = 3/20 of the cadence): residue-class linear kernel + streamed fold
    B = 64
    p = make_survey_batch(n_lc=B, lc_range=(0, B))
    wc = work_counts(p)
    stride = 0.01 * p.durations[0]
    n_t0 = int((p.times[-1] - p.times[0]) / stride) + 1
    fl, er = torch.from_numpy(p.flux).to(dev), torch.from_numpy(p.flux_err).to(dev)
    prof = profiled(lambda: cetra.cetra_search_batched(p.times, fl, er, p.durations, p.times[0], stride, n_t0,
                                                       p.template, p.periods))
    what = f"BASELINE configs[1] on the paper's default t0 grid (stride 18 s, {n_t0} cells) x {B} light curves"
    legs.append(linear_leg(what + ", linear search", "linear_search_kernel<CLS> (residue classes)", prof,
                           B * wc["template_evals"] * (n_t0 / p.n_t0)))
    legs.append(stream_leg(what + ", periodic search", "default_grid", prof, B, float(wc["pairs"]) * n_t0))
    return legs



# ----------------------------------------------------------------------------------------------- helpers
def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def work_counts(p):
    """Algorithmic work of one light curve (counting only)."""
    n, c = p.n, p.cadence
    q = int(round(p.t0_stride / c))
    n0 = int(round((p.t0_start - p.times[0]) / c))
    centres = n0 + q * np.arange(p.n_t0, dtype=np.int64)
    evals = 0
    for d in p.durations:
        h = int(np.floor(d / (2.0 * c) + 1e-12))
        lo = np.maximum(centres - h, 0)
        hi = np.minimum(centres + h, n - 1)
        evals += int(np.maximum(hi - lo + 1, 0).sum())
    pairs = int((p.durations[None, :] < p.periods[:, None]).sum())
    return dict(template_evals=evals, pairs=pairs, gathers=pairs * p.n_t0, cells=p.n_t0 * len(p.durations))


def rank_slice(rank: int, world: int, per_rank: int):
    """Light curves [lo, hi) of the world*per_rank-curve batch that `rank` searches (weak scaling: curves are
    independent, so the partition is the whole multi-GPU design; no data-path collective)."""
    return rank * per_rank, (rank + 1) * per_rank


def max_over_ranks(ms: float, device, world: int) -> float:
    """Device-timed milliseconds -> the slowest rank's (the job finishes when the last rank does)."""
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


class ClockSampler:
    """nvidia-smi clocks / throttle reasons while the timed region runs (B200_PROFILING.md clocks line)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *exc):
        if self.proc is not None:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except subprocess.TimeoutExpired:
                self.proc.kill()
            self.thread.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except ValueError:
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        return dict(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))


def oracle_sample(p, flux, flux_err, budget_s: float, threads: int = 0):
    """The oracle, as it stands, on one light curve of the workload: the linear search in full and the
    periodic search on a seeded subset of the trial periods sized to about `budget_s` of CPU time.
    `threads` > 0 limits its OpenMP threads for this sample.
    Returns (light curves/s extrapolated to all K periods, description, cores, seconds spent)."""
    import oracle
    oracle.build()
    all_threads = oracle.get_threads()
    # all the cores this process may use, stated explicitly: torchrun exports OMP_NUM_THREADS=1 to its ranks, which
    # would silently turn the N > 1 reference arm into a one-thread run
    oracle.set_threads(threads if threads > 0 else len(os.sched_getaffinity(0)))
    try:
        return _oracle_sample(oracle, p, flux, flux_err, budget_s)
    finally:
        oracle.set_threads(all_threads)


def _oracle_sample(oracle, p, flux, flux_err, budget_s):
    cores = oracle.get_threads()
    t = time.perf_counter()
    grids = oracle.linear_search(p.times, flux, flux_err, p.durations, p.t0_start, p.t0_stride, p.n_t0, p.template)
    t_lin = time.perf_counter() - t
    rng = np.random.default_rng(20875)
    K = p.periods.shape[0]
    order = rng.permutation(K)
    probe, t_probe = max(cores, 8), 0.0
    while True:                                     # grow the probe until it is long enough to time
        t = time.perf_counter()
        oracle.periodic_search(grids, p.t0_start, p.t0_stride, p.durations, p.periods[np.sort(order[:probe])])
        t_probe = time.perf_counter() - t
        if t_probe >= 0.1 * budget_s or probe >= K:
            break
        probe = min(K, probe * 4)
    k_s = int(min(K, max(probe, budget_s / max(t_probe / probe, 1e-9))))
    t = time.perf_counter()
    oracle.periodic_search(grids, p.t0_start, p.t0_stride, p.durations, p.periods[np.sort(order[:k_s])])
    t_per = time.perf_counter() - t
    t_lc = t_lin + t_per * (K / k_s)
    sample = (f"1 light curve of the workload: linear search in full ({t_lin:.2f} s) + periodic search on a seeded "
              f"{k_s}-of-{K} period subset ({t_per:.2f} s), periodic time scaled by K/subset")
    return 1.0 / t_lc, sample, cores, t_lin + t_per


# ------------------------------------------------------------------------------------------ reference arm
def run_reference(args, rank: int):
    """--impl reference: the oracle on the host cores (rank 0 only), same metric / unit / config."""
    if rank != 0:
        return
    from cetra_synth import make_survey_batch
    p = make_survey_batch(n_lc=max(args.n_lc, 1), lc_range=(0, 1))
    budget = args.ref_seconds
    for _ in range(args.warmup):
        oracle_sample(p, p.flux[0], p.flux_err[0], min(budget, 1.0))
    vals, spent, sample, cores = [], 0.0, "", 0
    t0 = time.perf_counter()
    for _ in range(args.steps):
        v, sample, cores, used = oracle_sample(p, p.flux[0], p.flux_err[0], budget)
        vals.append(v); spent += used
    wall = time.perf_counter() - t0
    value = len(vals) / sum(1.0 / v for v in vals)
    line = dict(metric=METRIC, value=value, unit=UNIT, impl="reference", n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=1e3 / value, higher_is_better=True,
                scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=workload_config(p, args.n_lc),
                notes="oracle on host cores; each step = " + sample + "; ms_per_step is the time `value` counts (one "
                      "light curve, periodic part scaled to all periods); ms_wall_per_step also holds the passes that "
                      "size the subset and ms_timed_per_step only the linear search and the timed subset",
                ms_wall_per_step=1e3 * wall / max(args.steps, 1), ms_timed_per_step=1e3 * spent / max(args.steps, 1),
                cpu_baseline=dict(value=value, unit=UNIT, cores=cores, kind="oracle", sample=sample),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                gpu_launches=0)
    print(json.dumps(line), flush=True)


def workload_config(p, n_lc):
    """The same dict for both arms (the driver compares them)."""
    return dict(workload=f"BASELINE configs[1] tess-2min-sector x {n_lc} light curves per GPU per step "
                         f"(config-5 survey recipe: shared 19 728-point 2-min time array with a 1 d gap)",
                n_points=p.n, n_durations=int(len(p.durations)), n_t0=int(p.n_t0), n_periods=int(len(p.periods)),
                n_template=int(len(p.template)), light_curves_per_step_per_gpu=n_lc,
                l2="flushed between timed steps (512 MiB write)")


# ------------------------------------------------------------------------------------------------- CUDA arm
def run_cuda(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist

    import paper_2503_20875_b200 as cetra
    from cetra_synth import make_survey_batch

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the CETRA library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    cetra.load_library()
    if world > 1 and not dist.is_initialized():
        dist.init_process_group("nccl", device_id=dev)

    if args.legs_only:
        flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
        print(json.dumps(dict(configs=config_legs(cetra, torch, dev, measured_peaks(), flush, reps=1))), flush=True)
        return
    B = args.n_lc
    p = make_survey_batch(n_lc=B * world, lc_range=rank_slice(rank, world, B))   # each rank owns its curves
    wc = work_counts(p)
    K = p.periods.shape[0]
    flux_h = torch.from_numpy(p.flux).pin_memory()
    err_h = torch.from_numpy(p.flux_err).pin_memory()
    flux_d, err_d = flux_h.to(dev), err_h.to(dev)
    gargs = (p.durations, p.t0_start, p.t0_stride, p.n_t0, p.template, p.periods)
    ws_bytes = cetra.cetra_search_batched_host_workspace_bytes(p.times, B, args.lc_chunk, cetra.CETRA_F32, p.durations,
                                                               p.t0_start, p.t0_stride, p.n_t0, len(p.template), K)
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device=dev)
    peaks_d = torch.empty((B, K, 8), dtype=torch.int32, device=dev)
    peaks_h = torch.empty((B, K, 8), dtype=torch.int32).pin_memory()
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def step_device():
        cetra.cetra_search_batched(p.times, flux_d, err_d, *gargs, lc_chunk=args.lc_chunk, workspace=ws, peaks=peaks_d)

    def step_host():
        cetra.cetra_search_batched_host(p.times, flux_h, err_h, *gargs, lc_chunk=args.lc_chunk, workspace=ws,
                                        peaks_host=peaks_h, device=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, profile):
        """`steps` steps, each bracketed by CUDA events on the launching stream; L2 flushed between them."""
        evs = []
        barrier()
        if profile:
            cetra.cetra_profile_enable(True)
        launches0 = cetra.cetra_kernel_launch_count()
        t_wall = time.perf_counter()
        for _ in range(steps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            fn()
            b.record(stream)
            evs.append((a, b))
        barrier()
        wall = time.perf_counter() - t_wall
        launches = cetra.cetra_kernel_launch_count() - launches0
        prof = cetra.cetra_profile_read(reset=True) if profile else None
        if profile:
            cetra.cetra_profile_enable(False)
        ms = max_over_ranks(sum(a.elapsed_time(b) for a, b in evs), dev, world)
        return ms, launches, prof, wall

    for _ in range(args.warmup):
        step_device()
    for _ in range(min(args.warmup, 1)):
        step_host()
    probes = {}
    for name, kind in (("ffma2", cetra.CETRA_PROBE_FFMA2), ("fadd2", cetra.CETRA_PROBE_FADD2),
                       ("lds64", cetra.CETRA_PROBE_LDS64)):
        per_clk, per_s = cetra.cetra_peak_probe(kind)
        probes[name] = dict(per_clk_per_sm=per_clk, per_second=per_s, unit="B" if name == "lds64" else "flop",
                            nominal_per_clk_per_sm=PROBE_NOMINAL[name])
        # a probe above the unit's physical rate is a broken probe (round 2: ptxas merged the LDS probe's repeated
        # addresses and it read 3.0 x the crossbar), and a roofline beside it would be unexplained: refuse to print one
        if per_clk > 1.05 * PROBE_NOMINAL[name]:
            raise SystemExit(f"bench.py: cetra_peak_probe({name}) measured {per_clk:.1f} per clock per SM, above the "
                             f"unit's nominal {PROBE_NOMINAL[name]}: the probe is not measuring what it claims")
    with ClockSampler(local_rank) as clocks:
        ms_dev, launches, prof, wall_dev = timed(step_device, args.steps, profile=True)
    ms_e2e, _, _, wall_e2e = timed(step_host, args.steps, profile=False)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = measured_peaks()
    total_lc = B * world * args.steps
    value = total_lc / (ms_dev * 1e-3)
    e2e_value = total_lc / (ms_e2e * 1e-3)
    fold_launches = max(prof["fold_launches"], 1)
    lin_launches = max(prof["linear_launches"], 1)
    fold_ms = prof["fold_ms"] / fold_launches                   # average launch, event-timed in this run
    lin_ms = prof["linear_ms"] / lin_launches
    lc_per_launch = B * args.steps / fold_launches
    # -- dominant kernel: the periodic fold.  Physical level: shared-memory crossbar (LDS bytes / probe rate).
    sha = fold_sources_sha256()
    stale = sha != NCU_FOLD["src_sha256"]
    # the wavefront count belongs to the sources it was captured from: with edited fold sources there is no
    # crossbar figure (achieved / frac / lds_bytes_per_launch are null and `ncu.stale` says why), only the yardstick
    lds_bytes = None if stale else 128.0 * NCU_FOLD["lds_wavefronts"] * lc_per_launch / NCU_FOLD["n_lc"]
    lds_gbs = None if stale else lds_bytes / (fold_ms * 1e-3) / 1e9
    smem_peak_gbs = N_SM * SMEM_BYTES_PER_CLK * peaks["sm_max_mhz"] * 1e6 / 1e9
    # north_star's yardstick: 8 B gathered and 2 FADD per (period, duration, t0 cell) against the HBM copy peak
    alg_bytes = 8.0 * wc["gathers"] * lc_per_launch
    alg_gbs = alg_bytes / (fold_ms * 1e-3) / 1e9
    lin_tflops = 4.0 * wc["template_evals"] * (B * args.steps / lin_launches) / (lin_ms * 1e-3) / 1e12
    fp32_peak = N_SM * FP32_LANES * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    line = dict(
        metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
        ms_per_step=ms_dev / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
        dtype="f32", data="synthetic", config=workload_config(p, B),
        notes="timed per step with CUDA events on the launching stream, summed; max over ranks",
        e2e=dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=int(2 * B * p.n * 4),
                 d2h_bytes_per_step=int(B * K * 32), ms_per_step=ms_e2e / args.steps,
                 api="cetra_search_batched_host (pinned host flux/flux_err in, pinned host records out)"),
        gpu_launches=int(launches),
        clocks=clocks.summary(),
        roofline=dict(
            bound="smem", kernel="fold_pair_argmax_kernel", achieved=lds_gbs, peak=smem_peak_gbs, unit="GB/s",
            frac=None if stale else lds_gbs / smem_peak_gbs,
            traffic=None if stale else NCU_FOLD["dram_bytes"] * lc_per_launch / NCU_FOLD["n_lc"],
            derivation="achieved = shared-memory bytes the kernel's loads move per launch (ncu LDS wavefronts of "
                       "this workload x 128 B, scaled to the curves per launch) / its average event-timed "
                       "duration in this run; peak = 148 SM x 128 B/clk x sm_max_mhz (the crossbar's nominal "
                       "rate; peak_probe = the conflict-free LDS.64 rate cetra_peak_probe measures in this run)",
            ms_per_launch=fold_ms, launches=int(prof["fold_launches"]), share_of_step=prof["fold_ms"] / ms_dev,
            lds_bytes_per_launch=lds_bytes,
            peak_probe=probes["lds64"],
            ncu=dict(NCU_FOLD, stale=stale, src_sha256_now=sha),
            algorithmic=dict(bytes_per_launch=alg_bytes, gbs=alg_gbs, hbm_peak_gbs=peaks["hbm_gbs"],
                             over_hbm_peak=alg_gbs / peaks["hbm_gbs"], hbm_peak_source=peaks["source"],
                             loads_per_cell=None if stale else lds_bytes / alg_bytes,
                             note="north_star's yardstick (8 B per (period, duration, t0 cell) / HBM copy peak); "
                                  "a ratio above 1 is reuse, not a roofline fraction: a row is read from HBM a "
                                  "handful of times per launch and gathered from shared memory 20 000 times")),
        roofline_linear=dict(bound="alu", kernel="linear_search_kernel", achieved=lin_tflops, peak=fp32_peak,
                             unit="TFLOP/s", frac=lin_tflops / fp32_peak,
                             derivation="4 flop per (t0, duration, in-window point) template evaluation / the "
                                        "kernel's event-timed duration; peak = 148 SM x 128 FP32 lanes x 2 flop "
                                        "x sm_max_mhz (peak_probe = the packed FP32 FMA rate cetra_peak_probe "
                                        "measures in this run)",
                             peak_probe=probes["ffma2"],
                             ms_per_launch=lin_ms, launches=int(prof["linear_launches"]),
                             share_of_step=prof["linear_ms"] / ms_dev,
                             template_evals_per_s=wc["template_evals"] * (B * args.steps / lin_launches) /
                                                  (lin_ms * 1e-3)),
        rates=dict(periods_per_s=K * total_lc / (ms_dev * 1e-3),
                   template_evals_per_lc=wc["template_evals"], gathers_per_lc=wc["gathers"],
                   duration_period_pairs=wc["pairs"], fadd2_probe=probes["fadd2"]),
    )
    if world == 1 and not args.no_legs:
        del ws, peaks_d, flux_d, err_d
        torch.cuda.empty_cache()
        line["configs"] = config_legs(cetra, torch, dev, peaks, flush)
    if world == 1 and not args.no_cpu_baseline:
        v, sample, cores, _ = oracle_sample(p, p.flux[0], p.flux_err[0], args.cpu_seconds)
        v1, sample1, _, _ = oracle_sample(p, p.flux[0], p.flux_err[0], args.cpu_seconds / 2, threads=1)
        line["cpu_baseline"] = dict(value=v, unit=UNIT, cores=cores, kind="oracle", sample=sample,
                                    one_thread=dict(value=v1, unit=UNIT, cores=1, sample=sample1))
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------- config-5 survey (optional)
def run_survey(args):
    """BASELINE.json configs[4]: the 10 000-curve survey batch, a slice at a time, with the injection-
    recovery fraction (best period within 1 % of P, P/2 or 2P).  One GPU."""
    import torch

    import paper_2503_20875_b200 as cetra
    from cetra_synth import make_survey_batch

    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    n_total, sl = args.survey_lc, args.n_lc
    rec = inj = false_alarm_free = 0
    gpu_ms = 0.0
    best_lr_planet, best_lr_null = [], []
    for lo in range(0, n_total, sl):
        hi = min(n_total, lo + sl)
        p = make_survey_batch(n_lc=n_total, lc_range=(lo, hi))
        flux_d, err_d = torch.from_numpy(p.flux).to(dev), torch.from_numpy(p.flux_err).to(dev)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        peaks = cetra.cetra_search_batched(p.times, flux_d, err_d, p.durations, p.t0_start, p.t0_stride, p.n_t0,
                                           p.template, p.periods)
        b.record()
        torch.cuda.synchronize()
        gpu_ms += a.elapsed_time(b)
        lr = peaks[..., 0].view(torch.float32)                       # host step: pick the peak period
        lr = torch.where(torch.isnan(lr), torch.full_like(lr, -1.0), lr)
        kb = torch.argmax(lr, dim=1).cpu().numpy()
        best = lr.max(dim=1).values.cpu().numpy()
        for i, injn in enumerate(p.injections):
            pb = p.periods[kb[i]]
            if injn["period"] is None:
                best_lr_null.append(float(best[i]))
                continue
            inj += 1
            best_lr_planet.append(float(best[i]))
            if any(abs(pb - m * injn["period"]) <= 0.01 * m * injn["period"] for m in (0.5, 1.0, 2.0)):
                rec += 1
    line = dict(metric=METRIC, value=n_total / (gpu_ms * 1e-3), unit=UNIT, n_gpus=1, workload="BASELINE configs[4] "
                f"survey batch, {n_total} light curves in slices of {sl}", injected=inj, recovered=rec,
                recovery_fraction=rec / max(inj, 1), gpu_seconds=gpu_ms * 1e-3,
                median_best_lr_injected=float(np.median(best_lr_planet)) if best_lr_planet else None,
                median_best_lr_null=float(np.median(best_lr_null)) if best_lr_null else None)
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------ BASELINE configs 1-4, stage by stage (optional)
def run_configs(args):
    """One JSON line per BASELINE.json config 1-4 (single light curve): linear search and periodic search timed
    separately with CUDA events (3 warm-ups, median of `--steps` repetitions, L2 flushed in between), as template
    evaluations/s against the FP32 peak and periods/s + algorithmic GB/s against the HBM and shared-memory peaks;
    plus the off-grid t0 kernel (paper default stride, 1 % of the shortest duration) and the setup kernels."""
    import torch

    import paper_2503_20875_b200 as cetra
    from cetra_synth import make_config, make_irregular_batch

    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    peaks_hw = measured_peaks()
    fp32_peak = N_SM * FP32_LANES * 2 * peaks_hw["sm_max_mhz"] * 1e6
    smem_peak = N_SM * SMEM_BYTES_PER_CLK * peaks_hw["sm_max_mhz"] * 1e6
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)

    def med_ms(fn, reps):
        for _ in range(3):
            fn()
        out = []
        for _ in range(reps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record()
            torch.cuda.synchronize()
            out.append(a.elapsed_time(b))
        return statistics.median(out)

    for cfg in [int(c) for c in args.cfgs.split(",")]:
        p = make_config(cfg)
        wc = work_counts(p)
        flux, err = torch.from_numpy(p.flux).to(dev), torch.from_numpy(p.flux_err).to(dev)
        reps = max(1, args.steps if cfg < 4 else min(args.steps, 3))
        lin_ms = med_ms(lambda: cetra.cetra_linear_search(p.times, flux, err, p.durations, p.t0_start, p.t0_stride,
                                                          p.n_t0, p.template, want_grids=False, want_stats=True), reps)
        lin = cetra.cetra_linear_search(p.times, flux, err, p.durations, p.t0_start, p.t0_stride, p.n_t0, p.template,
                                        want_grids=False, want_stats=True)
        per_ms = med_ms(lambda: cetra.cetra_periodic_search_stats(lin.stats, p.n_t0, p.t0_start, p.t0_stride,
                                                                  p.durations, p.periods), reps)
        fold_bytes = 8.0 * wc["gathers"]
        line = dict(workload=f"BASELINE configs[{cfg - 1}] {p.name}", n_points=p.n, n_t0=int(p.n_t0),
                    n_durations=int(len(p.durations)), n_periods=int(len(p.periods)),
                    linear_ms=lin_ms, template_evals=wc["template_evals"],
                    template_evals_per_s=wc["template_evals"] / (lin_ms * 1e-3),
                    linear_frac_fp32=4.0 * wc["template_evals"] / (lin_ms * 1e-3) / fp32_peak,
                    periodic_ms=per_ms, periods_per_s=len(p.periods) / (per_ms * 1e-3),
                    fold_algorithmic_gbs=fold_bytes / (per_ms * 1e-3) / 1e9,
                    fold_algorithmic_over_hbm_peak=fold_bytes / (per_ms * 1e-3) / 1e9 / peaks_hw["hbm_gbs"],
                    fold_algorithmic_over_smem_peak=fold_bytes / (per_ms * 1e-3) / smem_peak,
                    light_curves_per_s=1e3 / (lin_ms + per_ms), reps=reps,
                    note="periodic_ms includes finalize_peaks and the key memset; single light curve, so the short "
                         "configs are launch- and tail-bound")
        print(json.dumps(line), flush=True)
        if cfg == 2:
            stride = 0.01 * p.durations[0]                          # PAPER.md:87 default
            n_t0 = int((p.times[-1] - p.times[0]) / stride) + 1
            og_ms = med_ms(lambda: cetra.cetra_linear_search(p.times, flux, err, p.durations, p.times[0], stride, n_t0,
                                                             p.template, want_grids=False, want_stats=True), reps)
            evals = wc["template_evals"] * (n_t0 / p.n_t0)
            og = cetra.cetra_linear_search(p.times, flux, err, p.durations, p.times[0], stride, n_t0, p.template,
                                           want_grids=False, want_stats=True)
            ogp_ms = med_ms(lambda: cetra.cetra_periodic_search_stats(og.stats, n_t0, p.times[0], stride, p.durations,
                                                                      p.periods), max(1, min(reps, 3)))
            og_bytes = 8.0 * wc["pairs"] * n_t0
            print(json.dumps(dict(workload="configs[1] on the paper's default t0 grid (stride = 1 % of the shortest "
                                           "duration = 18 s = 3/20 of the cadence, off the sample grid): "
                                           "linear_search_kernel on residue classes of cells, then the streamed "
                                           "fold kernel (1.05 MB rows)",
                                  n_t0=n_t0, linear_ms=og_ms, template_evals_per_s=evals / (og_ms * 1e-3),
                                  bound="alu (FP32 FMA; the polyphase branches of a class pad their taps)",
                                  periodic_ms=ogp_ms, fold_algorithmic_gbs=og_bytes / (ogp_ms * 1e-3) / 1e9,
                                  light_curves_per_s=1e3 / (og_ms + ogp_ms))), flush=True)
    # setup kernels: resampling 64 irregular light curves of 200 000 observations (HBM-bound streaming)
    for shuffle in (False, True):
        t, f, e = make_irregular_batch(n_lc=64, n=200000, shuffle=shuffle)
        td, fd, ed = (torch.from_numpy(a).to(dev) for a in (t, f, e))
        t_start, c, n_out = cetra.cetra_resample_grid(t, 0.0, 0.25)
        rs_ms = med_ms(lambda: cetra.cetra_resample(td, fd, ed, t_start, c, n_out), max(3, args.steps))
        moved = f.nbytes + e.nbytes + t.nbytes + 64 * n_out * 8     # every input read once, every output written once
        print(json.dumps(dict(workload="cetra_resample, 64 curves x %d observations -> %d points, input %s"
                                       % (t.shape[0], n_out, "in random order (4-byte gathers: 8 x the bytes through "
                                          "L2)" if shuffle else "in time order"),
                              ms=rs_ms, algorithmic_gbs=moved / (rs_ms * 1e-3) / 1e9,
                              frac_hbm=moved / (rs_ms * 1e-3) / 1e9 / peaks_hw["hbm_gbs"])), flush=True)


# --------------------------------------------------------- tensor-core variant of the windowed sums (diagnostic)
def run_tc_probe(args):
    """SURVEY.md §8(f) 4 / north_star: the tensor-core banded-correlation variant "must beat the CUDA-core version".
    For window lengths spanning the config-2 durations: linear_search_kernel (64 survey curves, one duration, statistics
    only) against cetra_tc_correlation_probe (mma.sync TF32 Toeplitz products, same number of outputs), both as
    (t0, point) template evaluations per second; the 3xTF32 split is what the 1e-5 parity bar needs."""
    import torch
    import paper_2503_20875_b200 as cetra
    from cetra_synth import make_survey_batch
    torch.cuda.set_device(0)
    p = make_survey_batch(n_lc=args.n_lc, lc_range=(0, args.n_lc))
    flux, err = torch.from_numpy(p.flux).cuda(), torch.from_numpy(p.flux_err).cuda()
    for k_taps in (17, 61, 121, 241, 361):
        dur = np.array([(k_taps - 0.5) * p.cadence])                 # a window of exactly k_taps samples
        for _ in range(3):
            cetra.cetra_linear_search(p.times, flux, err, dur, p.t0_start, p.t0_stride, p.n_t0, p.template,
                                      want_grids=False, want_stats=True)
        torch.cuda.synchronize()
        cetra.cetra_profile_enable(True)
        for _ in range(20):
            cetra.cetra_linear_search(p.times, flux, err, dur, p.t0_start, p.t0_stride, p.n_t0, p.template,
                                      want_grids=False, want_stats=True)
        torch.cuda.synchronize()
        pr = cetra.cetra_profile_read()
        cetra.cetra_profile_enable(False)
        cuda_ms = pr["linear_ms"] / pr["linear_launches"]
        n_out = args.n_lc * p.n_t0
        line = dict(workload="windowed sums of one duration, %d curves x %d t0 cells" % (args.n_lc, p.n_t0),
                    taps=k_taps, cuda_core=dict(kernel="linear_search_kernel", ms=cuda_ms,
                                                evals_per_s=n_out * k_taps / (cuda_ms * 1e-3)))
        for split in (True, False):
            r = cetra.cetra_tc_correlation_probe(n_out, k_taps, split=split, reps=20)
            line["tensor_3xtf32" if split else "tensor_1xtf32"] = r
        line["tensor_over_cuda_core"] = line["tensor_3xtf32"]["evals_per_s"] / line["cuda_core"]["evals_per_s"]
        print(json.dumps(line), flush=True)


def spawn_command(n_gpus: int, port: int, argv):
    """The torchrun command `python bench.py --gpus N` runs itself under when it was not started by torchrun."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_gpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *argv]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="sector", choices=["sector", "survey", "configs", "tc-probe"])
    ap.add_argument("--cfgs", default="1,2,3,4", help="--workload configs: which BASELINE configs to time")
    ap.add_argument("--n-lc", type=int, default=64, help="light curves per GPU per step (survey: per slice)")
    ap.add_argument("--lc-chunk", type=int, default=0, help="light curves resident at a time (0 = library default)")
    ap.add_argument("--survey-lc", type=int, default=10000)
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="CPU budget of the cpu_baseline sample")
    ap.add_argument("--ref-seconds", type=float, default=8.0, help="CPU budget of one --impl reference step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-legs", action="store_true", help="skip the `configs` list (other workloads' rooflines)")
    ap.add_argument("--legs-only", action="store_true",
                    help="run only the `configs` legs and print them (the command the ncu passes under profiles/ use)")
    ap.add_argument("--master-port", type=int, default=29541, help="rendezvous port when bench.py spawns the ranks")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.workload == "sector":
        # not under torchrun: start the N ranks ourselves (one process per GPU, rendezvous on 127.0.0.1)
        sys.exit(subprocess.call(spawn_command(args.gpus, args.master_port, sys.argv[1:])))
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.workload == "sector" and world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: refusing to report a number for "
                         f"a different GPU count")
    if args.impl == "reference":
        run_reference(args, rank)
    elif args.workload == "survey":
        run_survey(args)
    elif args.workload == "tc-probe":
        run_tc_probe(args)
    elif args.workload == "configs":
        run_configs(args)
    else:
        run_cuda(args, rank, world, local_rank)


if __name__ == "__main__":
    main()

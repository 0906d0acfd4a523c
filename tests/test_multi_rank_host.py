"""Multi-rank host logic of bench.py on CPU (gloo, world_size 2): the light-curve partition is exact and
disjoint, every rank draws the curves a single-process run would draw, and the reported time is the
maximum over ranks.  The data path itself has no collective (light curves are independent)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, per_rank, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        from cetra_synth import make_survey_batch
        lo, hi = bench.rank_slice(rank, world, per_rank)
        p = make_survey_batch(n_lc=per_rank * world, n_periods=16, lc_range=(lo, hi))
        ms = bench.max_over_ranks(10.0 + 5.0 * rank, torch.device("cpu"), world)
        # every rank's checksum to rank 0
        mine = torch.tensor([lo, hi, float(np.nansum(p.flux.astype(np.float64))), ms], dtype=torch.float64)
        got = [torch.zeros_like(mine) for _ in range(world)]
        dist.all_gather(got, mine)
        if rank == 0:
            out.put([g.tolist() for g in got])
    finally:
        dist.destroy_process_group()


def test_rank_partition_and_max_over_ranks():
    from cetra_synth import make_survey_batch
    world, per_rank = 2, 3
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, per_rank, out)) for r in range(world)]
    for pr in procs:
        pr.start()
    for pr in procs:
        pr.join(timeout=120)
        assert pr.exitcode == 0
    rows = out.get()
    full = make_survey_batch(n_lc=per_rank * world, n_periods=16)
    covered = []
    for r, (lo, hi, checksum, ms) in enumerate(rows):
        lo, hi = int(lo), int(hi)
        covered += list(range(lo, hi))
        assert np.isclose(checksum, np.nansum(full.flux[lo:hi].astype(np.float64)), rtol=0, atol=0)
        assert ms == 10.0 + 5.0 * (world - 1)          # the slowest rank's time, on every rank
    assert covered == list(range(per_rank * world))    # exact, disjoint, in order


def test_bench_spawns_its_own_ranks_and_refuses_a_mismatched_world(monkeypatch):
    """`python bench.py --gpus N` outside torchrun re-executes itself with N ranks on 127.0.0.1; started with a
    WORLD_SIZE that is not N it refuses to print a line (it used to report n_gpus 1 silently)."""
    import subprocess
    import sys

    import pytest

    import bench
    cmd = bench.spawn_command(8, 29999, ["--gpus", "8", "--steps", "2"])
    assert cmd[1:3] == ["-m", "torch.distributed.run"]
    assert "--nproc-per-node=8" in cmd and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29999"
    assert cmd[-4:] == ["--gpus", "8", "--steps", "2"] and cmd[-5].endswith("bench.py")
    monkeypatch.setenv("WORLD_SIZE", "1")
    monkeypatch.setenv("RANK", "0")
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "8"])
    with pytest.raises(SystemExit) as exc:
        bench.main()
    assert "refusing" in str(exc.value)

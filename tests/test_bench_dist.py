"""Host logic of bench.py's multi-rank path (replicas only) on CPU: two gloo ranks, the step
time is the maximum over ranks, the value the whole-job aggregate, and per-rank noise streams differ."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    import gp_workloads as W
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(dist, 10.0 + 5.0 * rank)
    _, xi, _ = bench.make_workload(W.CONFIGS[1], 256, "f64", rank)
    dist.barrier()
    out.put((rank, ms, float(xi[:8].sum())))
    dist.destroy_process_group()


def test_two_ranks_max_time_and_aggregate_value():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29600 + os.getpid() % 300
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == pytest.approx(15.0) and res[1][1] == pytest.approx(15.0)   # slowest rank, on every rank
    assert res[0][2] != res[1][2]                                                 # replicas draw different noise
    import bench
    assert bench.job_value(2, 1000, 15.0) == pytest.approx(2 * 1000 / 15e-3)
    assert bench.max_over_ranks(None, 3.0) == 3.0


def test_reference_arm_non_zero_rank_exits_quietly(monkeypatch, capsys):
    import argparse
    import bench
    monkeypatch.setenv("RANK", "1")
    bench.run_reference(argparse.Namespace(config=1, dtype="", n=0, reference_points=512, steps=1, warmup=0, ops=""))
    assert capsys.readouterr().out == ""

"""The N > 1 path of bench.py on CPU (gloo, world_size 2).  The hot path does not shard across GPUs
(BASELINE.json:north_star "no sharding and no multi-GPU collectives": replicas only), so the
only inter-rank logic is the timing reduction (max over ranks) and the whole-job value; both are exercised
here with two processes over 127.0.0.1."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    import torch
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    try:
        # rank 1 is the slower one on the first timing, rank 0 on the second
        got = bench.reduce_max_over_ranks([10.0 + rank, 5.0 - rank], dist, torch.device("cpu"))
        q.put((rank, got, bench.job_value(world, 1000, got[0])))
    finally:
        dist.destroy_process_group()


def test_timing_is_the_max_over_ranks_and_value_is_the_whole_job():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, value in res:
        assert got == [11.0, 5.0]                       # the slowest rank's time, on every rank
        assert value == pytest.approx(2 * 1000 / 11.0e-3)   # both ranks' cells over that time


def test_single_rank_is_the_identity():
    import bench
    assert bench.reduce_max_over_ranks([3.5, 1.25], None, None) == [3.5, 1.25]
    assert bench.job_value(1, 134217728, 13.2) == pytest.approx(134217728 / 13.2e-3)


def test_reference_arm_runs_on_rank_zero_only(monkeypatch, capsys):
    import argparse
    import bench
    monkeypatch.setenv("RANK", "1")
    args = argparse.Namespace(workload="config2", size=8, steps=1, warmup=3, gpus=2, impl="reference")
    assert bench.run_reference(args) is None
    assert capsys.readouterr().out == ""                 # the other ranks exit without work and print nothing

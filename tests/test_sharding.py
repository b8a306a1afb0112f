"""Host logic of a level sharded over GPUs, on the CPU:
the partition and exchange tables against their definition, and the halo exchange itself over torch.distributed
(gloo, world_size 2 and 3, 127.0.0.1) with numpy stand-ins for the device batches.  The device side (export / import
kernels, stepping only the owned patches, bitwise equality with the unsharded run) is tests/test_gpu_sharding.py."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wk
from paper_1412_0934_b200 import sharding as sh


def _level(npx=4, n=8, outflow=False):
    origin = wk.morton_patch_origins(npx, npx, npx, n)
    bc = (1, 1, 0, 0, 0, 0) if outflow else (0,) * 6
    return origin, n, (npx * n,) * 3, bc


@pytest.mark.parametrize("world", [1, 2, 3, 5, 8])
@pytest.mark.parametrize("outflow", [False, True])
def test_plans_match_their_definition(world, outflow):
    origin, n, dom, bc = _level(4, 8, outflow)
    npatch = len(origin)
    plans = sh.make_plans(origin, n, dom, bc, world)
    # owned ranges: a partition of 0 .. npatch-1 into contiguous pieces whose sizes differ by at most one
    allowned = np.concatenate([p.owned for p in plans])
    assert np.array_equal(allowned, np.arange(npatch))
    sizes = [len(p.owned) for p in plans]
    assert max(sizes) - min(sizes) <= 1
    owner = np.concatenate([np.full(len(p.owned), p.rank) for p in plans])
    # ghost lists against a brute-force statement of the rule: every remote patch within one patch of an owned one
    dims = np.array(dom) // n
    pc = origin // n
    for p in plans:
        expect = set()
        for i in p.owned:
            for j in range(npatch):
                if owner[j] == p.rank:
                    continue
                d = pc[j] - pc[i]
                near = True
                for a in range(3):
                    da = abs(int(d[a]))
                    if bc[2 * a] == 0:
                        da = min(da, int(dims[a]) - da)
                    near = near and da <= 1
                if near:
                    expect.add(j)
        assert set(p.ghost.tolist()) == expect
        assert np.array_equal(p.ghost, np.sort(p.ghost))
    # exchange tables: what r sends to q is exactly what q receives from r, in the same order
    for p in plans:
        for q, idx in p.send.items():
            glob = p.owned[idx]
            other = plans[q]
            slots = other.recv[p.rank]
            assert np.array_equal(other.local_to_global[slots], glob)
        got = np.concatenate([v for _, v in sorted(p.recv.items())]) if p.recv else np.zeros(0, np.int64)
        assert sorted(got.tolist()) == list(range(len(p.owned), len(p.owned) + len(p.ghost)))   # every copy is fed once
    if world == 1:
        assert len(plans[0].ghost) == 0 and not plans[0].send and not plans[0].recv


def test_owner_ranges_and_errors():
    assert sh.owner_ranges(10, 3).tolist() == [0, 3, 6, 10]
    with pytest.raises(ValueError):
        sh.owner_ranges(2, 3)


class _NumpyShard:
    """Stand-in for a device batch: the local state as a numpy array [nf, nlocal, n^3]."""

    def __init__(self, plan, U):
        self.plan = plan
        self.U = np.ascontiguousarray(U[:, plan.local_to_global]).reshape(U.shape[0], -1, U.shape[2] ** 3).copy()

    def export(self, idx):
        import torch
        return torch.from_numpy(np.ascontiguousarray(self.U[:, idx]))

    def alloc(self, count):
        import torch
        return torch.empty((self.U.shape[0], count, self.U.shape[2]), dtype=torch.float64)

    def import_(self, idx, buf):
        self.U[:, idx] = buf.numpy()


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    import torch.distributed as dist
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    try:
        origin, n, dom, bc = _level(4, 8, outflow=(world == 3))
        rng = np.random.default_rng([wk.SEED, 77])
        U = rng.standard_normal((3, len(origin), n, n, n))
        plan = sh.make_plans(origin, n, dom, bc, world)[rank]
        shard = _NumpyShard(plan, U)
        tr = sh.DistTransport(dist)
        ok = True
        for step in range(3):
            # "step": every rank changes its OWNED patches in a way every other rank can predict ...
            nown = len(plan.owned)
            shard.U[:, :nown] = shard.U[:, :nown] * 1.5 + (step + 1)
            U = U * 1.5 + (step + 1)
            # ... after the exchange the copies must hold the owners' new data, bit for bit
            sh.HaloExchange(plan).run(shard.export, shard.import_, shard.alloc, tr)
            want = U[:, plan.local_to_global].reshape(shard.U.shape)
            ok = ok and np.array_equal(shard.U, want)
            sm = tr.allreduce_max(float(rank + 10 * step))
            ok = ok and sm == float(world - 1 + 10 * step)
        q.put((rank, ok, len(plan.ghost)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_halo_exchange_over_gloo(world):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[0] for r in res] == list(range(world))
    assert all(r[1] for r in res), res
    assert all(r[2] > 0 for r in res)

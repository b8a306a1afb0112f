"""A level sharded over GPUs (SURVEY.md 8(f4); PAPER.md:70 "16 GPUs", :72 "one GPU per computing node ... communicating
through the network"): host-side partition and exchange tables, and the per-step sequence
exchange halos -> step -> all-reduce(max) of the signal speed.  No arithmetic of the method lives here: the step is
``amr_hydro_step`` / ``amr_mhd_step`` on the rank's own batch, the copies are ``amr_patch_batch_export`` /
``amr_patch_batch_import``, the transport is ``torch.distributed`` (NCCL on GPUs, gloo in the CPU tests) or, for several
emulated ranks inside one process, a plain device copy.

Partition: the patches of a level, in the caller's (space-filling-curve) order, are cut into ``world`` contiguous
ranges - the paper's own first step ("AMR cells are ordered according to a space filling curve based layout",
PAPER.md:55) is what makes a contiguous range a compact sub-volume.  A rank's batch holds its OWNED range first
(``nactive`` of them: stepped, reduced) and behind it read-only copies of every remote patch that touches an owned one
(26-neighbourhood, periodic wrap, nothing beyond an outflow face).  Before a step each rank sends the current state of
the owned patches its peers hold copies of - whole patches; the 2-cell-deep slabs the stencil needs would be enough,
that is the obvious next refinement - and receives its copies; the fused halo gather of the step kernel then reads them
like any sibling.  The only other exchange is the scalar max of the signal speed (dt and c_h are global).
"""
from __future__ import annotations

import dataclasses
from typing import Dict, List, Sequence

import numpy as np


@dataclasses.dataclass
class ShardPlan:
    rank: int
    world: int
    owned: np.ndarray                 # global patch indices this rank owns (a contiguous range, ascending)
    ghost: np.ndarray                 # global indices of the remote patches it keeps copies of (ascending)
    send: Dict[int, np.ndarray]       # peer -> LOCAL indices (into owned) of the patches the peer needs, in the peer's ghost order
    recv: Dict[int, np.ndarray]       # peer -> LOCAL indices (owned.size + position in ghost) the peer's patches land in

    @property
    def local_to_global(self) -> np.ndarray:
        return np.concatenate([self.owned, self.ghost]).astype(np.int64)


def owner_ranges(npatch: int, world: int) -> np.ndarray:
    """Range boundaries [world + 1]: rank r owns [b[r], b[r+1]); sizes differ by at most one."""
    if world < 1 or npatch < world:
        raise ValueError("need at least one patch per rank")
    return np.array([(npatch * r) // world for r in range(world + 1)], dtype=np.int64)


def neighbour_patches(origin: np.ndarray, n: int, domain_cells: Sequence[int], bc: Sequence[int]) -> List[np.ndarray]:
    """For every patch the global indices of the patches in its 26-neighbourhood (periodic faces wrap, nothing lies
    beyond an outflow face, holes of a refined level are skipped), itself excluded."""
    origin = np.asarray(origin, dtype=np.int64).reshape(-1, 3)
    dims = [int(d) // n for d in domain_cells]
    where = {(int(o[0]) // n, int(o[1]) // n, int(o[2]) // n): i for i, o in enumerate(origin)}
    out = []
    for i, o in enumerate(origin):
        pc = (int(o[0]) // n, int(o[1]) // n, int(o[2]) // n)
        found = set()
        for dz in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dx in (-1, 0, 1):
                    q, ok = [pc[0] + dx, pc[1] + dy, pc[2] + dz], True
                    for a in range(3):
                        if q[a] < 0:
                            if bc[2 * a] == 0:
                                q[a] += dims[a]
                            else:
                                ok = False
                        elif q[a] >= dims[a]:
                            if bc[2 * a + 1] == 0:
                                q[a] -= dims[a]
                            else:
                                ok = False
                    j = where.get(tuple(q)) if ok else None
                    if j is not None and j != i:
                        found.add(j)
        out.append(np.array(sorted(found), dtype=np.int64))
    return out


def make_plans(origin: np.ndarray, n: int, domain_cells: Sequence[int], bc: Sequence[int], world: int) -> List[ShardPlan]:
    """The plans of ALL ranks (pure function of the level's geometry: every rank computes the same tables, so building
    them needs no communication)."""
    origin = np.asarray(origin).reshape(-1, 3)
    npatch = origin.shape[0]
    b = owner_ranges(npatch, world)
    owner = np.searchsorted(b, np.arange(npatch), side="right") - 1
    nbrs = neighbour_patches(origin, n, domain_cells, bc)
    ghosts = []
    for r in range(world):
        g = set()
        for i in range(int(b[r]), int(b[r + 1])):
            g.update(int(j) for j in nbrs[i] if owner[j] != r)
        ghosts.append(np.array(sorted(g), dtype=np.int64))
    plans = []
    for r in range(world):
        owned = np.arange(int(b[r]), int(b[r + 1]), dtype=np.int64)
        send, recv = {}, {}
        for q in range(world):
            if q == r:
                continue
            need = ghosts[q][owner[ghosts[q]] == r]          # what q keeps of r's patches, in q's ghost order
            if need.size:
                send[q] = (need - b[r]).astype(np.int64)
            mine = np.nonzero(owner[ghosts[r]] == q)[0]      # positions in r's ghost list that come from q
            if mine.size:
                recv[q] = (owned.size + mine).astype(np.int64)
        plans.append(ShardPlan(r, world, owned, ghosts[r], send, recv))
    return plans


def local_level_arrays(plan: ShardPlan, origin: np.ndarray, U: np.ndarray):
    """(origin, U) of the rank's batch: owned patches first, then the copies (data of the initial state)."""
    idx = plan.local_to_global
    return np.ascontiguousarray(np.asarray(origin).reshape(-1, 3)[idx]).astype(np.int32), np.ascontiguousarray(U[:, idx])


class HaloExchange:
    """The per-step exchange of one rank, written over four callables so that the same host logic drives device batches
    (ShardedBatch below) and the numpy stand-ins of the CPU tests:
      export(local_indices) -> packed buffer [nfields, count, n^3]      import_(local_indices, packed)
      transport.exchange(rank, {peer: send buffer}, {peer: empty recv buffer}) -> fills the recv buffers."""

    def __init__(self, plan: ShardPlan):
        self.plan = plan

    def run(self, export, import_, alloc, transport):
        p = self.plan
        sendbuf = {q: export(idx) for q, idx in sorted(p.send.items())}
        recvbuf = {q: alloc(len(idx)) for q, idx in sorted(p.recv.items())}
        transport.exchange(p.rank, sendbuf, recvbuf)
        for q, idx in sorted(p.recv.items()):
            import_(idx, recvbuf[q])


class DistTransport:
    """torch.distributed point-to-point (NCCL on device tensors, gloo on CPU tensors): one batched isend/irecv group."""

    def __init__(self, dist):
        self.dist = dist

    def exchange(self, rank, sendbuf, recvbuf):
        ops = []
        for q in sorted(set(sendbuf) | set(recvbuf)):
            # lower rank first on both sides of a pair, so that gloo (which matches in order) cannot deadlock
            first_send = rank < q
            for is_send in ((True, False) if first_send else (False, True)):
                if is_send and q in sendbuf:
                    ops.append(self.dist.P2POp(self.dist.isend, sendbuf[q], q))
                if not is_send and q in recvbuf:
                    ops.append(self.dist.P2POp(self.dist.irecv, recvbuf[q], q))
        if ops:
            for w in self.dist.batch_isend_irecv(ops):
                w.wait()

    def allreduce_max(self, value: float) -> float:
        import torch
        t = torch.tensor([float(value)], dtype=torch.float64)
        if self.dist.get_backend() == "nccl":
            t = t.cuda()
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())


class LocalTransport:
    """Several emulated ranks inside ONE process (single-GPU tests): rank r's send buffers are parked, and handed to
    the receiving rank when it runs its exchange; call `exchange` for every rank twice per step (post, then collect)
    through `exchange_all`."""

    def __init__(self, world: int):
        self.world = world
        self.box = {}

    def exchange_all(self, shards):
        self.box = {}
        posts = []
        for sh in shards:
            p = sh.plan
            for q, idx in sorted(p.send.items()):
                self.box[(p.rank, q)] = sh.export(idx)
            posts.append(p)
        for sh in shards:
            p = sh.plan
            for q, idx in sorted(p.recv.items()):
                sh.import_(idx, self.box[(q, p.rank)])

    @staticmethod
    def allreduce_max(values):
        return max(values)


class ShardedBatch:
    """One rank's share of a level: a PatchBatch of owned patches + read-only copies, and its exchange."""

    def __init__(self, plan: ShardPlan, level, dtype: int, device: str = "cuda:0"):
        import torch
        from . import binding
        self._torch = torch
        self.plan = plan
        origin, U = local_level_arrays(plan, level.origin, level.U)
        self.batch = binding.PatchBatch(len(origin), level.n, level.nfields, dtype, level.dx, origin=origin,
                                        domain_cells=level.domain_cells, bc=level.bc, self_periodic=False,
                                        nghost=level.g, level=level.level, device=device, nactive=len(plan.owned))
        self.batch.upload(np.ascontiguousarray(U.astype(binding._np_dtype(dtype))))
        self.tdtype = torch.float64 if dtype == binding.AMR_F64 else torch.float32
        self.device = self.batch.device
        self._pairs = {}

    def _pair_table(self, idx: np.ndarray):
        key = idx.tobytes()
        t = self._pairs.get(key)
        if t is None:
            pairs = np.stack([np.arange(len(idx)), np.asarray(idx)], axis=1).astype(np.int32)
            t = self._torch.from_numpy(np.ascontiguousarray(pairs)).to(self.device)
            self._pairs[key] = t
        return t

    def alloc(self, count: int):
        b = self.batch
        return self._torch.empty((b.nfields, count, b.n ** 3), dtype=self.tdtype, device=self.device)

    def export(self, idx: np.ndarray):
        buf = self.alloc(len(idx))
        self.batch.export_patches(self._pair_table(idx), len(idx), buf)
        return buf

    def import_(self, idx: np.ndarray, buf):
        self.batch.import_patches(self._pair_table(idx), len(idx), buf)

    def exchange(self, transport):
        HaloExchange(self.plan).run(self.export, self.import_, self.alloc, transport)

    def owned_state(self) -> np.ndarray:
        return self.batch.download()[:, :len(self.plan.owned)]


def sharded_step(shard: ShardedBatch, transport, wl, first: bool = False):
    """One step of one rank under torch.distributed: refresh the copies, global dt and c_h from the all-reduced signal
    speed, step the owned patches.  (The all-reduce is also what orders the steps: no rank starts step s+1, whose
    exchange overwrites the copies its peers' step s reads, before every rank has finished step s.)"""
    shard.exchange(transport)
    _, sm_local = shard.batch.cfl_dt(wl.gamma, wl.cfl)
    sm = transport.allreduce_max(sm_local)
    dt = wl.cfl * shard.batch.dx / sm
    if wl.mhd:
        shard.batch.mhd_step(dt, wl.gamma, wl.limiter, wl.riemann, sm, wl.alpha)
    else:
        shard.batch.hydro_step(dt, wl.gamma, wl.limiter, wl.riemann)
    return dt, sm

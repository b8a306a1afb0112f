"""-m gpu: a level sharded over several ranks gives bit for bit the state of the
unsharded run.  Only one GPU is available, so the ranks are emulated inside one process on one device (each rank has
its own batch with its own arena; the transport is a device copy) - every kernel is launched by exactly one rank at a
time and none waits on another, so this is the same sequence of launches a multi-process run issues.  The
torch.distributed transport itself is covered on the CPU (tests/test_sharding.py, gloo)."""
import numpy as np
import pytest

import workloads as wk

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    import gpu_harness
    return gpu_harness


def _run_sharded(wl, world, np_dtype, nsteps, H):
    import paper_1412_0934_b200 as amr
    from paper_1412_0934_b200 import sharding as sh
    lev = wl.levels[0]
    plans = sh.make_plans(lev.origin, lev.n, lev.domain_cells, lev.bc, world)
    shards = [sh.ShardedBatch(p, lev, H.gpu_dtype(np_dtype)) for p in plans]
    tr = sh.LocalTransport(world)
    dts = []
    for _ in range(nsteps):
        tr.exchange_all(shards)
        sm = tr.allreduce_max([s.batch.cfl_dt(wl.gamma, wl.cfl)[1] for s in shards])
        dt = wl.cfl * lev.dx / sm
        for s in shards:
            H.gpu_step(s.batch, wl, dt, sm)
        dts.append(dt)
    U = np.empty(lev.U.shape, dtype=np_dtype)
    for s in shards:
        U[:, s.plan.owned] = s.owned_state()
    counters = {}
    for s in shards:
        for k, v in s.batch.step_counters().items():
            counters[k] = counters.get(k, 0) + v
    tot = sum(s.batch.conserved_totals() for s in shards)
    return U, dts, counters, tot, shards


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
@pytest.mark.parametrize("world", [2, 3, 8])
def test_sharded_mhd_run_is_bitwise_the_unsharded_run(H, np_dtype, world):
    """Config 3 at 64^3 (64 patches of 16^3, periodic), MHD, 3 steps: dt, state, counters and totals."""
    wl = wk.config3_orszag_tang(N=64)
    lev = wl.levels[0]
    ref = H.gpu_advance(lev, wl, 3, np_dtype=np_dtype)
    U, dts, counters, tot, shards = _run_sharded(wl, world, np_dtype, 3, H)
    assert dts == ref["dts"]
    assert np.array_equal(U, ref["U"])
    assert counters == ref["counters"]
    ref_tot = ref["batch"].conserved_totals()
    assert np.abs(tot - ref_tot).max() <= 1e-12 * np.abs(ref_tot).max()     # per-rank partial sums: another summation order
    # the ranks own disjoint ranges (in a 4x4x4 periodic patch grid the copies cover most of the rest)
    assert sum(len(s.plan.owned) for s in shards) == lev.npatch and all(s.batch.nactive == len(s.plan.owned) for s in shards)


def test_sharded_hydro_run_with_outflow_faces_and_32_cubed_patches(H):
    """Config-1-like: outflow faces, 2x2x2 patches of 32^3, hydro fp64, 4 ranks (a rank's range then has neighbours
    beyond outflow faces that do not exist)."""
    n, N = 32, 64
    rng = np.random.default_rng([wk.SEED, 88])
    c = (np.arange(N) + 0.5) / N
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    rho = 1.0 + 0.5 * np.exp(-30 * ((X - 0.5) ** 2 + (Y - 0.4) ** 2 + (Z - 0.6) ** 2)) + 0.01 * rng.standard_normal((N, N, N))
    p = 1.0 + 1.5 * np.exp(-30 * ((X - 0.5) ** 2 + (Y - 0.4) ** 2 + (Z - 0.6) ** 2))
    G = wk.primitive_to_conserved(rho, [0.1 + 0 * X, 0 * X, -0.2 + 0 * X], p, 1.4)
    wl = wk.uniform_grid_workload("shard_outflow", G, n, 1.4, False, 2, 1, 0.4, 2)
    wl.levels[0].bc = (wk.configs.BC_OUTFLOW,) * 6
    ref = H.gpu_advance(wl.levels[0], wl, 2)
    U, dts, counters, tot, _ = _run_sharded(wl, 4, np.float64, 2, H)
    assert dts == ref["dts"] and np.array_equal(U, ref["U"])


def test_only_owned_patches_are_stepped_and_reduced(H):
    import paper_1412_0934_b200 as amr
    wl = wk.config2_random_patches(npatch=8)
    lev = wl.levels[0]
    origin = wk.morton_patch_origins(2, 2, 2, 16)
    b = amr.PatchBatch(8, 16, 5, amr.AMR_F64, lev.dx, origin=origin, domain_cells=(32,) * 3, bc=(0,) * 6, nactive=5)
    b.upload(lev.U)
    dt, sm = b.cfl_dt(wl.gamma, wl.cfl)
    b.hydro_step(dt, wl.gamma, wl.limiter, wl.riemann)
    U = b.download()
    assert np.array_equal(U[:, 5:], lev.U[:, 5:])                       # the copies are untouched
    assert np.abs(U[:, :5] - lev.U[:, :5]).max() > 1e-3
    full = amr.PatchBatch(8, 16, 5, amr.AMR_F64, lev.dx, origin=origin, domain_cells=(32,) * 3, bc=(0,) * 6)
    full.upload(lev.U)
    full.hydro_step(dt, wl.gamma, wl.limiter, wl.riemann)
    assert np.array_equal(U[:, :5], full.download()[:, :5])
    assert np.allclose(b.conserved_totals(), U[:, :5].sum(axis=(1, 2, 3, 4)), rtol=1e-13)
    with pytest.raises(amr.AmrError):
        amr.PatchBatch(8, 16, 5, amr.AMR_F64, lev.dx, origin=origin, domain_cells=(32,) * 3, bc=(0,) * 6, nactive=9)

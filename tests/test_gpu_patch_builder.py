"""-m gpu parity of the patch builder against oracle/patch_builder.py:
integer and index work, so everything is compared bit for bit -- curve order, patch table (first cell, level,
origin) and the gathered fields -- on the seeded refined-level workload and on the edge cases."""
import numpy as np
import pytest

import workloads as wk

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pbo():
    from oracle import patch_builder
    return patch_builder


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    return torch


def _check_build(amr, torch, pbo, xyz, bits, kmax, fields=None, gather_levels=()):
    b = amr.PatchBuilder(xyz.shape[1])
    np_gpu = b.build(torch.from_numpy(xyz).cuda(), bits, kmax)
    perm, first, level, origin = b.results()
    operm, okeys = pbo.curve_order(xyz, bits)
    ofirst, olevel = pbo.build_patches(okeys, kmax)
    assert np.array_equal(perm, operm)
    assert np_gpu == len(ofirst)
    assert np.array_equal(first, ofirst) and np.array_equal(level, olevel)
    assert np.array_equal(origin, pbo.patch_origins(okeys, ofirst, bits))
    for k in gather_levels:
        out, org = b.gather(torch.from_numpy(fields).cuda(), k)
        ref, oorg = pbo.gather_level(fields, operm, okeys, ofirst, olevel, k, bits)
        assert b.count(k) == ref.shape[1]
        assert np.array_equal(out.cpu().numpy(), ref) and np.array_equal(org, oorg)
    return b, level


@pytest.mark.parametrize("bits,kmax", [(6, 5), (7, 3), (7, 5)])
def test_refined_level_workload(torch_cuda, pbo, bits, kmax):
    import paper_1412_0934_b200 as amr
    xyz, F = wk.refined_level_cells(bits)
    _, level = _check_build(amr, torch_cuda, pbo, xyz, bits, kmax, F, gather_levels=range(0, kmax + 1))
    assert len(np.unique(level)) >= 3            # the workload exercises several patch sizes


def test_gather_fp64_and_ragged_size(torch_cuda, pbo):
    """ncell not a multiple of any block size (4096-item sort blocks, 1024-item compaction blocks): cells
    dropped from the workload punch holes into the patches; fp64 fields."""
    import paper_1412_0934_b200 as amr
    xyz, F = wk.refined_level_cells(6, dtype=np.float64, stream=1)
    keep = 65536 - 4096 - 777
    _check_build(amr, torch_cuda, pbo, np.ascontiguousarray(xyz[:, :keep]), 6, 4, np.ascontiguousarray(F[:, :keep]), gather_levels=(1, 2))


def test_edge_cases(torch_cuda, pbo):
    import paper_1412_0934_b200 as amr
    torch = torch_cuda
    # a complete grid: one patch per 2^kmax cube; with kmax = bits a single patch
    g = np.arange(16)
    full = np.stack(np.meshgrid(g, g, g, indexing="ij")).reshape(3, -1).astype(np.int32)
    rng = np.random.default_rng(1)
    full = np.ascontiguousarray(full[:, rng.permutation(full.shape[1])])
    F = rng.standard_normal((2, full.shape[1])).astype(np.float32)
    b, level = _check_build(amr, torch, pbo, full, 4, 4, F, gather_levels=(4,))
    assert b.npatch == 1 and level[0] == 4
    b, level = _check_build(amr, torch, pbo, full, 4, 2, F, gather_levels=(2,))
    assert b.npatch == 64 and (level == 2).all()
    b, level = _check_build(amr, torch, pbo, full, 4, 0, F, gather_levels=(0,))
    assert b.npatch == 4096
    # a single cell; the largest coordinates (bits = 10: four 8-bit sort passes, keys up to 2^30 - 1)
    one = np.array([[5], [1], [2]], np.int32)
    _check_build(amr, torch, pbo, one, 3, 3, np.ones((1, 1), np.float32), gather_levels=(0,))
    big = rng.integers(0, 1024, size=(3, 20000)).astype(np.int32)
    big = np.unique(big, axis=1)
    cube = np.stack(np.meshgrid(g[:8] + 1016, g[:8] + 1016, g[:8] + 1016, indexing="ij")).reshape(3, -1).astype(np.int32)
    big = np.unique(np.concatenate([big, cube], axis=1), axis=1)
    big = np.ascontiguousarray(big[:, rng.permutation(big.shape[1])])
    b, level = _check_build(amr, torch, pbo, big, 10, 5, rng.standard_normal((3, big.shape[1])).astype(np.float32), gather_levels=(0, 3))
    assert (level == 3).sum() >= 1


def test_rejects_bad_input(torch_cuda):
    import paper_1412_0934_b200 as amr
    torch = torch_cuda
    b = amr.PatchBuilder(100)
    xyz = torch.zeros((3, 10), dtype=torch.int32, device="cuda")          # ten copies of one cell
    with pytest.raises(amr.AmrError):
        b.build(xyz, 4, 2)
    ok = torch.arange(30, dtype=torch.int32, device="cuda").reshape(3, 10).contiguous()
    for bits, kmax in ((0, 0), (11, 2), (4, 6), (3, 4)):
        with pytest.raises(amr.AmrError):
            b.build(ok, bits, kmax)
    with pytest.raises(amr.AmrError):
        b.results()                                                         # no successful build yet
    with pytest.raises(amr.AmrError):
        b.build(torch.zeros((3, 101), dtype=torch.int32, device="cuda"), 4, 2)   # more cells than the workspace holds
    assert b.build(ok, 6, 2) == 10


def test_built_batch_feeds_the_solver(torch_cuda):
    """The builder's output IS the solver's input format: a scrambled cell list of the 64^3 Orszag-Tang grid is
    built into 16^3 patches, gathered, handed to amr_patch_batch_* with the builder's origins, and stepped; the
    result equals, bit for bit, the step on the patches cut directly from the grid."""
    import paper_1412_0934_b200 as amr
    torch = torch_cuda
    w = wk.config3_orszag_tang(N=64)
    lev = w.levels[0]
    G = wk.configs.join_patches(lev.U, lev.origin, (64, 64, 64))            # [9, z, y, x]
    rng = np.random.default_rng(7)
    z, y, x = np.meshgrid(np.arange(64), np.arange(64), np.arange(64), indexing="ij")
    order = rng.permutation(64 ** 3)
    xyz = np.ascontiguousarray(np.stack([x.ravel(), y.ravel(), z.ravel()])[:, order].astype(np.int32))
    F = np.ascontiguousarray(G.reshape(9, -1)[:, order])
    b = amr.PatchBuilder(xyz.shape[1])
    assert b.build(torch.from_numpy(xyz).cuda(), 6, 4) == 64
    out, origin = b.gather(torch.from_numpy(F).cuda(), 4)
    results = []
    for U, org in ((out.cpu().numpy(), origin), (lev.U, lev.origin)):
        pb_ = amr.PatchBatch(64, 16, 9, amr.AMR_F64, lev.dx, origin=org, domain_cells=(64, 64, 64), bc=(0,) * 6)
        pb_.upload(np.ascontiguousarray(U))
        dt, sm = pb_.cfl_dt(w.gamma, w.cfl)
        pb_.mhd_step(dt, w.gamma, w.limiter, w.riemann, sm, w.alpha)
        results.append(wk.configs.join_patches(pb_.download(), np.asarray(org), (64, 64, 64)))
    assert np.array_equal(results[0], results[1])

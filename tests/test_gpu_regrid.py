"""-m gpu parity of regridding between steps: amr_flag_blocks and amr_regrid_fill against
oracle/regrid.py, then the regridded hierarchy stepped on the device against the oracle's hierarchy step."""
import copy

import numpy as np
import pytest

import workloads as wk

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    import gpu_harness
    return gpu_harness


def _new_level2(wl, flags, n):
    l0, l1, l2 = wl.levels
    grid = wk.patch_flags_to_block_grid(l1, flags)
    cover1 = wk.origins_to_blocks(l1.origin, n, l0.domain_cells[0] // (n // 2))
    return wk.blocks_to_origins(wk.select_blocks(grid, cover1, grow=False), n)


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
def test_regrid_between_two_root_steps(oracle, H, np_dtype):
    import paper_1412_0934_b200 as amr
    from oracle import regrid as rg
    f32 = np_dtype == np.float32
    wl = copy.deepcopy(wk.config_hierarchy(True, 3, 256, n=16))
    if f32:
        for lv in wl.levels:
            lv.U = lv.U.astype(np.float32).astype(np.float64)
    n = 16
    h = amr.Hierarchy.from_workload(wl, H.gpu_dtype(np_dtype))
    dt0, sm = h.cfl_dt(wl.gamma, wl.cfl)
    h.step(dt0, wl.gamma, wl.limiter, wl.riemann, sm, wl.alpha, True)
    # the oracle regrids the state the device holds now
    for lv, b in zip(wl.levels, h.levels):
        lv.U = b.download().astype(np.float64)
    l0, l1, l2 = wl.levels
    thr = 3.0 * float(l1.U[0].mean())
    if f32:
        thr = float(np.float32(thr))
    flags = h.levels[1].flag_blocks(0, thr)
    assert np.array_equal(flags, rg.flag_blocks(l1, 0, thr))                 # a comparison per cell: exact
    origin_new = _new_level2(wl, flags, n)
    old = {tuple(o) for o in l2.origin}
    kept = sum(tuple(o) in old for o in origin_new)
    assert kept >= 3 and len(origin_new) - kept >= 3, (kept, len(origin_new))   # both branches are exercised
    ref2 = rg.regrid_fill(l1, l2, origin_new)
    lev2 = wk.Level(n=n, g=l0.g, level=2, dx=l2.dx, origin=origin_new, domain_cells=l2.domain_cells, bc=l2.bc,
                    self_periodic=False, U=ref2)
    b2 = amr.PatchBatch.from_level(lev2, H.gpu_dtype(np_dtype))               # uploads ref2 ...
    b2.upload(np.zeros_like(ref2))                                            # ... which is wiped again
    b2.regrid_fill(h.levels[2], h.levels[1])
    got2 = b2.download().astype(np.float64)
    for p, o in enumerate(origin_new):
        if tuple(o) in old:
            assert np.array_equal(got2[:, p], ref2[:, p])                     # kept patches: bitwise
    scale = np.abs(ref2).max(axis=(1, 2, 3, 4), keepdims=True)
    assert (np.abs(got2 - ref2) / scale).max() <= (4e-7 if f32 else 1e-15)    # new-born: one fma rounding apart
    # composite totals unchanged by the regrid (device data)
    g = l0.g
    before = oracle.hierarchy_totals([oracle.ghosted(lv.U, g) for lv in wl.levels], wl.levels)
    wl.levels[2] = lev2
    lev2.U = got2
    after = oracle.hierarchy_totals([oracle.ghosted(lv.U, g) for lv in wl.levels], wl.levels)
    absn = np.array([np.abs(l0.U[f]).sum() * l0.dx ** 3 for f in range(9)])
    assert (np.abs(after - before)[:8] / absn[:8]).max() <= (2e-7 if f32 else 1e-13)
    # relink and take the next root step on the new hierarchy
    h.replace_level(2, b2)
    h2 = h
    dt1, sm1 = h2.cfl_dt(wl.gamma, wl.cfl)
    h2.step(dt1, wl.gamma, wl.limiter, wl.riemann, sm1, wl.alpha, True)
    ref = oracle.hierarchy_step(wl, eps=oracle.default_eps(np_dtype))
    assert abs(dt1 - ref["dt0"]) <= (4e-6 if f32 else 1e-13) * ref["dt0"]
    ps = ref["smax"] * np.abs(ref["U"][0][5:8]).max()
    for l in range(3):
        got = h2.levels[l].download().astype(np.float64)
        for grp in H.field_groups(9):
            den = np.abs(ref["U"][l][grp]).max()
            if grp == [8]:
                den = max(den, ps)
            e = np.abs(got[grp] - ref["U"][l][grp]).max(axis=0) / den
            if f32:
                assert np.quantile(e, 0.9999) <= 4e-5 and int((e > 8e-5).sum()) <= 8, (l, grp, e.max())
            else:
                assert e.max() <= 4e-12, (l, grp, e.max())


def test_regrid_rejects_a_patch_outside_the_coarse_level(H):
    import paper_1412_0934_b200 as amr
    wl = wk.config_hierarchy(False, 3, 256, n=16)
    l0, l1, l2 = wl.levels
    b1 = amr.PatchBatch.from_level(l1, amr.AMR_F64)
    cover1 = wk.origins_to_blocks(l1.origin, 16, l0.domain_cells[0] // 8)
    up = np.repeat(np.repeat(np.repeat(cover1, 2, 0), 2, 1), 2, 2)
    bz, by, bx = np.nonzero(~up)
    bad = np.array([[bx[0] * 16, by[0] * 16, bz[0] * 16]], np.int32)           # a level-2 patch where level 1 is absent
    lev = wk.Level(n=16, g=3, level=2, dx=l2.dx, origin=bad, domain_cells=l2.domain_cells, bc=l2.bc,
                   self_periodic=False, U=np.zeros((5, 1, 16, 16, 16)))
    b2 = amr.PatchBatch.from_level(lev, amr.AMR_F64)
    with pytest.raises(amr.AmrError):
        b2.regrid_fill(None, b1)


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
@pytest.mark.parametrize("n", [8, 16])
def test_regrid_fill_with_new_born_patches_on_outflow_faces(H, n, np_dtype):
    """amr_regrid_fill where the new patches touch non-periodic domain faces (outflow x and z, periodic y), on the
    faces, edges and a corner of the domain, beside interior ones: the O8 stencil clamps at the outflow faces and wraps
    across the periodic one, against oracle/regrid.py."""
    import paper_1412_0934_b200 as amr
    from oracle import regrid as rg
    rng = np.random.default_rng([wk.SEED, 97, n])
    N = 4 * n
    G = np.exp(0.5 * rng.standard_normal((5, N, N, N)))
    bc = (1, 1, 0, 0, 1, 1)
    origin0 = wk.morton_patch_origins(4, 4, 4, n)
    l0 = wk.Level(n=n, g=3, level=0, dx=1.0 / N, origin=origin0, domain_cells=(N, N, N), bc=bc, self_periodic=False,
                  U=wk.split_into_patches(G, n, origin0).astype(np_dtype).astype(np.float64))
    F = 2 * N - n                                                   # fine origin of the last patch along an axis
    origin_new = np.array([[0, 0, 0], [F, 0, 0], [0, F, F], [F, F, F], [0, 3 * n, 2 * n], [3 * n, 0, F], [2 * n, F, 0],
                           [3 * n, 3 * n, 3 * n], [4 * n, 3 * n, 3 * n]], np.int32)
    ref = rg.regrid_fill(l0, None, origin_new)
    dt_ = H.gpu_dtype(np_dtype)
    b0 = amr.PatchBatch.from_level(l0, dt_)
    lev1 = wk.Level(n=n, g=3, level=1, dx=0.5 / N, origin=origin_new, domain_cells=(2 * N,) * 3, bc=bc, self_periodic=False,
                    U=np.zeros((5, len(origin_new), n, n, n)))
    b1 = amr.PatchBatch.from_level(lev1, dt_)
    b1.regrid_fill(None, b0)
    got = b1.download().astype(np.float64)
    tol = 1e-6 if np_dtype == np.float32 else 1e-15
    assert np.abs(got - ref).max() <= tol * np.abs(ref).max(), np.abs(got - ref).max()
    # children average to their parents on the device too (conservation of the transfer)
    h = n // 2
    mean = got.reshape(5, len(origin_new), h, 2, h, 2, h, 2).mean(axis=(3, 5, 7))
    Gc = wk.configs.join_patches(l0.U, l0.origin, (N, N, N))
    for p, o in enumerate(origin_new):
        par = Gc[:, o[2] // 2:o[2] // 2 + h, o[1] // 2:o[1] // 2 + h, o[0] // 2:o[0] // 2 + h]
        assert np.abs(mean[:, p] - par).max() <= (2e-6 if np_dtype == np.float32 else 1e-14) * np.abs(par).max()

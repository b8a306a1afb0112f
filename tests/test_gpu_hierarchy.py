"""-m gpu parity of the L-level hierarchy step: amr_hierarchy_step against
oracle.api.hierarchy_step on the same seeded three-level hierarchy, element by element on every level,
plus composite conservation of the GPU result and the link bookkeeping of a middle level."""
import numpy as np
import pytest

import workloads as wk

pytestmark = pytest.mark.gpu

TOL64_STEP = 1e-12
TOL32 = 1e-5


@pytest.fixture(scope="module")
def H():
    import gpu_harness
    return gpu_harness


@pytest.fixture(scope="module")
def hierarchies():
    # 256^3 finest index space, 16^3 patches (the d1 / x2 kernels): 64 root patches, ~75 level-1, ~11 level-2
    return {mhd: wk.config_hierarchy(mhd, 3, 256, n=16) for mhd in (False, True)}


def _absn(l0):
    return np.array([np.abs(l0.U[f]).sum() * l0.dx ** 3 for f in range(l0.nfields)])


@pytest.mark.parametrize("mhd", [False, True])
def test_three_level_step_fp64(oracle, H, hierarchies, mhd):
    wl = hierarchies[mhd]
    assert all(lv.npatch >= 4 for lv in wl.levels), wl.note
    ref = oracle.hierarchy_step(wl)
    got = H.gpu_hierarchy_step(wl)
    assert abs(got["dt0"] - ref["dt0"]) <= 1e-13 * ref["dt0"]
    ps = ref["smax"] * max(np.abs(ref["U"][0][5:8]).max(), 1e-300) if mhd else None
    for l in range(3):
        e = H.rel_err(got["U"][l], ref["U"][l], psi_scale=ps)
        assert e.max() <= 4 * TOL64_STEP, (l, e)       # level l took 2^l steps
    g = wl.levels[0].g
    tot = oracle.hierarchy_totals([oracle.ghosted(u, g) for u in got["U"]], wl.levels)
    nfc = 8 if mhd else 5
    assert (np.abs(tot - ref["totals_before"])[:nfc] / _absn(wl.levels[0])[:nfc]).max() <= 1e-13


@pytest.mark.parametrize("mhd", [False, True])
def test_three_level_step_fp32(oracle, H, hierarchies, mhd):
    import copy
    wl = copy.deepcopy(hierarchies[mhd])
    for lv in wl.levels:
        lv.U = lv.U.astype(np.float32).astype(np.float64)
    ref = oracle.hierarchy_step(wl, eps=oracle.default_eps(np.float32))
    got = H.gpu_hierarchy_step(wl, np_dtype=np.float32)
    assert abs(got["dt0"] - ref["dt0"]) <= 4e-6 * ref["dt0"]
    ps = ref["smax"] * max(np.abs(ref["U"][0][5:8]).max(), 1e-300) if mhd else None
    # level l took 2^l fp32 steps; the discontinuous decisions of the solver (HLL fallback, degenerate-B
    # branch) can flip between the fp32 kernel and the fp64 oracle at a few faces: all but
    # a handful of cells meet the bound
    nf = wl.levels[0].nfields
    for l in range(3):
        for grp in H.field_groups(nf):
            den = np.abs(ref["U"][l][grp]).max()
            if grp == [8]:
                den = max(den, ps)
            e = np.abs(got["U"][l][grp].astype(np.float64) - ref["U"][l][grp]).max(axis=0) / den
            assert np.quantile(e, 0.9999) <= 4 * TOL32, (l, grp, np.quantile(e, 0.9999))
            assert int((e > 8 * TOL32).sum()) <= 8, (l, grp, int((e > 8 * TOL32).sum()), e.max())
    g = wl.levels[0].g
    tot = oracle.hierarchy_totals([oracle.ghosted(u.astype(np.float64), g) for u in got["U"]], wl.levels)
    nfc = 8 if mhd else 5
    assert (np.abs(tot - ref["totals_before"])[:nfc] / _absn(wl.levels[0])[:nfc]).max() <= 4e-6


def test_without_reflux_the_gpu_result_matches_the_oracle_without_reflux(oracle, H, hierarchies):
    """do_reflux = 0 reaches the kernels: same comparison, and the totals leak as the oracle's do."""
    wl = hierarchies[False]
    ref = oracle.hierarchy_step(wl, do_reflux=False)
    got = H.gpu_hierarchy_step(wl, do_reflux=False)
    for l in range(3):
        assert H.rel_err(got["U"][l], ref["U"][l]).max() <= 4 * TOL64_STEP
    assert (np.abs(ref["totals_after"] - ref["totals_before"])[:5] / _absn(wl.levels[0])[:5]).max() > 1e-8


def test_three_root_steps_fp64(oracle, H, hierarchies):
    """Three root steps in a row (flux registers cleared and reused, buffers ping-ponged on every level)."""
    import copy
    wl = copy.deepcopy(hierarchies[False])
    got = H.gpu_hierarchy_step(wl, nsteps=3)
    dts = []
    for _ in range(3):
        r = oracle.hierarchy_step(wl)
        dts.append(r["dt0"])
        for l, lv in enumerate(wl.levels):
            lv.U = r["U"][l]
    assert np.allclose(got["dts"], dts, rtol=1e-12, atol=0)
    for l in range(3):
        assert H.rel_err(got["U"][l], wl.levels[l].U).max() <= 1e-11


def test_link_order_is_enforced(H, hierarchies):
    import paper_1412_0934_b200 as amr
    wl = hierarchies[False]
    b = [amr.PatchBatch.from_level(lv, amr.AMR_F64) for lv in wl.levels]
    l12 = amr.LevelLink(b[1], b[2])
    with pytest.raises(amr.AmrError):
        amr.LevelLink(b[0], b[1])          # root upwards only
    l12.close()
    l01 = amr.LevelLink(b[0], b[1])
    l12 = amr.LevelLink(b[1], b[2])
    with pytest.raises(amr.AmrError):
        amr.LevelLink(b[1], b[2])          # one child level per batch
    with pytest.raises(amr.AmrError):
        l01.close()                        # the finer link records into l01's blocks
    l12.close()
    l01.close()


def test_four_level_step_fp64(oracle, H):
    """L = 4: two middle levels (each the fine side of one link and the coarse side of the next), 15 level steps
    per root step."""
    wl = wk.config_hierarchy(True, 4, 256, n=16, thresholds=(1.8, 2.8, 4.0))
    assert all(lv.npatch >= 4 for lv in wl.levels), wl.note
    ref = oracle.hierarchy_step(wl)
    got = H.gpu_hierarchy_step(wl)
    assert abs(got["dt0"] - ref["dt0"]) <= 1e-13 * ref["dt0"]
    ps = ref["smax"] * max(np.abs(ref["U"][0][5:8]).max(), 1e-300)
    for l in range(4):
        e = H.rel_err(got["U"][l], ref["U"][l], psi_scale=ps)
        assert e.max() <= 8 * TOL64_STEP, (l, e)
    g = wl.levels[0].g
    tot = oracle.hierarchy_totals([oracle.ghosted(u, g) for u in got["U"]], wl.levels)
    assert (np.abs(tot - ref["totals_before"])[:8] / _absn(wl.levels[0])[:8]).max() <= 1e-13


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
def test_three_level_step_patch_size_8(oracle, H, np_dtype):
    """8^3 patches run the first kernel (godunov_step.cuh, 8x8 tiles): its flux capture in all three link roles."""
    import copy
    f32 = np_dtype == np.float32
    wl = copy.deepcopy(wk.config_hierarchy(True, 3, 128, n=8, thresholds=(2.5, 3.5)))
    if f32:
        for lv in wl.levels:
            lv.U = lv.U.astype(np.float32).astype(np.float64)
    ref = oracle.hierarchy_step(wl, eps=oracle.default_eps(np_dtype))
    got = H.gpu_hierarchy_step(wl, np_dtype=np_dtype)
    ps = ref["smax"] * max(np.abs(ref["U"][0][5:8]).max(), 1e-300)
    for l in range(3):
        for grp in H.field_groups(9):
            den = np.abs(ref["U"][l][grp]).max()
            if grp == [8]:
                den = max(den, ps)
            e = np.abs(got["U"][l][grp].astype(np.float64) - ref["U"][l][grp]).max(axis=0) / den
            if f32:
                assert np.quantile(e, 0.9999) <= 4 * TOL32 and int((e > 8 * TOL32).sum()) <= 8, (l, grp, e.max())
            else:
                assert e.max() <= 4 * TOL64_STEP, (l, grp, e.max())
    g = wl.levels[0].g
    tot = oracle.hierarchy_totals([oracle.ghosted(u.astype(np.float64), g) for u in got["U"]], wl.levels)
    assert (np.abs(tot - ref["totals_before"])[:8] / _absn(wl.levels[0])[:8]).max() <= (4e-6 if f32 else 1e-13)


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
def test_overlapped_levels_give_the_bits_of_the_serial_schedule(H, hierarchies, np_dtype, monkeypatch):
    """amr_hierarchy_step runs the levels on their own streams (a level's first substep beside its parent's step).
    With AMR_HIERARCHY_OVERLAP=0 everything goes to the caller's stream in program order; three root steps must
    give bitwise the same state either way (any missing cross-level dependency shows up as a difference)."""
    wl = hierarchies[True]
    monkeypatch.setenv("AMR_HIERARCHY_OVERLAP", "0")
    serial = H.gpu_hierarchy_step(wl, np_dtype=np_dtype, nsteps=3)
    for rep in range(3):
        monkeypatch.setenv("AMR_HIERARCHY_OVERLAP", "1")
        over = H.gpu_hierarchy_step(wl, np_dtype=np_dtype, nsteps=3)
        assert serial["dts"] == over["dts"]
        for l in range(3):
            assert np.array_equal(serial["U"][l], over["U"][l]), (rep, l)

"""-m gpu parity of the PPM hydro sweeps (reading R-PPM) against the PPM oracle,
element by element on the same seeded inputs: configs 1 and 2 (the hydro configs of BASELINE.json) in fp64 at 1e-12
per step and fp32 at 1e-5, every solver and direction, outflow across sibling patches, other patch sizes, the
prolongation halo as a source, and the API's argument checks."""
import numpy as np
import pytest

import workloads as wk

pytestmark = pytest.mark.gpu

TOL64_STEP, TOL64_MULTI, TOL32 = 1e-12, 1e-10, 1e-5
RS_HLL, RS_HLLC = 0, 1


@pytest.fixture(scope="module")
def H():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    import gpu_harness
    return gpu_harness


def test_config1_sod_ppm_20_steps_fp64(oracle, H):
    """Config 1 with PPM: 32^3 patch, outflow, HLLC, cfl 0.4, 20 steps (60 sweeps, alternating order)."""
    wl = wk.config1_sod()
    lev = wl.levels[0]
    ref = oracle.ppm_advance(lev, wl, 20)
    got = H.gpu_ppm_advance(lev, wl, 20)
    assert np.allclose(got["dts"], ref["dts"], rtol=1e-12, atol=0)
    err = H.rel_err(got["U"], ref["U"])
    assert err.max() <= TOL64_MULTI, err
    one = H.rel_err(H.gpu_ppm_advance(lev, wl, 1)["U"], oracle.ppm_advance(lev, wl, 1)["U"])
    assert one.max() <= TOL64_STEP, one
    # j/k invariance of the GPU result, bitwise
    assert np.array_equal(got["U"][0, 0], np.broadcast_to(got["U"][0, 0, 5, 7, :], got["U"][0, 0].shape))


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
def test_config2_random_patches_ppm(oracle, H, np_dtype):
    """Config 2 with PPM: 512 self-periodic 16^3 patches, one step at the CFL-reduced dt; conservation."""
    wl = wk.config2_random_patches(npatch=512)
    lev = wl.levels[0]
    f32 = np.dtype(np_dtype) == np.float32
    if f32:
        lev.U = lev.U.astype(np.float32).astype(np.float64)
    ref = oracle.ppm_advance(lev, wl, 1)
    got = H.gpu_ppm_advance(lev, wl, 1, np_dtype=np_dtype)
    err = H.rel_err(got["U"], ref["U"])
    assert err.max() <= (TOL32 if f32 else TOL64_STEP), err
    tot = got["batch"].conserved_totals()
    tot0 = lev.U.sum(axis=(1, 2, 3, 4))
    absn = np.abs(lev.U).sum(axis=(1, 2, 3, 4))
    assert (np.abs(tot - tot0) / absn).max() <= (2e-6 if f32 else 1e-13)
    gc = got["counters"]
    rc = {k: sum(c[k] for c in ref["counters"]) for k in gc}
    assert gc["nonpositive_rho_after"] == rc["nonpositive_rho_after"] == 0
    if not f32:
        assert gc == rc, (gc, rc)


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
@pytest.mark.parametrize("rs", [RS_HLL, RS_HLLC])
@pytest.mark.parametrize("d", [0, 1, 2])
def test_every_direction_and_solver_single_sweep(oracle, H, np_dtype, rs, d):
    """One sweep along each direction with each solver on a periodic 2x2x2 tiling of smooth-plus-noise data
    (halo cells come from sibling patches through the neighbour table)."""
    import paper_1412_0934_b200 as amr
    rng = np.random.default_rng([wk.SEED, 400 + d])
    N, n = 32, 16
    c = (np.arange(N) + 0.5) / N
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    rho = 1.0 + 0.3 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) + 0.05 * rng.standard_normal((N, N, N))
    v = [0.6 * np.sin(2 * np.pi * (Y + Z)) + 0.05 * rng.standard_normal((N, N, N)) for _ in range(3)]
    p = 1.0 + 0.2 * np.cos(2 * np.pi * Z) + 0.02 * rng.standard_normal((N, N, N))
    G = wk.primitive_to_conserved(rho, v, p, 1.4)
    wl = wk.uniform_grid_workload("ppm_sweep", G, n, 1.4, False, 2, rs, 0.3, 1)
    lev = wl.levels[0]
    f32 = np.dtype(np_dtype) == np.float32
    if f32:
        lev.U = lev.U.astype(np.float32).astype(np.float64)
    g = lev.g
    Ug = oracle.ghosted(lev.U, g)
    oracle.fill_ghosts(Ug, g, lev.origin, lev.domain_cells, lev.bc, False)
    dt = 0.3 * lev.dx / oracle.smax(Ug, g, wl.gamma)
    ref = oracle.interior(oracle.ppm_sweep(Ug, g, d, dt, lev.dx, wl.gamma, rs)["U"], g)
    b = amr.PatchBatch.from_level(lev, H.gpu_dtype(np_dtype))
    b.hydro_sweep_ppm(dt, wl.gamma, rs, d)
    err = H.rel_err(b.download(), ref)
    assert err.max() <= (TOL32 if f32 else TOL64_STEP), err
    assert np.abs(ref - lev.U).max() > 1e-3


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
def test_outflow_across_sibling_patches_and_other_patch_sizes(oracle, H, np_dtype):
    """Outflow faces on a 2x2x2 tiling (the clamp lands in the patch itself along the sweep), n = 8 and n = 32,
    three steps with alternating sweep order."""
    f32 = np.dtype(np_dtype) == np.float32
    for n in (8, 32):
        N = 2 * n
        rng = np.random.default_rng([wk.SEED, 410 + n])
        c = (np.arange(N) + 0.5) / N
        Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
        rho = 1.0 + 0.5 * np.exp(-40 * ((X - 0.4) ** 2 + (Y - 0.5) ** 2 + (Z - 0.6) ** 2))
        p = 1.0 + 2.0 * np.exp(-40 * ((X - 0.4) ** 2 + (Y - 0.5) ** 2 + (Z - 0.6) ** 2))
        v = [0.2 + 0 * X, -0.1 + 0 * X, 0.05 + 0 * X]
        G = wk.primitive_to_conserved(rho, v, p, 1.4)
        wl = wk.uniform_grid_workload("ppm_outflow", G, n, 1.4, False, 2, RS_HLLC, 0.4, 3)
        lev = wl.levels[0]
        lev.bc = (wk.configs.BC_OUTFLOW,) * 6
        if f32:
            lev.U = lev.U.astype(np.float32).astype(np.float64)
        if f32:      # per step (A17)
            b_err = []
            import paper_1412_0934_b200 as amr
            b = amr.PatchBatch.from_level(lev, amr.AMR_F32)
            U = b.download()
            for step_no in range(3):
                dt, sm = b.cfl_dt(wl.gamma, wl.cfl)
                b.hydro_step_ppm(dt, wl.gamma, RS_HLLC, step_no % 2)
                Ug = oracle.ghosted(U.astype(np.float64), lev.g)
                for d in oracle.PPM_ORDERS[step_no % 2]:
                    oracle.fill_ghosts(Ug, lev.g, lev.origin, lev.domain_cells, lev.bc, False)
                    Ug = oracle.ppm_sweep(Ug, lev.g, d, dt, lev.dx, wl.gamma, RS_HLLC)["U"]
                U = b.download()
                b_err.append(H.rel_err(U, oracle.interior(Ug, lev.g)).max())
            assert max(b_err) <= TOL32, b_err
        else:
            ref = oracle.ppm_advance(lev, wl, 3)
            got = H.gpu_ppm_advance(lev, wl, 3)
            err = H.rel_err(got["U"], ref["U"])
            assert err.max() <= 3 * TOL64_STEP, (n, err)


def test_prolongation_halo_as_a_source(oracle, H):
    """A fine-level batch whose halo regions are not covered by siblings: the sweeps read the prolongation halo
    buffer (filled through amr_prolong_ghosts, then the link is destroyed: PPM records no flux registers)."""
    import paper_1412_0934_b200 as amr
    wl = wk.config4_two_level(False, nfine=64, threshold=3.0)
    lc, lf = wl.levels
    bc = amr.PatchBatch.from_level(lc, amr.AMR_F64)
    bf = amr.PatchBatch.from_level(lf, amr.AMR_F64)
    link = amr.LevelLink(bc, bf)
    with pytest.raises(amr.AmrError):
        bf.hydro_sweep_ppm(1e-4, wl.gamma, RS_HLLC, 0)          # linked: refused
    link.prolong_ghosts(0.0)
    link.close()
    g = lf.g
    Uc = oracle.ghosted(lc.U, g)
    oracle.fill_ghosts(Uc, g, lc.origin, lc.domain_cells, lc.bc, False)
    Uf = oracle.ghosted(lf.U, g)
    dt = 0.2 * lf.dx / max(oracle.smax(Uf, g, wl.gamma), oracle.smax(Uc, g, wl.gamma))
    for d in (0, 1, 2):
        mask = oracle.fill_ghosts(Uf, g, lf.origin, lf.domain_cells, lf.bc, False)
        oracle.prolong_ghosts(Uf, mask, lf, Uc, Uc, lc, 0.0)
        assert (mask == 2).any()
        ref = oracle.interior(oracle.ppm_sweep(Uf, g, d, dt, lf.dx, wl.gamma, RS_HLLC)["U"], g)
        b = amr.PatchBatch.from_level(lf, amr.AMR_F64)
        # same halo contents: copy the prolonged halo through a fresh link
        l2 = amr.LevelLink(bc, b)
        l2.prolong_ghosts(0.0)
        l2.close()
        b.hydro_sweep_ppm(dt, wl.gamma, RS_HLLC, d)
        err = H.rel_err(b.download(), ref)
        assert err.max() <= TOL64_STEP, (d, err)


def test_ppm_api_rejects_bad_arguments(H):
    import paper_1412_0934_b200 as amr
    b = amr.PatchBatch(1, 16, 5, amr.AMR_F64, 0.1, self_periodic=True)
    b.upload(np.ones((5, 1, 16, 16, 16)))
    for args in ((0.0, 1.4, 1, 0), (1e-3, 1.0, 1, 0), (1e-3, 1.4, 2, 0), (1e-3, 1.4, 1, 3), (1e-3, 1.4, 1, -1)):
        with pytest.raises(amr.AmrError):
            b.hydro_sweep_ppm(*args)
    with pytest.raises(amr.AmrError):
        b.hydro_step_ppm(1e-3, 1.4, 1, 2)                                      # order
    m = amr.PatchBatch(1, 16, 9, amr.AMR_F32, 0.1, self_periodic=True)
    with pytest.raises(amr.AmrError):
        m.hydro_sweep_ppm(1e-3, 1.4, 1, 0)                                     # 9 fields
    # a uniform state is preserved bitwise by a full step
    U = np.ones((5, 1, 16, 16, 16)) * np.array([1.3, 0.4, -0.7, 0.2, 3.0]).reshape(5, 1, 1, 1, 1)
    b.upload(U)
    b.hydro_step_ppm(1e-3, 1.4, 1, 0)
    assert np.array_equal(b.download(), U)

"""-m gpu parity tests proper: the CUDA path (through the C-ABI, via the Python binding) against the
CPU oracle, element by element on the same seeded inputs.  Tolerances: BASELINE.json:north_star
(fp64 <= 1e-12 per step, <= 1e-10 after 20 steps; fp32 <= 1e-5; conserved totals 1e-13), error norm
of reading A18 (tests/gpu_harness.rel_err)."""
import numpy as np
import pytest

import workloads as wk

pytestmark = pytest.mark.gpu

TOL64_STEP, TOL64_MULTI, TOL32 = 1e-12, 1e-10, 1e-5


@pytest.fixture(scope="module")
def H():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    import gpu_harness
    return gpu_harness


def _psi_scale(ref, ch):
    return ch * np.abs(ref[5:8]).max()


def test_config1_sod_20_steps_fp64(oracle, H):
    """Config 1: one 32^3 patch, outflow, minmod + HLLC, cfl 0.4, 20 steps, dt from amr_cfl_dt."""
    wl = wk.config1_sod()
    lev = wl.levels[0]
    ref1 = oracle.advance(lev, wl, 1)
    got1 = H.gpu_advance(lev, wl, 1)
    assert H.rel_err(got1["U"], ref1["U"]).max() <= TOL64_STEP
    ref = oracle.advance(lev, wl, 20)
    got = H.gpu_advance(lev, wl, 20)
    assert np.allclose(got["dts"], ref["dts"], rtol=1e-12, atol=0)
    assert H.rel_err(got["U"], ref["U"]).max() <= TOL64_MULTI
    # P3 on the GPU: j/k invariance bitwise, no transverse momentum
    U = got["U"][:, 0]
    assert np.array_equal(U, np.broadcast_to(U[:, :1, :1, :], U.shape))
    assert not U[2].any() and not U[3].any()
    # P1/P2: against the exact Riemann solution (tests/golden/sod_exact.txt is used by the oracle pin;
    # here the same L1 bound is asserted on the GPU profile through the oracle's agreement)
    assert np.abs(U[0, 0, 0] - ref["U"][0, 0, 0, 0]).max() < 1e-12


def test_config2_random_patches_fp64(oracle, H):
    """Config 2: 512 self-periodic 16^3 patches, MC + HLLC, one step at the CFL-reduced dt."""
    wl = wk.config2_random_patches()
    lev = wl.levels[0]
    ref = oracle.advance(lev, wl, 1)
    got = H.gpu_advance(lev, wl, 1)
    assert abs(got["smaxs"][0] - ref["smaxs"][0]) <= 1e-14 * ref["smaxs"][0]
    assert H.rel_err(got["U"], ref["U"]).max() <= TOL64_STEP
    # conserved totals: GPU reduction vs oracle long-double sums, and conservation itself (P5)
    b = got["batch"]
    tot = b.conserved_totals()
    tref = oracle.totals(oracle.ghosted(ref["U"], lev.g), lev.g)
    absn = np.abs(ref["U"]).sum(axis=(1, 2, 3, 4))
    assert (np.abs(tot - tref) / absn).max() <= 1e-13
    t0 = oracle.totals(oracle.ghosted(lev.U, lev.g), lev.g)
    assert (np.abs(tot - t0) / absn).max() <= 1e-13


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
def test_config3_orszag_tang_small(oracle, H, np_dtype):
    """Config 3 at 64^3 (64 patches of 16^3, Morton order): MC + HLLD + GLM, 5 steps."""
    wl = wk.config3_orszag_tang(N=64)
    lev = wl.levels[0]
    lev.U = lev.U.astype(np_dtype).astype(np.float64)     # A17: oracle starts from the rounded data
    ref = oracle.advance(lev, wl, 5)
    got = H.gpu_advance(lev, wl, 5, np_dtype=np_dtype)
    tol = TOL64_MULTI if np_dtype == np.float64 else TOL32
    err = H.rel_err(got["U"], ref["U"], psi_scale=_psi_scale(ref["U"], ref["smaxs"][-1]))
    assert err.max() <= tol, err
    if np_dtype == np.float64:
        got1 = H.gpu_advance(lev, wl, 1)
        ref1 = oracle.advance(lev, wl, 1)
        e1 = H.rel_err(got1["U"], ref1["U"], psi_scale=_psi_scale(ref1["U"], ref1["smaxs"][-1]))
        assert e1.max() <= TOL64_STEP, e1
        tot = got["batch"].conserved_totals()
        t0 = oracle.totals(oracle.ghosted(lev.U, lev.g), lev.g)
        absn = np.abs(lev.U).sum(axis=(1, 2, 3, 4))
        absn = np.array([absn[0], absn[1:4].max(), absn[1:4].max(), absn[1:4].max(), absn[4],
                         absn[5:8].max(), absn[5:8].max(), absn[5:8].max()])   # A18 grouping
        assert (np.abs(tot - t0)[:8] / absn).max() <= 1e-13


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
def test_config5_turbulence_small(oracle, H, np_dtype):
    """Config 5 recipe at 64^3 as 8 patches of 32^3 (several tiles per patch, Mach 3, beta = 100).
    fp64: whole 3-step evolution against the oracle.  fp32: the 1e-5 bound is per step (north_star
    gives the fp64 bound "per step" and the fp32 one beside it; A17): at this resolution the
    Mach-3 field is rough at grid scale and fp32 round-off (of the oracle's own fp32 build just the
    same) grows 2-3x per step, so each step is checked from the GPU's own state of that step."""
    G = wk.configs.turbulence_state(64)
    wl = wk.uniform_grid_workload("config5_small", G, 32, 5.0 / 3.0, True, wk.configs.LIM_MC, wk.configs.RS_HLLD, 0.3, 3)
    lev = wl.levels[0]
    lev.U = lev.U.astype(np_dtype).astype(np.float64)
    if np_dtype == np.float64:
        ref = oracle.advance(lev, wl, 3)
        got = H.gpu_advance(lev, wl, 3, np_dtype=np_dtype)
        err = H.rel_err(got["U"], ref["U"], psi_scale=_psi_scale(ref["U"], ref["smaxs"][-1]))
        assert err.max() <= TOL64_MULTI, err
    else:
        errs, U, _ = H.per_step_parity(oracle, lev, wl, 3, np_dtype)
        assert max(e.max() for e in errs) <= TOL32, errs
        # and the whole run stays as close to the fp64 oracle as the oracle's own fp32 build does
        ref = oracle.advance(lev, wl, 3)
        ref32 = oracle.advance(lev, wl, 3, dtype=np.float32)
        ps = _psi_scale(ref["U"], ref["smaxs"][-1])
        e_gpu, e_o32 = H.rel_err(U, ref["U"], ps), H.rel_err(ref32["U"], ref["U"], ps)
        assert e_gpu.max() <= 2.0 * e_o32.max() + 1e-6, (e_gpu, e_o32)


def _random_level(nf, n, npx, seed, outflow=False, np_dtype=np.float64):
    rng = np.random.default_rng([wk.SEED, 99, seed])
    N = n * npx
    rho = np.exp(0.4 * rng.standard_normal((N, N, N)))
    v = 0.8 * rng.standard_normal((3, N, N, N))
    p = np.exp(0.3 * rng.standard_normal((N, N, N)))
    B = 0.7 * rng.standard_normal((3, N, N, N)) if nf == 9 else None
    G = wk.primitive_to_conserved(rho, v, p, 5.0 / 3.0, B=B)
    if nf == 9:
        G[8] = 0.1 * rng.standard_normal((N, N, N))
    bc = (wk.configs.BC_OUTFLOW,) * 6 if outflow else (wk.configs.BC_PERIODIC,) * 6
    wl = wk.uniform_grid_workload("random", G, n, 5.0 / 3.0, nf == 9, wk.configs.LIM_MC,
                                  wk.configs.RS_HLLD if nf == 9 else wk.configs.RS_HLLC, 0.3, 1, bc=bc)
    wl.levels[0].U = wl.levels[0].U.astype(np_dtype).astype(np.float64)
    return wl


@pytest.mark.parametrize("nf", [5, 9])
@pytest.mark.parametrize("limiter", [0, 1, 2])
@pytest.mark.parametrize("rs_exact", [False, True])
@pytest.mark.parametrize("n", [8, 16])
def test_every_limiter_and_solver_fp64(oracle, H, nf, limiter, rs_exact, n):
    """One step of every (limiter x Riemann solver) on rough random data (white noise: shocks at every
    face, all HLLD regions, positivity fallbacks), periodic 2x2x2 patches; n=8 runs the 8x8 tile."""
    wl = _random_level(nf, n, 2, seed=nf * 10 + n)
    lev = wl.levels[0]
    rs = (wk.configs.RS_HLLD if nf == 9 else wk.configs.RS_HLLC) if rs_exact else wk.configs.RS_HLL
    ref = oracle.advance(lev, wl, 1, limiter=limiter, riemann_solver=rs)
    got = H.gpu_advance(lev, wl, 1, limiter=limiter, riemann=rs)
    err = H.rel_err(got["U"], ref["U"], psi_scale=_psi_scale(ref["U"], ref["smaxs"][0]) if nf == 9 else None)
    assert err.max() <= TOL64_STEP, err
    # event counters: cells are counted once; a face on the boundary between two tiles of one patch is
    # counted by both tiles (include/amr_godunov.h), so face counts may exceed the oracle's slightly
    gc, rc = got["counters"], ref["counters"][0]
    if n == 16:
        assert gc["positivity_fallback_cells"] == rc["positivity_fallback_cells"]
        assert gc["nonpositive_rho_after"] == rc["nonpositive_rho_after"]
        assert rc["hll_fallback_faces"] <= gc["hll_fallback_faces"] <= 1.05 * rc["hll_fallback_faces"] + 4


@pytest.mark.parametrize("nf", [5, 9])
def test_every_solver_fp32(oracle, H, nf):
    wl = _random_level(nf, 16, 2, seed=7 + nf, np_dtype=np.float32)
    lev = wl.levels[0]
    ref = oracle.advance(lev, wl, 2)
    got = H.gpu_advance(lev, wl, 2, np_dtype=np.float32)
    err = H.rel_err(got["U"], ref["U"], psi_scale=_psi_scale(ref["U"], ref["smaxs"][0]) if nf == 9 else None)
    assert err.max() <= TOL32, err


@pytest.mark.parametrize("nf", [5, 9])
@pytest.mark.parametrize("limiter", [0, 1, 2])
@pytest.mark.parametrize("rs_exact", [False, True])
@pytest.mark.parametrize("n", [16, 32])
def test_every_limiter_and_solver_fp32(oracle, H, nf, limiter, rs_exact, n):
    """The fp32 path is a kernel of its own (two cells per thread, packed f32x2 arithmetic, branch-free
    Riemann solvers; n = 16 runs its 16x16 tile, n = 32 its 32x8 tile): one step of every
    (limiter x Riemann solver) on rough random data against the fp64 oracle started from the fp32-rounded
    data (A17), and the event counters against the oracle's."""
    wl = _random_level(nf, n, 2, seed=nf * 10 + n + 1, np_dtype=np.float32)
    lev = wl.levels[0]
    rs = (wk.configs.RS_HLLD if nf == 9 else wk.configs.RS_HLLC) if rs_exact else wk.configs.RS_HLL
    eps32 = oracle.default_eps(np.float32)      # the degeneracy thresholds (A7) are the batch dtype's
    ref = oracle.advance(lev, wl, 1, limiter=limiter, riemann_solver=rs, eps=eps32)
    got = H.gpu_advance(lev, wl, 1, np_dtype=np.float32, limiter=limiter, riemann=rs)
    ps = _psi_scale(ref["U"], ref["smaxs"][0]) if nf == 9 else None
    err = H.rel_err(got["U"], ref["U"], psi_scale=ps)
    # white noise with |B| ~ p ~ rho ~ 1 puts many faces next to HLLD's degenerate states, where fp32
    # round-off of ANY evaluation order is amplified: the bound is 1e-5, or twice what the oracle's own
    # fp32 build does on the same data if that is larger (A17)
    ref32 = oracle.advance(lev, wl, 1, dtype=np.float32, limiter=limiter, riemann_solver=rs)
    e_o32 = H.rel_err(ref32["U"], ref["U"], psi_scale=ps)
    assert err.max() <= max(TOL32, 2.0 * e_o32.max()), (err, e_o32)
    # decisions are taken in fp32 on the GPU and in fp64 by the oracle: a cell or face within round-off of
    # a threshold may flip, so the counts agree closely rather than exactly; faces on tile boundaries are
    # counted by both tiles (include/amr_godunov.h)
    gc, rc = got["counters"], ref["counters"][0]
    assert abs(gc["positivity_fallback_cells"] - rc["positivity_fallback_cells"]) <= 2 + 0.02 * rc["positivity_fallback_cells"]
    assert gc["nonpositive_rho_after"] == rc["nonpositive_rho_after"]
    assert 0.95 * rc["hll_fallback_faces"] - 4 <= gc["hll_fallback_faces"] <= 1.10 * rc["hll_fallback_faces"] + 4


def _config_shaped(kind, nf, n):
    """64^3 config-shaped data on n^3 patches: config 3 (Orszag-Tang) or the config-5 recipe (Mach-3 turbulence,
    beta = 100); nf = 5 takes the same gas without the field (E loses B^2/2)."""
    wl = wk.config3_orszag_tang(N=64, n=n) if kind == "config3" else wk.config5_turbulence(N=64, n=n)
    lev = wl.levels[0]
    U = lev.U.copy()
    if nf == 5:
        U[4] -= 0.5 * (U[5] ** 2 + U[6] ** 2 + U[7] ** 2)
        U = np.ascontiguousarray(U[:5])
        wl = wk.Workload(wl.name + "_hydro", [lev], wl.gamma, False, wl.limiter, wk.configs.RS_HLLC, wl.cfl, 1, 0.0)
    lev.U = U.astype(np.float32).astype(np.float64)
    return wl


@pytest.mark.parametrize("kind", ["config3", "config5"])
@pytest.mark.parametrize("nf", [5, 9])
@pytest.mark.parametrize("limiter", [0, 1, 2])
@pytest.mark.parametrize("rs_exact", [False, True])
@pytest.mark.parametrize("n", [16, 32])
def test_every_limiter_and_solver_fp32_at_the_plain_bound(oracle, H, kind, nf, limiter, rs_exact, n):
    """north_star's fp32 bound, plain: one step of EVERY (limiter x Riemann solver x hydro/MHD) on config-shaped
    data (config 3's Orszag-Tang vortex and config 5's turbulence at 64^3, n = 16 and n = 32 patches) within
    1e-5 of the fp64 oracle started from the fp32-rounded data (A17) -- no allowance for the oracle's own fp32
    error and no quantile; the only cells excused are those the ORACLE shows to touch a face within round-off
    of a discontinuous decision (see below).  (The white-noise cases above stay as stress tests with their
    documented bound.)  Event counters as the oracle's."""
    wl = _config_shaped(kind, nf, n)
    lev = wl.levels[0]
    rs = (wk.configs.RS_HLLD if nf == 9 else wk.configs.RS_HLLC) if rs_exact else wk.configs.RS_HLL
    ref = oracle.advance(lev, wl, 1, limiter=limiter, riemann_solver=rs, eps=oracle.default_eps(np.float32))
    got = H.gpu_advance(lev, wl, 1, np_dtype=np.float32, limiter=limiter, riemann=rs)
    ps = _psi_scale(ref["U"], ref["smaxs"][0]) if nf == 9 else None
    # per cell: the largest error over the field groups, each normalised as in rel_err (A18)
    e_cell = np.zeros(got["U"].shape[1:])
    for grp in H.field_groups(nf):
        den = np.abs(ref["U"][grp]).max()
        if grp == [8]:
            den = max(den, ps)
        e_cell = np.maximum(e_cell, np.abs(got["U"][grp].astype(np.float64) - ref["U"][grp]).max(axis=0) / den)
    bad = np.argwhere(e_cell > TOL32)
    # The one allowance (A7 / A19, measured: config 5 at 64^3 with minmod + HLLD has ONE face with p_T* = -9e-8 p_T,
    # which the oracle sends to the HLL fallback and fp32 arithmetic does not): a cell may miss the bound only if
    # the oracle itself says one of its faces sits within fp32 round-off of a discontinuous decision; at most 4.
    assert len(bad) <= 4, (len(bad), e_cell.max())
    if len(bad):
        assert nf == 9 and rs == wk.configs.RS_HLLD, (bad, e_cell.max())
        ok = H.cells_next_to_a_marginal_decision(oracle, lev, wl, ref["dts"][0], ref["smaxs"][0], limiter, rs,
                                                 oracle.default_eps(np.float32), bad)
        assert all(ok), (bad, ok, e_cell[tuple(bad.T)])
    assert abs(got["dts"][0] - ref["dts"][0]) <= 4e-6 * ref["dts"][0]
    gc, rc = got["counters"], ref["counters"][0]
    assert gc["nonpositive_rho_after"] == rc["nonpositive_rho_after"] == 0
    assert abs(gc["positivity_fallback_cells"] - rc["positivity_fallback_cells"]) <= 2 + 0.02 * rc["positivity_fallback_cells"]


@pytest.mark.parametrize("n,npx", [(24, 2), (48, 1), (64, 1)])
@pytest.mark.parametrize("nf", [5, 9])
def test_other_patch_sizes_fp32(oracle, H, n, npx, nf):
    """Patch sizes beside 16 and 32: n = 48 runs three 16x16 tiles per direction, n = 64 two 32-wide tiles (the
    x halo of a tile then lies inside the same patch), n = 24 falls back to the scalar 8x8 tile; a single
    periodic patch is its own neighbour in all 26 directions."""
    wl = _random_level(nf, n, npx, seed=nf + n, np_dtype=np.float32)
    lev = wl.levels[0]
    ref = oracle.advance(lev, wl, 1, eps=oracle.default_eps(np.float32))
    got = H.gpu_advance(lev, wl, 1, np_dtype=np.float32)
    # White noise puts ~5 % of the faces into the HLL fallback (p* <= 0, A7).  That decision is discontinuous and
    # is taken in the batch dtype, so a face within fp32 round-off of the threshold may decide differently from
    # the fp64 oracle; such a face changes its two cells by O(1e-4).  Everything else must meet the bound.
    nbad = 0
    for grp in H.field_groups(nf):
        den = np.abs(ref["U"][grp]).max()
        if grp == [8]:
            den = max(den, ref["smaxs"][0] * np.abs(ref["U"][5:8]).max())
        e = np.abs(got["U"][grp].astype(np.float64) - ref["U"][grp]).max(axis=0) / den
        nbad = max(nbad, int((e > 2 * TOL32).sum()))
        assert np.quantile(e, 0.9999) <= TOL32, (grp, np.quantile(e, 0.9999))
    assert nbad <= 8, nbad
    gc, rc = got["counters"], ref["counters"][0]
    # faces on the boundary between two tiles of a patch are counted by both tiles (include/amr_godunov.h)
    assert 0.95 * rc["hll_fallback_faces"] - 4 <= gc["hll_fallback_faces"] <= 1.25 * rc["hll_fallback_faces"] + 4


@pytest.mark.parametrize("nf", [5, 9])
@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
def test_outflow_multi_patch(oracle, H, nf, np_dtype):
    """O0 (ii): outflow clamp on a 2x2x2-patch domain (edge and corner regions clamp into siblings)."""
    wl = _random_level(nf, 16, 2, seed=3, outflow=True, np_dtype=np_dtype)
    lev = wl.levels[0]
    if np_dtype == np.float64:
        ref = oracle.advance(lev, wl, 2)
        got = H.gpu_advance(lev, wl, 2)
        err = H.rel_err(got["U"], ref["U"], psi_scale=_psi_scale(ref["U"], ref["smaxs"][0]) if nf == 9 else None)
        assert err.max() <= TOL64_MULTI, err
    else:
        errs, _, _ = H.per_step_parity(oracle, lev, wl, 2, np_dtype)
        assert max(e.max() for e in errs) <= TOL32, errs


@pytest.mark.parametrize("outflow", [False, True])
def test_ghost_cells_seen_through_the_api(oracle, H, outflow):
    """amr_patch_batch_download(with_ghosts=1) == oracle O0 fill, all three layers, bit for bit."""
    import paper_1412_0934_b200 as amr
    wl = _random_level(9, 16, 2, seed=11, outflow=outflow)
    lev = wl.levels[0]
    b = amr.PatchBatch.from_level(lev, amr.AMR_F64)
    b.fill_ghosts()
    got = b.download(with_ghosts=True)
    ref = oracle.ghosted(lev.U, lev.g)
    oracle.fill_ghosts(ref, lev.g, lev.origin, lev.domain_cells, lev.bc, lev.self_periodic)
    assert np.array_equal(got, ref)
    # upload with ghosts ignores the ghost layer
    junk = ref.copy()
    junk[:, :, :3] = -7.0
    b.upload(junk, with_ghosts=True)
    assert np.array_equal(b.download(), lev.U)


def test_cfl_fused_equals_standalone(oracle, H):
    """P15 on the GPU: the smax fused into the step epilogue is bitwise the standalone reduction's."""
    import paper_1412_0934_b200 as amr
    for nf, npd in ((5, np.float64), (9, np.float64), (5, np.float32), (9, np.float32)):
        wl = _random_level(nf, 16, 2, seed=21 + nf, np_dtype=npd)
        lev = wl.levels[0]
        r = H.gpu_advance(lev, wl, 1, np_dtype=npd)
        b = r["batch"]
        _, fused = b.cfl_dt(wl.gamma, wl.cfl)
        b2 = amr.PatchBatch(lev.npatch, lev.n, nf, H.gpu_dtype(npd), lev.dx, origin=lev.origin,
                            domain_cells=lev.domain_cells, bc=lev.bc)
        b2.upload(r["U"])
        _, alone = b2.cfl_dt(wl.gamma, wl.cfl)
        assert fused == alone
        ref = oracle.smax(oracle.ghosted(r["U"].astype(np.float64), lev.g), lev.g, wl.gamma)
        assert abs(alone - ref) <= (1e-14 if npd == np.float64 else 1e-6) * ref


def test_uniform_state_is_preserved_bitwise(H):
    """P4 on the GPU: flux differences cancel exactly; psi only decays by exp(-alpha ch dt/dx)."""
    import paper_1412_0934_b200 as amr
    n, npx = 16, 2
    G = np.empty((9, 32, 32, 32))
    prim = wk.primitive_to_conserved(np.full((32, 32, 32), 1.3), (np.full((32, 32, 32), 0.4),) * 3,
                                     np.full((32, 32, 32), 0.7), 5.0 / 3.0,
                                     B=(np.full((32, 32, 32), 0.3), np.full((32, 32, 32), -0.2), np.full((32, 32, 32), 0.5)))
    G[:] = prim
    G[8] = 0.25
    wl = wk.uniform_grid_workload("uniform", G, n, 5.0 / 3.0, True, 2, 2, 0.3, 1)
    lev = wl.levels[0]
    b = amr.PatchBatch.from_level(lev, amr.AMR_F64)
    dt, sm = b.cfl_dt(wl.gamma, wl.cfl)
    b.mhd_step(dt, wl.gamma, 2, 2, sm, 0.4)
    U = b.download()
    assert np.array_equal(U[:8], lev.U[:8])
    assert np.allclose(U[8], 0.25 * np.exp(-0.4 * sm * dt / lev.dx), rtol=1e-15)


@pytest.mark.parametrize("mhd", [False, True])
def test_two_level_step_fp64(oracle, H, mhd):
    """Config 4 at 64^3 fine index space: O9 (coarse step, two fine substeps with prolonged halos,
    restriction, reflux) against the oracle, and composite conservation (P13) on the GPU result."""
    wl = wk.config4_two_level(mhd, nfine=64, threshold=3.0)
    lc, lf = wl.levels
    ref = oracle.two_level_step(wl)
    got = H.gpu_two_level_step(wl)
    assert abs(got["dt0"] - ref["dt0"]) <= 1e-13 * ref["dt0"]
    ps = ref["smax"] * max(np.abs(ref["Uc"][5:8]).max(), 1e-300) if mhd else None
    ec = H.rel_err(got["Uc"], ref["Uc"], psi_scale=ps)
    ef = H.rel_err(got["Uf"], ref["Uf"], psi_scale=ps)
    assert ec.max() <= 2 * TOL64_STEP and ef.max() <= 2 * TOL64_STEP, (ec, ef)
    tot = oracle.composite_totals(oracle.ghosted(got["Uc"], lc.g), lc, oracle.ghosted(got["Uf"], lf.g), lf)
    nfc = 8 if mhd else 5
    absn = np.array([np.abs(lc.U[f]).sum() * lc.dx ** 3 for f in range(lc.nfields)])
    assert (np.abs(tot - ref["totals_before"])[:nfc] / absn[:nfc]).max() <= 1e-13


@pytest.mark.parametrize("mhd", [False, True])
def test_two_level_step_fp32(oracle, H, mhd):
    """Config 4 (fp32, as BASELINE.json states it) at 64^3 fine index space: the fp32 kernel's prolongation
    halo source (4-byte copies from the odd-aligned halo buffer) and flux-register capture, against the
    fp64 oracle started from the fp32-rounded data; composite conservation to fp32 round-off (P13)."""
    wl = wk.config4_two_level(mhd, nfine=64, threshold=3.0)
    lc, lf = wl.levels
    lc.U = lc.U.astype(np.float32).astype(np.float64)
    lf.U = lf.U.astype(np.float32).astype(np.float64)
    ref = oracle.two_level_step(wl, eps=oracle.default_eps(np.float32))   # A7 thresholds of the batch dtype
    got = H.gpu_two_level_step(wl, np_dtype=np.float32)
    assert abs(got["dt0"] - ref["dt0"]) <= 4e-6 * ref["dt0"]
    ps = ref["smax"] * max(np.abs(ref["Uc"][5:8]).max(), 1e-300) if mhd else None
    ec = H.rel_err(got["Uc"], ref["Uc"], psi_scale=ps)
    ef = H.rel_err(got["Uf"], ref["Uf"], psi_scale=ps)
    assert ec.max() <= 2 * TOL32 and ef.max() <= 2 * TOL32, (ec, ef)
    tot = oracle.composite_totals(oracle.ghosted(got["Uc"].astype(np.float64), lc.g), lc,
                                  oracle.ghosted(got["Uf"].astype(np.float64), lf.g), lf)
    nfc = 8 if mhd else 5
    absn = np.array([np.abs(lc.U[f]).sum() * lc.dx ** 3 for f in range(lc.nfields)])
    assert (np.abs(tot - ref["totals_before"])[:nfc] / absn[:nfc]).max() <= 2e-6


@pytest.mark.parametrize("mhd", [False, True])
@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
def test_two_level_step_with_fine_patches_on_outflow_faces(oracle, H, mhd, np_dtype):
    """The boundary readings of O8 / O9: fine patches ON the outflow x faces.  Halo cells beyond
    the face are clamped copies or prolongations at the clamped cell, fine faces on the domain face are not
    refluxed.  Against the oracle, plus its own pin on the GPU result: the totals change only by the boundary
    pressure force (tests/test_oracle_amr.py)."""
    wl = wk.two_level_outflow(mhd)
    lc, lf = wl.levels
    f32 = np.dtype(np_dtype) == np.float32
    if f32:
        lc.U = lc.U.astype(np.float32).astype(np.float64)
        lf.U = lf.U.astype(np.float32).astype(np.float64)
    ref = oracle.two_level_step(wl, eps=oracle.default_eps(np_dtype))
    got = H.gpu_two_level_step(wl, np_dtype=np_dtype)
    tol = TOL32 if f32 else TOL64_STEP
    ps = ref["smax"] * np.abs(ref["Uc"][5:8]).max() if mhd else None
    ec = H.rel_err(got["Uc"], ref["Uc"], psi_scale=ps)
    ef = H.rel_err(got["Uf"], ref["Uf"], psi_scale=ps)
    assert ec.max() <= 2 * tol and ef.max() <= 2 * tol, (ec, ef)
    tot = oracle.composite_totals(oracle.ghosted(got["Uc"].astype(np.float64), lc.g), lc,
                                  oracle.ghosted(got["Uf"].astype(np.float64), lf.g), lf)
    d = tot - ref["totals_before"]
    keep = [0, 2, 3, 4] + ([5, 6, 7] if mhd else [])
    assert np.abs(d[keep]).max() <= (2e-6 if f32 else 1e-13)
    expect = got["dt0"] * (1.0 - 0.4)
    assert abs(d[1] - expect) <= (1e-4 if f32 else 1e-11) * expect


def test_prolonged_halo_seen_through_the_api(oracle, H):
    """O8 through the API: after amr_prolong_ghosts the fine ghosts equal the oracle's (theta = 0.5)."""
    import paper_1412_0934_b200 as amr
    wl = wk.config4_two_level(False, nfine=64, threshold=3.0)
    lc, lf = wl.levels
    bc = amr.PatchBatch.from_level(lc, amr.AMR_F64)
    bf = amr.PatchBatch.from_level(lf, amr.AMR_F64)
    link = amr.LevelLink(bc, bf)
    dt, sm = bc.cfl_dt(wl.gamma, wl.cfl)
    bc.hydro_step(dt, wl.gamma, wl.limiter, wl.riemann)
    link.prolong_ghosts(0.5)
    got = bf.download(with_ghosts=True)
    g = lc.g
    Uc = oracle.ghosted(lc.U, g)
    oracle.fill_ghosts(Uc, g, lc.origin, lc.domain_cells, lc.bc, False)
    Ucn = oracle.step(Uc, g, dt, lc.dx, wl.gamma, wl.limiter, wl.riemann)["U"]
    oracle.fill_ghosts(Ucn, g, lc.origin, lc.domain_cells, lc.bc, False)
    Uf = oracle.ghosted(lf.U, g)
    mask = oracle.fill_ghosts(Uf, g, lf.origin, lf.domain_cells, lf.bc, False)
    oracle.prolong_ghosts(Uf, mask, lf, Uc, Ucn, lc, 0.5)
    assert (mask == 2).any()
    assert H.rel_err(got, Uf).max() <= TOL64_STEP


def test_api_rejects_bad_arguments(H):
    import paper_1412_0934_b200 as amr
    with pytest.raises(amr.AmrError):
        amr.PatchBatch(1, 12, 5, amr.AMR_F64, 0.1, self_periodic=True)          # n not a multiple of 8
    with pytest.raises(amr.AmrError):
        amr.PatchBatch(1, 16, 7, amr.AMR_F64, 0.1, self_periodic=True)          # nfields
    with pytest.raises(amr.AmrError):
        amr.PatchBatch(2, 16, 5, amr.AMR_F64, 0.1, origin=[[0, 0, 0], [0, 0, 0]], domain_cells=(32, 16, 16))
    b = amr.PatchBatch(1, 16, 5, amr.AMR_F64, 0.1, self_periodic=True)
    b.upload(np.ones((5, 1, 16, 16, 16)))
    for args in ((0.0, 1.4, 1, 1), (1e-3, 1.0, 1, 1), (1e-3, float("nan"), 1, 1), (1e-3, 1.4, 5, 1), (1e-3, 1.4, 1, 2)):
        with pytest.raises(amr.AmrError):
            b.hydro_step(*args)
    with pytest.raises(amr.AmrError):
        b.mhd_step(1e-3, 1.4, 1, 2, 1.0, 0.4)                                   # MHD step on 5 fields
    m = amr.PatchBatch(1, 16, 9, amr.AMR_F32, 0.1, self_periodic=True)
    with pytest.raises(amr.AmrError):
        m.mhd_step(1e-3, 1.4, 1, 1, 1.0, 0.4)                                   # HLLC in the MHD step
    with pytest.raises(amr.AmrError):
        m.mhd_step(1e-3, 1.4, 1, 2, 0.0, 0.4)                                   # ch <= 0


def _degenerate_level(case, n, np_dtype):
    """32^3 periodic grid of 2^3 patches (or one self-neighbouring patch): white-noise gas (|v| ~ c_s) with the field
    configurations at which HLLD's formulas degenerate (A7)."""
    rng = np.random.default_rng([wk.SEED, 98, ["zero", "along_z", "strong", "tiny", "static", "one_patch"].index(case)])
    N = n if case == "one_patch" else 32
    rho = np.exp(0.4 * rng.standard_normal((N, N, N)))
    v = 0.8 * rng.standard_normal((3, N, N, N))
    p = np.exp(0.3 * rng.standard_normal((N, N, N)))
    B = np.zeros((3, N, N, N))
    if case == "along_z":          # B_n = 0 on every x and y face, B_t = 0 on every z face
        B[2] = 0.5
    elif case == "strong":         # beta ~ 0.01
        B[:] = 10.0 * rng.standard_normal((3, N, N, N))
    elif case == "tiny":           # B_n^2 far below eps p_T*: the rotational waves are skipped everywhere (A7)
        B[:] = 1e-9 * rng.standard_normal((3, N, N, N))
    elif case == "static":         # gas at rest in a uniform oblique field: an exact equilibrium
        rho[:], p[:], v[:] = 1.0, 0.7, 0.0
        B[0], B[1], B[2] = 0.3, -0.4, 0.5
    elif case == "one_patch":
        B[:] = 0.7 * rng.standard_normal((3, N, N, N))
    G = wk.primitive_to_conserved(rho, v, p, 5.0 / 3.0, B=B)
    wl = wk.uniform_grid_workload("degenerate_" + case, G, n, 5.0 / 3.0, True, wk.configs.LIM_MC, wk.configs.RS_HLLD, 0.3, 1)
    wl.levels[0].U = wl.levels[0].U.astype(np_dtype).astype(np.float64)
    return wl


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
@pytest.mark.parametrize("n", [16, 32])
@pytest.mark.parametrize("case", ["zero", "along_z", "strong", "tiny", "static", "one_patch"])
def test_degenerate_mhd_states(oracle, H, case, n, np_dtype):
    """HLLD where its formulas degenerate: B = 0 (the solver must reduce to HLLC: same bits for rho, m, E as the
    oracle's path through the same branch), B_n = 0 with B_t != 0 and the reverse, beta ~ 0.01, |B| ~ 1e-9, an exact
    static equilibrium (preserved bitwise), and a single patch that is its own neighbour in all 26 directions.
    One step against the oracle at the stated bounds; event counters as the oracle's (cells equal in fp64)."""
    wl = _degenerate_level(case, n, np_dtype)
    lev = wl.levels[0]
    f32 = np.dtype(np_dtype) == np.float32
    eps = oracle.default_eps(np_dtype)
    ref = oracle.advance(lev, wl, 1, eps=eps)
    got = H.gpu_advance(lev, wl, 1, np_dtype=np_dtype)
    assert np.isfinite(got["U"]).all()
    rel = abs(got["smaxs"][0] - ref["smaxs"][0]) / ref["smaxs"][0]
    assert rel <= (1e-6 if f32 else 1e-14), rel
    if case == "static":
        assert np.array_equal(got["U"], lev.U.astype(np_dtype))
        return
    ps = _psi_scale(ref["U"], ref["smaxs"][0])
    U = got["U"].astype(np.float64)
    if case in ("zero", "tiny"):
        # B (and psi) are zero or 1e-9: compare the gas, and B on its own scale
        err = H.rel_err(U[:5], ref["U"][:5])
        assert err.max() <= (TOL32 if f32 else TOL64_STEP), err
        if case == "zero":
            assert not U[5:].any() and not ref["U"][5:].any()
        else:
            db = np.abs(U[5:8] - ref["U"][5:8]).max() / np.abs(ref["U"][5:8]).max()
            assert db <= (TOL32 if f32 else TOL64_STEP), db
    else:
        err = H.rel_err(U, ref["U"], psi_scale=ps)
        assert err.max() <= (TOL32 if f32 else TOL64_STEP), err
    if not f32:
        # the GPU counts every cell once and a face on the boundary between two tiles twice (include/amr_godunov.h);
        # the oracle counts, per patch, the cells whose face states it consumes: its interior and the face neighbours
        # beyond it, so a fallback cell next to a patch boundary appears in two patches' counts
        gc, rc = got["counters"], ref["counters"][0]
        assert 0.7 * rc["positivity_fallback_cells"] - 2 <= gc["positivity_fallback_cells"] <= rc["positivity_fallback_cells"], (gc, rc)
        assert gc["nonpositive_rho_after"] == rc["nonpositive_rho_after"] == 0
        assert rc["hll_fallback_faces"] <= gc["hll_fallback_faces"] <= 1.25 * rc["hll_fallback_faces"] + 4, (gc, rc)
        assert rc["degenerate_D"] <= gc["degenerate_D"] <= 1.25 * rc["degenerate_D"] + 4, (gc, rc)


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
@pytest.mark.parametrize("nf", [5, 9])
def test_blast_wave_contrast(oracle, H, nf, np_dtype):
    """A strong explosion into a thin medium: pressure contrast 1e6 and density contrast 1e3 across a spherical
    interface that cuts through patch corners (32^3, 2^3 patches of 16^3, outflow faces), three steps from rest.
    The positivity fallback (A10) and the solver's supersonic branches carry the step; every step from the previous
    GPU state within the stated bounds, and no non-positive density afterwards."""
    N, n = 32, 16
    x = (np.arange(N) + 0.5) / N
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    r2 = (X - 0.47) ** 2 + (Y - 0.52) ** 2 + (Z - 0.5) ** 2
    inside = r2 < 0.18 ** 2
    rho = np.where(inside, 1.0, 1e-3)
    p = np.where(inside, 1e3, 1e-3)
    v = np.zeros((3, N, N, N))
    B = None
    if nf == 9:
        B = np.zeros((3, N, N, N))
        B[0], B[1] = 0.5, 0.5
    G = wk.primitive_to_conserved(rho, v, p, 5.0 / 3.0, B=B)
    wl = wk.uniform_grid_workload("blast", G, n, 5.0 / 3.0, nf == 9, wk.configs.LIM_MINMOD,
                                  wk.configs.RS_HLLD if nf == 9 else wk.configs.RS_HLLC, 0.3, 3,
                                  bc=(wk.configs.BC_OUTFLOW,) * 6)
    lev = wl.levels[0]
    lev.U = lev.U.astype(np_dtype).astype(np.float64)
    f32 = np.dtype(np_dtype) == np.float32
    errs, U, batch = H.per_step_parity(oracle, lev, wl, 3, np_dtype)
    assert max(e.max() for e in errs) <= (TOL32 if f32 else TOL64_STEP), errs
    assert (U[0] > 0).all() and np.isfinite(U).all()
    assert batch.step_counters()["nonpositive_rho_after"] == 0

"""Pins P13, P14: the oracle's two-level operators (O8 prolongation, O9
restriction / reflux / step order) against conservation and exactness properties."""
import numpy as np
import pytest

import workloads as wk


@pytest.fixture(scope="module")
def small_two_level():
    # 64^3 fine index space: root 32^3 = 8 patches, 16 of 64 aligned 8^3 blocks refined
    return {mhd: wk.config4_two_level(mhd, nfine=64, threshold=3.0) for mhd in (False, True)}


@pytest.mark.parametrize("mhd", [False, True])
def test_composite_conservation(oracle, small_two_level, mhd):
    """P13: composite totals of rho, m, E, B unchanged over one coarse step with two fine substeps
    to 1e-13 of sum|U|; without the reflux the same run leaks at the 1e-5..1e-4 level, so the
    pin does see the flux correction."""
    wl = small_two_level[mhd]
    lc, lf = wl.levels
    assert 4 <= lf.npatch <= 40
    r = oracle.two_level_step(wl)
    nf = lc.nfields
    absn = np.array([np.abs(lc.U[f]).sum() * lc.dx ** 3 for f in range(nf)])
    rel = np.abs(r["totals_after"] - r["totals_before"])[:8 if mhd else 5] / absn[:8 if mhd else 5]
    assert rel.max() < 1e-13, rel
    r2 = oracle.two_level_step(wl, do_reflux=False)
    rel2 = np.abs(r2["totals_after"] - r2["totals_before"])[:5] / absn[:5]
    assert rel2.max() > 1e-6
    # the fine level really advanced by two half steps and the root by one
    assert np.abs(r["Uf"] - lf.U).max() > 1e-3 and np.abs(r["Uc"] - lc.U).max() > 1e-3


def test_restriction_is_the_mean_of_children(oracle, small_two_level):
    wl = small_two_level[False]
    lc, lf = wl.levels
    Uc = oracle.ghosted(np.zeros_like(lc.U), lc.g)
    Uf = oracle.ghosted(lf.U, lf.g)
    oracle.restrict(Uf, lf, Uc, lc)
    G = wk.configs.join_patches(oracle.interior(Uc, lc.g), lc.origin, (32, 32, 32))
    for p, (ox, oy, oz) in enumerate(lf.origin):
        blk = lf.U[:, p].reshape(5, 8, 2, 8, 2, 8, 2).mean(axis=(2, 4, 6))
        got = G[:, oz // 2:oz // 2 + 8, oy // 2:oy // 2 + 8, ox // 2:ox // 2 + 8]
        assert np.allclose(got, blk, rtol=1e-14, atol=1e-15)
    # the initial root data ARE the 2x2x2 means of the fine data (workload recipe)
    Gc0 = wk.configs.join_patches(lc.U, lc.origin, (32, 32, 32))
    covered = G[0] != 0
    assert np.allclose(G[:, covered], Gc0[:, covered], rtol=1e-14, atol=1e-14)


def _one_fine_patch_setup(oracle, coarse_fn):
    """A single 16^3 fine patch (origin aligned to its size, as every patch must be) in a
    2x2x2-patch periodic root; every fine ghost cell must come from prolongation."""
    n, g = 16, 3
    origin0 = wk.morton_patch_origins(2, 2, 2, n)
    c = np.arange(32) + 0.5
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    Gc = coarse_fn(X, Y, Z)
    lc = wk.Level(n=n, g=g, level=0, dx=1 / 32, origin=origin0, domain_cells=(32, 32, 32), bc=(0,) * 6,
                  self_periodic=False, U=wk.split_into_patches(Gc, n, origin0))
    lf = wk.Level(n=n, g=g, level=1, dx=1 / 64, origin=np.array([[16, 16, 16]], np.int32),
                  domain_cells=(64, 64, 64), bc=(0,) * 6, self_periodic=False, U=np.zeros((Gc.shape[0], 1, n, n, n)))
    Uc = oracle.ghosted(lc.U, g)
    oracle.fill_ghosts(Uc, g, lc.origin, lc.domain_cells, lc.bc, False)
    Uf = oracle.ghosted(lf.U, g)
    mask = oracle.fill_ghosts(Uf, g, lf.origin, lf.domain_cells, lf.bc, False)
    assert mask[0, 0, 0, 0] == 0 and mask[0, 5, 5, 5] == 1
    return lc, lf, Uc, Uf, mask, Gc


def test_prolongation_is_conservative(oracle):
    """P14: the 8 children of a coarse cell average to the parent value (checked on the coarse
    cells that lie completely inside the fine ghost shell)."""
    rng = np.random.default_rng([wk.SEED, 14])
    noise = rng.standard_normal((5, 32, 32, 32))
    lc, lf, Uc, Uf, mask, Gc = _one_fine_patch_setup(oracle, lambda X, Y, Z: noise)
    oracle.prolong_ghosts(Uf, mask, lf, Uc, Uc, lc, 0.0)
    assert (mask == 0).sum() == 0
    # fine ghost indices -2,-1 (array 1,2) form the coarse cell 7; 16,17 (array 19,20) the coarse cell 16
    for (a0, C0) in ((1, 7), (19, 16)):
        for (a1, C1) in ((1, 7), (7, 10), (19, 16)):
            kids = Uf[:, 0, a0:a0 + 2, a1:a1 + 2, 7:9]
            assert np.allclose(kids.mean(axis=(1, 2, 3)), Gc[:, C0, C1, 10], rtol=1e-14, atol=1e-15)


def test_prolongation_reproduces_linear_fields_and_time_interpolates(oracle):
    lin = lambda X, Y, Z: np.stack([1.0 + 0.01 * X - 0.02 * Y + 0.005 * Z] * 5)
    lc, lf, Uc, Uf, mask, Gc = _one_fine_patch_setup(oracle, lin)
    Uc2 = Uc * 3.0
    oracle.prolong_ghosts(Uf, mask.copy(), lf, Uc, Uc2, lc, 0.5)
    # fine cell centres in coarse-cell units: (16 + i + 0.5)/2
    i = np.arange(-3, 19)
    x = (16 + i + 0.5) / 2
    Zf, Yf, Xf = np.meshgrid(x, x, x, indexing="ij")
    exact = 2.0 * (1.0 + 0.01 * Xf - 0.02 * Yf + 0.005 * Zf)     # (1-theta)*1 + theta*3 = 2
    ghost = mask[0] == 0
    assert np.allclose(Uf[0, 0][ghost], exact[ghost], rtol=1e-14, atol=0)
    assert np.all(Uf[0, 0][~ghost] == 0)                          # interiors untouched


def test_prolongation_is_limited_at_extrema(oracle):
    """minmod: a coarse cell that is a local extremum is injected without slope."""
    def bump(X, Y, Z):
        f = np.ones((5, 32, 32, 32))
        f[:, 7, 7, 10] = 5.0
        return f
    lc, lf, Uc, Uf, mask, Gc = _one_fine_patch_setup(oracle, bump)
    oracle.prolong_ghosts(Uf, mask, lf, Uc, Uc, lc, 0.0)
    assert np.all(Uf[:, 0, 1:3, 1:3, 7:9] == 5.0)
    assert np.all(Uf[:, 0, 1:3, 1:3, 9:11] == 1.0)


# ---- boundary readings of O8 / O9: fine patches ON non-periodic domain faces (A12/A14) ----

@pytest.mark.parametrize("mhd", [False, True])
def test_two_level_outflow_totals_change_only_by_the_boundary_fluxes(oracle, mhd):
    """Fine patches touch both OUTFLOW x faces; the gas at the faces is uniform and at rest for the whole
    step, so the only boundary flux is the pressure force: d(sum m_x dV) = dt0 (p_left - p_right) A with
    A = 1, and rho, m_y, m_z, E (and B) are conserved to round-off.  A reflux that wrapped through the
    outflow face would add dt0/dx0 (F_coarse(far face) - F_fine(near face)) = O(p_right - p_left) to the
    cells on the far side and fail both checks."""
    wl = wk.two_level_outflow(mhd)
    lc, lf = wl.levels
    r = oracle.two_level_step(wl)
    nf = lc.nfields
    absn = np.array([max(np.abs(lc.U[f]).sum() * lc.dx ** 3, 1.0) for f in range(nf)])
    d = (r["totals_after"] - r["totals_before"]) / absn
    keep = [0, 2, 3, 4] + ([5, 6, 7] if mhd else [])
    assert np.abs(d[keep]).max() < 1e-13, d
    expect = r["dt0"] * (1.0 - 0.4)
    got = r["totals_after"][1] - r["totals_before"][1]
    assert abs(got - expect) < 1e-12 * expect, (got, expect)
    # the step did something on both levels (the jump sits inside the second fine patch)
    assert np.abs(r["Uf"][:, 1] - lf.U[:, 1]).max() > 1e-3 and np.abs(r["Uc"] - lc.U).max() > 1e-3
    # ... and nothing at all next to the faces, bitwise (uniform state at rest, zero-gradient ghosts)
    assert np.array_equal(r["Uf"][:, 0, :, :, :4], lf.U[:, 0, :, :, :4])
    assert np.array_equal(r["Uf"][:, 2, :, :, -4:], lf.U[:, 2, :, :, -4:])


def test_two_level_outflow_uniform_state_is_a_fixed_point(oracle):
    wl = wk.two_level_outflow(True)
    for lv in wl.levels:
        lv.U[...] = lv.U[:, :1, :1, :1, :1]          # the lower-left cell's state everywhere
        lv.U[1:4] = 0.3 * lv.U[0]                    # ... moving (outflow faces see a uniform flow)
        lv.U[4] += 0.5 * 3 * 0.09 * lv.U[0]
    r = oracle.two_level_step(wl)
    assert np.array_equal(r["Uf"][:8], wl.levels[1].U[:8])
    # the covered root cells went through the 8-cell mean (a sum of eight equal numbers rounds): 1 ulp
    assert np.abs(r["Uc"][:8] - wl.levels[0].U[:8]).max() <= 4e-16


def test_prolongation_beyond_an_outflow_face_takes_the_clamped_cell(oracle):
    """O0 rule (ii) + O8: a fine ghost cell beyond an OUTFLOW face takes the value of the clamped in-domain
    fine cell; where no fine patch covers that cell it is the prolongation AT that cell (parent and child
    parity of the clamped index), never data from the far side of the domain."""
    wl = wk.two_level_outflow(False)
    lc, lf = wl.levels
    g, n = lf.g, lf.n
    rng = np.random.default_rng([wk.SEED, 141])
    lc.U[...] = rng.standard_normal(lc.U.shape)
    Uc = oracle.ghosted(lc.U, g)
    oracle.fill_ghosts(Uc, g, lc.origin, lc.domain_cells, lc.bc, False)
    Uf = oracle.ghosted(np.zeros_like(lf.U), g)
    mask = oracle.fill_ghosts(Uf, g, lf.origin, lf.domain_cells, lf.bc, False)
    # patch 0 = (0,16,16): beyond the face, inside the patch's y-z footprint, O0 clamps onto the patch itself;
    # the edge / corner regions beyond the face are left for O8
    assert mask[0, g + 4, g + 4, 0] == 1 and mask[0, g + 4, 0, 0] == 0 and mask[0, 0, 0, 0] == 0
    oracle.prolong_ghosts(Uf, mask, lf, Uc, Uc, lc, 0.0)
    assert (mask == 0).sum() == 0
    for ii in range(g):                                # array x index ii <-> i = ii - g < 0; clamped: array index g
        assert np.array_equal(Uf[:, 0, :, :g, ii], Uf[:, 0, :, :g, g])
        assert np.array_equal(Uf[:, 0, :g, :, ii], Uf[:, 0, :g, :, g])
        assert np.array_equal(Uf[:, 0, n + g:, n + g:, ii], Uf[:, 0, n + g:, n + g:, g])
    # same at the upper face for patch 2 = (48,32,32)
    for ii in range(n + g, n + 2 * g):
        assert np.array_equal(Uf[:, 2, :, :g, ii], Uf[:, 2, :, :g, n + g - 1])
    # the clamped cells themselves are ordinary prolongations: children average to the parent
    kids = Uf[:, 0, g + 2:g + 4, 1:3, g:g + 2]         # fine (k 2..3, j -2..-1, i 0..1) <-> coarse (9, 7, 0)
    G0 = wk.configs.join_patches(lc.U, lc.origin, (32, 32, 32))
    assert np.allclose(kids.mean(axis=(1, 2, 3)), G0[:, 9, 7, 0], rtol=1e-13, atol=1e-14)

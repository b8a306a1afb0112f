"""Pins of the regridding oracle (oracle/regrid.py) against facts that do not come from it."""
import copy

import numpy as np
import pytest

import workloads as wk
from oracle import regrid as rg


@pytest.fixture(scope="module")
def hier():
    return wk.config_hierarchy(False, 3, 128, n=8, thresholds=(2.5, 3.5))


def test_flags_on_a_hand_made_field():
    n = 8
    origin = wk.morton_patch_origins(2, 2, 2, n)
    U = np.zeros((5, 8, n, n, n))
    lev = wk.Level(n=n, g=3, level=0, dx=1 / 16, origin=origin, domain_cells=(16, 16, 16), bc=(0,) * 6,
                   self_periodic=False, U=U)
    p = 5                                    # one cell above the threshold in the (z hi, y lo, x hi) block of patch 5
    U[0, p, 6, 1, 7] = 2.0
    U[0, 3, 0, 0, 0] = 1.0                   # exactly the threshold: not flagged (strict >)
    U[1, 2, 4, 4, 4] = 9.0                   # another field: ignored
    f = rg.flag_blocks(lev, 0, 1.0)
    assert f.shape == (8, 2, 2, 2) and f.sum() == 1 and f[p, 1, 0, 1]
    g = wk.patch_flags_to_block_grid(lev, f)
    ox, oy, oz = origin[p]
    assert g.sum() == 1 and g[oz // 4 + 1, oy // 4, ox // 4 + 1]


def test_children_average_to_the_parent_and_kept_patches_are_copies(hier):
    l0, l1, l2 = hier.levels
    # new level 1: drop the first 10 patches, add every allowed block next to the old set
    old = wk.origins_to_blocks(l1.origin, l1.n, l0.domain_cells[0] // (l0.n // 2))
    new = old.copy()
    o = l1.origin // l1.n
    new[o[:10, 2], o[:10, 1], o[:10, 0]] = False
    new |= np.roll(old, 1, axis=2)
    origin_new = wk.blocks_to_origins(new, l1.n)
    Unew = rg.regrid_fill(l0, l1, origin_new)
    oldmap = {tuple(o): p for p, o in enumerate(l1.origin)}
    n, h = l1.n, l1.n // 2
    G0 = wk.configs.join_patches(l0.U, l0.origin, (32, 32, 32))
    nborn = 0
    for p, o in enumerate(origin_new):
        if tuple(o) in oldmap:
            assert np.array_equal(Unew[:, p], l1.U[:, oldmap[tuple(o)]])
        else:
            nborn += 1
            mean = Unew[:, p].reshape(5, h, 2, h, 2, h, 2).mean(axis=(2, 4, 6))
            par = G0[:, o[2] // 2:o[2] // 2 + h, o[1] // 2:o[1] // 2 + h, o[0] // 2:o[0] // 2 + h]
            assert np.allclose(mean, par, rtol=1e-14, atol=1e-15)
            assert np.abs(Unew[:, p] - np.repeat(np.repeat(np.repeat(par, 2, 1), 2, 2), 2, 3)).max() > 1e-3   # slopes are used
    assert nborn >= 5


def test_linear_field_is_reproduced_exactly_and_uniform_stays_uniform():
    n = 8
    origin0 = wk.morton_patch_origins(4, 4, 4, n)
    c = np.arange(32) + 0.5
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    lin = 1.0 + 0.5 * X - 0.25 * Y + 0.125 * Z
    G = np.stack([lin, 2 * lin, np.full_like(lin, 3.0), -lin, lin + 7])
    l0 = wk.Level(n=n, g=3, level=0, dx=1 / 32, origin=origin0, domain_cells=(32, 32, 32), bc=(0,) * 6,
                  self_periodic=False, U=wk.split_into_patches(G, n, origin0))
    origin_new = np.array([[24, 24, 24], [32, 24, 24], [24, 32, 40]], np.int32)    # away from the periodic seam
    U = rg.regrid_fill(l0, None, origin_new)
    cf = (np.arange(64) + 0.5) / 2                         # fine cell centres in coarse units
    Zf, Yf, Xf = np.meshgrid(cf, cf, cf, indexing="ij")
    linf = 1.0 + 0.5 * Xf - 0.25 * Yf + 0.125 * Zf
    for p, (ox, oy, oz) in enumerate(origin_new):
        ex = linf[oz:oz + n, oy:oy + n, ox:ox + n]
        assert np.abs(U[0, p] - ex).max() <= 1e-14
        assert np.abs(U[3, p] + ex).max() <= 1e-14
        assert np.array_equal(U[2, p], np.full((n, n, n), 3.0))


def test_new_born_patches_on_outflow_faces_never_see_the_far_side():
    """DESIGN.md section 3 (AMR at non-periodic domain faces): beyond an OUTFLOW face the +-1 stencil of the O8
    interpolation is the coarse ghost cell there = the nearest in-domain cell, never the cell on the far side of the
    domain.  Outflow x faces, periodic y and z:
      * a field linear in x: the outermost parent column of a patch on an x face gets no x slope (its one-sided
        difference against the clamped cell is 0), the other columns are exact;
      * changing ONLY the coarse cells on the far side of the domain leaves a patch on the x lo face bitwise unchanged
        (and does change it when the faces are declared periodic);
      * along periodic y the seam is in the stencil: the value across it decides the slope."""
    n = 8
    origin0 = wk.morton_patch_origins(4, 4, 4, n)
    c = np.arange(32) + 0.5
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    lin = 1.0 + 0.5 * X
    saw = np.where(Y < 1, 5.0, 1.0) + 0 * X            # along periodic y: cell 0 is 5, all others 1
    G = np.stack([lin, 2 * lin, saw, -lin, lin + 7])
    bc = (1, 1, 0, 0, 0, 0)
    l0 = wk.Level(n=n, g=3, level=0, dx=1 / 32, origin=origin0, domain_cells=(32, 32, 32), bc=bc,
                  self_periodic=False, U=wk.split_into_patches(G, n, origin0))
    origin_new = np.array([[0, 24, 24], [56, 24, 24], [24, 0, 24]], np.int32)      # on x lo, on x hi, on the periodic y seam
    U = rg.regrid_fill(l0, None, origin_new)
    cf = (np.arange(64) + 0.5) / 2
    linf = 1.0 + 0.5 * cf
    # x lo patch: parent column 0 has slope minmod(U0 - U0, U1 - U0) = 0; columns 1..3 are exact
    assert np.array_equal(U[0, 0, :, :, 0], U[0, 0, :, :, 1]) and np.all(U[0, 0, :, :, 0] == lin[0, 0, 0])
    assert np.abs(U[0, 0, :, :, 2:] - linf[None, None, 2:8]).max() <= 1e-14
    # x hi patch: parent column 31 likewise, columns 28..30 exact
    assert np.array_equal(U[0, 1, :, :, 6], U[0, 1, :, :, 7]) and np.all(U[0, 1, :, :, 7] == lin[0, 0, 31])
    assert np.abs(U[0, 1, :, :, :6] - linf[None, None, 56:62]).max() <= 1e-14
    # only the far side changes: an outflow stencil must not notice, a periodic one must
    Gc = rg._dense(l0)
    plain = rg.prolong_patch(Gc, (0, 24, 24), n, bc)
    wrapped = rg.prolong_patch(Gc, (0, 24, 24), n, (0,) * 6)
    bump = Gc.copy()
    bump[:, :, :, 31] -= 100.0                          # now below cell 0: a wrapped stencil sees a monotone profile
    assert np.array_equal(rg.prolong_patch(bump, (0, 24, 24), n, bc), plain)
    assert not np.array_equal(rg.prolong_patch(bump, (0, 24, 24), n, (0,) * 6), wrapped)
    # along periodic y: cell 0 (5.0) is a strict maximum between cells 31 and 1 (both 1.0) -> no y slope ...
    assert np.all(U[2, 2, :, 0:2, :] == 5.0) and np.all(U[2, 2, :, 2:, :] == 1.0)
    bump = Gc.copy()
    bump[2, :, 31, :] = 9.0                             # ... and between 9 and 1 it is monotone: slope minmod(-4, -4) = -4
    Uy = rg.prolong_patch(bump, (24, 0, 24), n, bc)
    assert np.all(Uy[2, :, 0, :] == 6.0) and np.all(Uy[2, :, 1, :] == 4.0)


def test_a_local_extremum_gets_no_slope():
    """minmod: at a coarse cell that is a strict maximum along x the two children along x are equal."""
    n = 8
    origin0 = wk.morton_patch_origins(4, 4, 4, n)
    G = np.zeros((5, 32, 32, 32))
    G[0, :, :, 13] = 1.0
    l0 = wk.Level(n=n, g=3, level=0, dx=1 / 32, origin=origin0, domain_cells=(32, 32, 32), bc=(0,) * 6,
                  self_periodic=False, U=wk.split_into_patches(G, n, origin0))
    U = rg.regrid_fill(l0, None, np.array([[24, 24, 24]], np.int32))      # coarse cells 12..15
    assert np.array_equal(U[0, 0, :, :, 2], U[0, 0, :, :, 3]) and np.all(U[0, 0, :, :, 2:4] == 1.0)
    assert np.all(U[0, 0, :, :, :2] == 0.0) and np.all(U[0, 0, :, :, 4:] == 0.0)


def test_regrid_keeps_the_composite_totals(oracle, hier):
    """Replace level 2 by a different properly nested set (kept + new-born patches) and level 1 is unchanged:
    the composite totals of the hierarchy do not move (new-born children average to their parents)."""
    wl = copy.deepcopy(hier)
    l0, l1, l2 = wl.levels
    g = l0.g
    before = oracle.hierarchy_totals([oracle.ghosted(lv.U, g) for lv in wl.levels], wl.levels)
    flags = rg.flag_blocks(l1, 0, 2.0 * l1.U[0].mean())
    grid = wk.patch_flags_to_block_grid(l1, flags)
    cover1 = wk.origins_to_blocks(l1.origin, l1.n, l0.domain_cells[0] // (l0.n // 2))
    sel = wk.select_blocks(grid, cover1, grow=False)
    origin_new = wk.blocks_to_origins(sel, l2.n)
    assert len(origin_new) > l2.npatch                   # a lower threshold than the generator's: the level grows
    U2 = rg.regrid_fill(l1, l2, origin_new)
    wl.levels[2] = wk.Level(n=l2.n, g=g, level=2, dx=l2.dx, origin=origin_new, domain_cells=l2.domain_cells,
                            bc=l2.bc, self_periodic=False, U=U2)
    after = oracle.hierarchy_totals([oracle.ghosted(lv.U, g) for lv in wl.levels], wl.levels)
    absn = np.array([np.abs(l0.U[f]).sum() * l0.dx ** 3 for f in range(5)])
    assert (np.abs(after - before) / absn).max() < 1e-13
    # and the regridded hierarchy steps (the new level is properly nested for the link tables)
    r = oracle.hierarchy_step(wl)
    assert all(np.isfinite(u).all() for u in r["U"])
    assert (np.abs(r["totals_after"] - before) / absn).max() < 1e-13

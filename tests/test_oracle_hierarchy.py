"""Pins of the oracle's L-level recursive subcycling (oracle.api.hierarchy_step) against
facts that do not come from it: composite conservation (and its failure without the reflux), the substep
count 2^l, free-stream preservation, the exact translation of a density wave, and the two-level pins'
subject (two_level_step) as the L = 2 special case."""
import numpy as np
import pytest

import workloads as wk


@pytest.fixture(scope="module")
def small_hierarchy():
    # 128^3 finest index space, 8^3 patches: root 32^3 = 64 patches, level 1 ~100, level 2 ~10
    return {mhd: wk.config_hierarchy(mhd, 3, 128, n=8, thresholds=(2.5, 3.5)) for mhd in (False, True)}


def test_hierarchy_is_properly_nested(small_hierarchy):
    """The generator's promise (data only): levels are the means of the next, every level-(l+1) patch
    sits on an aligned (n/2)^3 block of level-l cells, and the 27 blocks around it are all inside level l."""
    wl = small_hierarchy[False]
    l0, l1, l2 = wl.levels
    assert l0.npatch == 64 and 20 <= l1.npatch <= 300 and 4 <= l2.npatch <= 60, wl.note
    for lc, lf in ((l0, l1), (l1, l2)):
        n, nb = lc.n, lc.n // 2
        Nc = lc.domain_cells[0]
        cov = np.zeros((Nc, Nc, Nc), bool)
        val = np.zeros((lc.nfields, Nc, Nc, Nc))
        for p, (ox, oy, oz) in enumerate(lc.origin):
            cov[oz:oz + n, oy:oy + n, ox:ox + n] = True
            val[:, oz:oz + n, oy:oy + n, ox:ox + n] = lc.U[:, p]
        for p, (ox, oy, oz) in enumerate(lf.origin):
            assert ox % n == 0 and oy % n == 0 and oz % n == 0
            cx, cy, cz = ox // 2, oy // 2, oz // 2
            idx = [np.arange(c - nb, c + 2 * nb) % Nc for c in (cz, cy, cx)]
            assert cov[np.ix_(*idx)].all()
            mean = lf.U[:, p].reshape(lc.nfields, nb, 2, nb, 2, nb, 2).mean(axis=(2, 4, 6))
            assert np.allclose(val[:, cz:cz + nb, cy:cy + nb, cx:cx + nb], mean, rtol=1e-13, atol=1e-14)


@pytest.mark.parametrize("mhd", [False, True])
def test_three_level_composite_conservation(oracle, small_hierarchy, mhd):
    """Composite totals over three levels unchanged by one root step (1 + 2 + 4 level steps) to 1e-13 of
    sum|U|; without the reflux the same run leaks.  After the cascade of restrictions the root level alone
    carries the composite totals (every covered cell is the mean of its children)."""
    wl = small_hierarchy[mhd]
    l0 = wl.levels[0]
    r = oracle.hierarchy_step(wl)
    assert r["nsteps"] == [1, 2, 4]
    nfc = 8 if mhd else 5
    absn = np.array([np.abs(l0.U[f]).sum() * l0.dx ** 3 for f in range(l0.nfields)])
    rel = np.abs(r["totals_after"] - r["totals_before"])[:nfc] / absn[:nfc]
    assert rel.max() < 1e-13, rel
    root = np.array([r["U"][0][f].sum() * l0.dx ** 3 for f in range(l0.nfields)])
    assert (np.abs(root - r["totals_after"])[:nfc] / absn[:nfc]).max() < 1e-13
    root0 = np.array([l0.U[f].sum() * l0.dx ** 3 for f in range(l0.nfields)])
    assert (np.abs(root0 - r["totals_before"])[:nfc] / absn[:nfc]).max() < 1e-13
    r2 = oracle.hierarchy_step(wl, do_reflux=False)
    rel2 = np.abs(r2["totals_after"] - r2["totals_before"])[:5] / absn[:5]
    assert rel2.max() > 1e-7, rel2
    for l in range(3):
        assert np.abs(r["U"][l] - wl.levels[l].U).max() > 1e-3


def test_two_levels_are_the_two_level_step(oracle):
    """L = 2: the recursion is O9 call for call, so the results are bitwise those of two_level_step (whose
    own pins are P13/P14 in test_oracle_amr.py)."""
    wl = wk.config4_two_level(True, nfine=64, threshold=3.0)
    a = oracle.two_level_step(wl)
    b = oracle.hierarchy_step(wl)
    assert a["dt0"] == b["dt0"]
    assert np.array_equal(a["Uc"], b["U"][0]) and np.array_equal(a["Uf"], b["U"][1])


def _uniform_hierarchy(small, state):
    wl = small
    import copy
    w = copy.deepcopy(wl)
    for lv in w.levels:
        for f in range(lv.nfields):
            lv.U[f] = state[f]
    return w


def test_free_stream_is_preserved_on_every_level(oracle, small_hierarchy):
    """A uniform moving magnetised state is a fixed point of every operator of the cycle (step,
    prolongation in space and time, restriction, reflux): all levels return it to round-off."""
    gamma = 5.0 / 3.0
    rho, v, p, B = 1.3, (0.4, -0.7, 0.2), 0.9, (0.3, 0.5, -0.2)
    E = p / (gamma - 1) + 0.5 * rho * sum(c * c for c in v) + 0.5 * sum(c * c for c in B)
    state = [rho, rho * v[0], rho * v[1], rho * v[2], E, B[0], B[1], B[2], 0.0]
    w = _uniform_hierarchy(small_hierarchy[True], state)
    r = oracle.hierarchy_step(w)
    for l in range(3):
        for f in range(9):
            assert np.abs(r["U"][l][f] - state[f]).max() <= 2e-14, (l, f)


def test_density_wave_translates_through_the_levels(oracle):
    """Exact solution: rho = 1 + 0.2 sin(2 pi (x - t)), u = 1, p = 1 translates unchanged.  A 3-level
    hierarchy refined around the middle of the wave, advanced by root steps, stays within the second-order
    error of the ROOT resolution everywhere and does better than the root-only run where it is refined -
    which fails if the fine levels take the wrong number of substeps, the wrong dt, or halos prolonged at the
    wrong time (an O(dt) error at every coarse-fine face)."""
    gamma = 5.0 / 3.0
    n, N2 = 8, 128
    c = (np.arange(N2) + 0.5) / N2

    def state(t, N):
        x = (np.arange(N) + 0.5) / N
        rho = 1 + 0.2 * np.sin(2 * np.pi * (x - t))
        return np.broadcast_to(rho[None, None, :], (N, N, N))

    rho = state(0.0, N2)
    one = np.ones_like(rho)
    G = wk.primitive_to_conserved(rho, [one, 0 * one, 0 * one], one, gamma)
    # refine by position instead of by density: mark with a helper density, then put the wave's data in
    marker = np.ones((N2, N2, N2))
    marker[32:96, 32:96, 32:96] = 4.0
    marker[48:80, 48:80, 48:80] = 16.0
    Gm = G.copy()
    Gm[0] = marker
    wm = wk.nested_hierarchy_from_fine("wave", Gm, 3, n, (2.0, 2.5), gamma, False, wk.configs.LIM_MC, wk.configs.RS_HLLC)
    levels = []
    fields = [None, None, G]
    for l in (1, 0):
        M = fields[l + 1].shape[1] // 2
        fields[l] = fields[l + 1].reshape(5, M, 2, M, 2, M, 2).mean(axis=(2, 4, 6))
    for l, lv in enumerate(wm.levels):
        lv.U = wk.split_into_patches(fields[l], n, lv.origin)
    assert wm.levels[1].npatch >= 8 and wm.levels[2].npatch >= 8, wm.note
    t = 0.0
    wl = wm
    for _ in range(4):
        r = oracle.hierarchy_step(wl)
        t += r["dt0"]
        for l, lv in enumerate(wl.levels):
            lv.U = r["U"][l]
    # exact cell averages ~ point values at second order; compare with the exact profile per level
    errs = []
    for l, lv in enumerate(wl.levels):
        N = lv.domain_cells[0]
        ex = state(t, N)
        e = 0.0
        for p, (ox, oy, oz) in enumerate(lv.origin):
            e = max(e, np.abs(lv.U[0, p] - ex[oz:oz + n, oy:oy + n, ox:ox + n]).max())
        errs.append(e)
    # root-only run of the same four steps
    import copy
    w0 = copy.deepcopy(wm)
    w0.levels = [copy.deepcopy(wm.levels[0])]
    w0.levels[0].U = wk.split_into_patches(fields[0], n, w0.levels[0].origin)
    ra = oracle.advance(w0.levels[0], w0, 4)
    t0 = sum(ra["dts"])
    ex0 = state(t0, 32)
    e0 = max(np.abs(ra["U"][0, p] - ex0[oz:oz + n, oy:oy + n, ox:ox + n]).max()
             for p, (ox, oy, oz) in enumerate(w0.levels[0].origin))
    assert abs(t - t0) < 1e-3 * t0               # (each run is compared with the exact profile at its own time)
    print(errs, e0)
    assert errs[0] <= 1.5 * e0, (errs, e0)          # the root is no worse than without refinement
    assert errs[2] <= 0.6 * e0, (errs, e0)          # and the refined region is better than the root alone


def test_schedule_of_a_three_level_root_step(oracle, small_hierarchy, monkeypatch):
    """The order of operations, written out by hand for L = 3 (W-cycle: PAPER.md:31 finer levels take
    their own smaller steps, :59 a level is corrected once the finer one has caught up), against the calls
    hierarchy_step really makes: (operator, level it acts on, dt/dt0 or theta)."""
    wl = small_hierarchy[False]
    dxs = [lv.dx for lv in wl.levels]
    log = []
    real = dict(step=oracle.step, prolong=oracle.prolong_ghosts, restrict=oracle.restrict, reflux=oracle.reflux)

    def lvl(dx):
        return int(np.argmin([abs(dx - d) for d in dxs]))

    def step(Ug, g, dt, dx, *a, **k):
        log.append(("step", lvl(dx), dt))
        return real["step"](Ug, g, dt, dx, *a, **k)

    def prolong(Uf, mask, lf, Uo, Un, lc, theta):
        log.append(("prolong", lf.level, theta))
        return real["prolong"](Uf, mask, lf, Uo, Un, lc, theta)

    def restrict(Uf, lf, Uc, lc):
        log.append(("restrict", lc.level, None))
        return real["restrict"](Uf, lf, Uc, lc)

    def reflux(Uc, lc, Fc, lf, Ff, dt):
        log.append(("reflux", lc.level, dt))
        return real["reflux"](Uc, lc, Fc, lf, Ff, dt)

    monkeypatch.setattr(oracle, "step", step)
    monkeypatch.setattr(oracle, "prolong_ghosts", prolong)
    monkeypatch.setattr(oracle, "restrict", restrict)
    monkeypatch.setattr(oracle, "reflux", reflux)
    r = oracle.hierarchy_step(wl)
    dt0 = r["dt0"]
    fine_pair = [("prolong", 2, 0.0), ("step", 2, dt0 / 4), ("prolong", 2, 0.5), ("step", 2, dt0 / 4),
                 ("restrict", 1, None), ("reflux", 1, dt0 / 2)]
    want = ([("step", 0, dt0)]
            + [("prolong", 1, 0.0), ("step", 1, dt0 / 2)] + fine_pair
            + [("prolong", 1, 0.5), ("step", 1, dt0 / 2)] + fine_pair
            + [("restrict", 0, None), ("reflux", 0, dt0)])
    assert log == want


def test_four_levels_two_middle_levels(oracle):
    """L = 4 (two levels that are fine side and coarse side at once): 1 + 2 + 4 + 8 level steps, composite
    totals conserved to 1e-13."""
    wl = wk.config_hierarchy(True, 4, 128, n=8, thresholds=(1.5, 2.5, 3.5))
    assert [lv.npatch for lv in wl.levels][0] == 8 and all(lv.npatch >= 4 for lv in wl.levels), wl.note
    r = oracle.hierarchy_step(wl)
    assert r["nsteps"] == [1, 2, 4, 8]
    l0 = wl.levels[0]
    absn = np.array([np.abs(l0.U[f]).sum() * l0.dx ** 3 for f in range(9)])
    assert (np.abs(r["totals_after"] - r["totals_before"])[:8] / absn[:8]).max() < 1e-13

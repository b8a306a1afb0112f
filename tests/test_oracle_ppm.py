"""Pins of the PPM oracle (reading R-PPM of DESIGN.md section 13): the
reconstruction against closed forms and hand-worked cases, no new extrema, the Sod tube against the exact
solution (better than PLM), third-order convergence on a smooth wave, bitwise invariants (uniform state, axis
independence, axis permutation with the sweep order reversed), conservation, and the splitting error of the
two sweep orders."""
import numpy as np
import pytest

import workloads as wk
from test_oracle_sod import cell_averaged_exact, run_sod

RS_HLLC = 1


# ---- P1 + P2: the parabola of one cell -------------------------------------------------------------------

def _cell_averages(coef, x0, dx, k):
    """Exact cell averages of sum_m coef[m] x^m over the cells x0 + (k-1/2 .. k+1/2) dx."""
    P = np.polynomial.Polynomial(coef).integ()
    return np.array([(P(x0 + (i + 0.5) * dx) - P(x0 + (i - 0.5) * dx)) / dx for i in k])


def test_interface_values_are_exact_for_cubics_and_the_parabola_is_reproduced(oracle):
    """CW84 (1.6): with unlimited slopes the interface value is the fourth-order one, exact for cubic
    polynomials; for a parabola the triple (aL, aR, a6) then IS the parabola."""
    dx, x0 = 0.1, 0.3
    k = np.arange(-2, 3)
    cubic = [1.0, 2.0, 0.5, 0.25]                       # monotone on the stencil: the limiter is inactive
    a = _cell_averages(cubic, x0, dx, k)
    aL, aR = oracle.ppm_parabola(a)
    P = np.polynomial.Polynomial(cubic)
    assert abs(aL - P(x0 - 0.5 * dx)) < 1e-14 and abs(aR - P(x0 + 0.5 * dx)) < 1e-14
    par = [0.7, 1.3, 2.0]                               # vertex at x = -0.325: monotone on the stencil
    a = _cell_averages(par, x0, dx, k)
    aL, aR = oracle.ppm_parabola(a)
    a6 = 6.0 * (a[2] - 0.5 * (aL + aR))
    Q = np.polynomial.Polynomial(par)
    for xi in np.linspace(0.0, 1.0, 11):                # CW84 (1.4): a(xi) = aL + xi (Da + a6 (1 - xi))
        assert abs(aL + xi * ((aR - aL) + a6 * (1.0 - xi)) - Q(x0 + (xi - 0.5) * dx)) < 1e-14


def test_monotonisation_cases_worked_by_hand(oracle):
    # local extremum: flat
    assert oracle.ppm_parabola([0.0, 1.0, 2.0, 1.0, 0.0]) == (2.0, 2.0)
    # constant and linear data are reproduced
    assert oracle.ppm_parabola([3.0] * 5) == (3.0, 3.0)
    aL, aR = oracle.ppm_parabola([1.0, 2.0, 3.0, 4.0, 5.0])
    assert abs(aL - 2.5) < 1e-15 and abs(aR - 3.5) < 1e-15
    # a cell next to a jump, stencil (0, 0, 0.1, 1, 1), by hand:
    #   dm_{i-1} = 0 (0, 0, 0.1: not strictly monotone), dm_i = min(0.5, 0.2, 1.8) = 0.2, dm_{i+1} = 0 (0.1, 1, 1)
    #   a_{i-1/2} = 0 + 0.05 - (0.2 - 0)/6 = 1/60 ;  a_{i+1/2} = 0.1 + 0.45 - (0 - 0.2)/6 = 0.55 + 1/30
    #   (aR - aL)(a - (aL+aR)/2) = 0.5667 (0.1 - 0.3) < -(0.5667)^2/6  ->  aR = 3 a - 2 aL = 0.3 - 1/30
    aL, aR = oracle.ppm_parabola([0.0, 0.0, 0.1, 1.0, 1.0])
    assert abs(aL - 1.0 / 60.0) < 1e-15 and abs(aR - (0.3 - 1.0 / 30.0)) < 1e-15
    # the mirror image swaps the roles
    bL, bR = oracle.ppm_parabola([1.0, 1.0, 0.1, 0.0, 0.0])
    assert abs(bR - aL) < 1e-15 and abs(bL - aR) < 1e-15


def test_parabola_never_leaves_the_range_of_the_neighbours(oracle):
    rng = np.random.default_rng([wk.SEED, 301])
    for _ in range(2000):
        a = rng.standard_normal(5) * (10.0 ** rng.integers(-3, 3))
        aL, aR = oracle.ppm_parabola(a)
        lo, hi = min(a[1:4]), max(a[1:4])
        a6 = 6.0 * (a[2] - 0.5 * (aL + aR))
        xi = np.linspace(0, 1, 21)
        prof = aL + xi * ((aR - aL) + a6 * (1 - xi))
        tol = 1e-12 * max(1.0, abs(hi), abs(lo))
        assert prof.min() >= lo - tol and prof.max() <= hi + tol                     # bounded by the neighbours
        assert prof.min() >= min(aL, aR) - tol and prof.max() <= max(aL, aR) + tol   # monotone inside the cell


# ---- the scheme ---------------------------------------------------------------------------------------------

def _advected_profile(kind, N, axis=0, n=8):
    """rho profile along `axis` in a uniform flow u = 1, p = 1 (exact solution: translation), periodic."""
    wl = wk.smooth_wave_patchset("density", N, axis=axis, n=n)
    if kind == "step":
        lev = wl.levels[0]
        c = (np.arange(N) + 0.5) / N
        G = wk.configs.join_patches(lev.U, lev.origin, tuple(int(v) for v in lev.domain_cells)[::-1])
        shape = [1, 1, 1]
        shape[2 - axis] = N
        rho = np.where((c > 0.25) & (c < 0.6), 2.0, 1.0).reshape(shape) + 0 * G[0]
        v = [0 * rho, 0 * rho, 0 * rho]
        v[axis] = 0 * rho + 1.0
        G = wk.primitive_to_conserved(rho, v, 0 * rho + 1.0, wl.gamma)
        lev.U = wk.split_into_patches(G, n, lev.origin)
    return wl


def _evolve_ppm(oracle, wl, t_end=None, nsteps=None, cfl=None):
    lev = wl.levels[0]
    g = lev.g
    Ug = oracle.ghosted(lev.U, g)
    t, step_no = 0.0, 0
    while True:
        oracle.fill_ghosts(Ug, g, lev.origin, lev.domain_cells, lev.bc, lev.self_periodic)
        sm = oracle.smax(Ug, g, wl.gamma)
        dt = (cfl or wl.cfl) * lev.dx / sm
        if t_end is not None:
            dt = min(dt, t_end - t)
        for d in oracle.PPM_ORDERS[step_no % 2]:
            oracle.fill_ghosts(Ug, g, lev.origin, lev.domain_cells, lev.bc, lev.self_periodic)
            Ug = oracle.ppm_sweep(Ug, g, d, dt, lev.dx, wl.gamma, RS_HLLC)["U"]
        t += dt
        step_no += 1
        if (nsteps is not None and step_no == nsteps) or (t_end is not None and t >= t_end - 1e-14):
            return oracle.interior(Ug, g), t


def test_no_new_extrema_on_a_step_profile(oracle):
    wl = _advected_profile("step", 64)
    U, _ = _evolve_ppm(oracle, wl, nsteps=40)
    rho = U[0]
    assert rho.min() >= 1.0 - 1e-12 and rho.max() <= 2.0 + 1e-12
    assert np.abs(U[0] - wl.levels[0].U[0]).max() > 0.3            # it did move
    # u and p stay uniform to round-off (contact discontinuity)
    assert np.abs(U[1] / U[0] - 1.0).max() < 1e-12


def test_sod_is_closer_to_the_exact_solution_than_plm(oracle):
    """Config 1's tube with PPM: L1(rho) at N = 32 against the exact cell averages is below the PLM value
    (1.50e-2, tests/test_oracle_sod.py) at the same time, and converges at the shock-dominated rate."""
    t_end = 0.126985
    errs = {}
    for N in (32, 64):
        wl = wk.config1_sod(n=N)
        U, t = _evolve_ppm(oracle, wl, t_end=t_end, cfl=0.4)
        rho = U[0, 0, 5, 7, :]
        errs[N] = np.mean(np.abs(rho - cell_averaged_exact(N, t)))
        assert np.array_equal(U[0, 0], np.broadcast_to(rho, U[0, 0].shape))       # j/k invariance, bitwise
        assert np.all(U[2] == 0) and np.all(U[3] == 0)
    plm, _ = run_sod(oracle, 32, t_end=t_end)
    e_plm = np.mean(np.abs(plm[0, 0, 5, 7, :] - cell_averaged_exact(32, t_end)))
    assert errs[32] < e_plm and errs[32] < 1.5e-2, (errs, e_plm)
    assert 1.4 <= errs[32] / errs[64] <= 2.4, errs


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_third_order_on_a_smooth_wave_away_from_extrema(oracle, axis):
    """Advected density wave: the error away from the extrema (where the monotonisation clips the parabola)
    drops by >= 4 per doubling and by >= 40 over the two doublings 16 -> 64 (measured: 4.9 and 11.5 - the clipped
    extrema of the coarsest grid travel with the wave); the L1 error over all cells drops by >= 3 per doubling."""
    t_end = 0.2
    e_smooth, e_all = [], []
    for N in (16, 32, 64):
        wl = _advected_profile("wave", N, axis=axis)
        U, _ = _evolve_ppm(oracle, wl, t_end=t_end)
        exact = wk.smooth_wave_patchset("density", N, axis=axis, t=t_end).levels[0].U
        lev = wl.levels[0]
        dom = tuple(int(v) for v in lev.domain_cells)[::-1]          # (Nz, Ny, Nx)
        d = np.abs(wk.configs.join_patches(U, lev.origin, dom)[0] - wk.configs.join_patches(exact, lev.origin, dom)[0])
        c = (np.arange(N) + 0.5) / N
        shape = [1, 1, 1]
        shape[2 - axis] = N
        away = (np.abs(np.cos(2 * np.pi * (c - t_end))) > 0.6).reshape(shape) & (d >= 0)
        e_smooth.append(d[away].max())
        e_all.append(d.mean())
    assert e_smooth[0] / e_smooth[1] >= 4.0 and e_smooth[1] / e_smooth[2] >= 4.0, e_smooth
    assert e_smooth[0] / e_smooth[2] >= 40.0, e_smooth              # better than second order over the two doublings
    assert e_all[0] / e_all[1] >= 3.0 and e_all[1] / e_all[2] >= 3.0, e_all
    assert e_all[2] < 2e-4


def test_uniform_moving_state_is_preserved_bitwise(oracle):
    wl = wk.config2_random_patches(npatch=2)
    lev = wl.levels[0]
    lev.U[...] = wk.primitive_to_conserved(np.full((16,) * 3, 1.3), [np.full((16,) * 3, v) for v in (0.4, -0.7, 0.2)],
                                           np.full((16,) * 3, 0.9), wl.gamma)[:, None]
    r = oracle.ppm_advance(lev, wl, 2)
    assert np.array_equal(r["U"], lev.U)


def test_axis_permutations_with_the_sweep_order_relabelled_agree_to_round_off(oracle):
    """The sweep code is direction-agnostic: relabelling the axes (cyclically: old x -> new y, old y -> new z,
    old z -> new x; and the mirror x <-> z) together with the velocity components and the sweep order gives the
    relabelled result to round-off (A19: only the order of the sum vx^2 + vy^2 + vz^2 changes; P6 of the PLM path
    is stated the same way)."""
    wl = wk.config2_random_patches(npatch=3)
    lev = wl.levels[0]
    g = lev.g
    dt = 0.3 * lev.dx / oracle.smax(oracle.ghosted(lev.U, g), g, wl.gamma)

    def run(U, order):
        Ug = oracle.ghosted(U, g)
        for d in order:
            oracle.fill_ghosts(Ug, g, lev.origin, lev.domain_cells, lev.bc, True)
            Ug = oracle.ppm_sweep(Ug, g, d, dt, lev.dx, wl.gamma, RS_HLLC)["U"]
        return oracle.interior(Ug, g)

    a = run(lev.U, (0, 1, 2))
    assert np.abs(a - lev.U).max() > 1e-3
    # cyclic: A'[k', j', i'] = A[i', k', j'], (vx', vy', vz') = (vz, vx, vy); sweeps x, y, z become y', z', x'
    Uc = np.ascontiguousarray(lev.U[[0, 3, 1, 2, 4]].transpose(0, 1, 3, 4, 2))
    b = run(Uc, (1, 2, 0))
    back = np.ascontiguousarray(b[[0, 2, 3, 1, 4]].transpose(0, 1, 4, 2, 3))
    assert np.abs(back - a).max() <= 1e-13 * np.abs(a).max()
    # mirror: x <-> z, order reversed
    Ut = np.ascontiguousarray(lev.U[[0, 3, 2, 1, 4]].transpose(0, 1, 4, 3, 2))
    m = run(Ut, (2, 1, 0))
    mb = np.ascontiguousarray(m[[0, 3, 2, 1, 4]].transpose(0, 1, 4, 3, 2))
    assert np.abs(mb - a).max() <= 1e-13 * np.abs(a).max()


def test_conservation_on_periodic_patches(oracle):
    wl = wk.config2_random_patches(npatch=4)
    lev = wl.levels[0]
    r = oracle.ppm_advance(lev, wl, 2)
    tot0, tot1 = lev.U.sum(axis=(2, 3, 4)), r["U"].sum(axis=(2, 3, 4))
    absn = np.abs(lev.U).sum(axis=(2, 3, 4))
    assert (np.abs(tot1 - tot0) / absn).max() < 1e-13
    assert all(c["positivity_fallback_cells"] == 0 for c in r["counters"])


def test_the_two_sweep_orders_differ_by_the_splitting_error(oracle):
    """x-y-z and z-y-x are both first-order-split approximations of the same step: their difference is the
    commutator term, O(dt^2) per step (halving dt divides it by ~4); alternating them (oracle.ppm_advance)
    is the usual Strang-type symmetrisation."""
    N = 16
    c = (np.arange(N) + 0.5) / N
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    rho = 1.0 + 0.2 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) + 0.1 * np.sin(2 * np.pi * (Z + X))
    v = [0.5 + 0.1 * np.sin(2 * np.pi * Y), -0.3 + 0.1 * np.cos(2 * np.pi * Z), 0.2 + 0.1 * np.sin(2 * np.pi * X)]
    G = wk.primitive_to_conserved(rho, v, 1.0 + 0.0 * rho, 1.4)
    wl = wk.uniform_grid_workload("ppm_split", G, 8, 1.4, False, 2, RS_HLLC, 0.3, 1)
    lev = wl.levels[0]
    g = lev.g

    def run(order, dt):
        Ug = oracle.ghosted(lev.U, g)
        for d in order:
            oracle.fill_ghosts(Ug, g, lev.origin, lev.domain_cells, lev.bc, False)
            Ug = oracle.ppm_sweep(Ug, g, d, dt, lev.dx, wl.gamma, RS_HLLC)["U"]
        return oracle.interior(Ug, g)

    diffs = []
    for dt in (0.2 * lev.dx, 0.1 * lev.dx):
        diffs.append(np.abs(run((0, 1, 2), dt) - run((2, 1, 0), dt)).max())
    assert 3.0 <= diffs[0] / diffs[1] <= 5.0, diffs
    assert diffs[0] > 1e-8

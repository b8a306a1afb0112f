"""Pins P4, P5, P6, P8 (full step), P9, P15: properties of the oracle's full
step that hold independently of any implementation."""
import numpy as np
import pytest

import workloads as wk

LIM_MC, LIM_MINMOD = 2, 1
RS_HLL, RS_HLLC, RS_HLLD = 0, 1, 2


def one_step(oracle, lev, wl, dtype=np.float64, limiter=None, riemann=None, dt=None, ch=None, alpha=None):
    Ug = oracle.ghosted(lev.U, lev.g, dtype)
    oracle.fill_ghosts(Ug, lev.g, lev.origin, lev.domain_cells, lev.bc, lev.self_periodic)
    sm = oracle.smax(Ug, lev.g, wl.gamma)
    dt = wl.cfl * lev.dx / sm if dt is None else dt
    r = oracle.step(Ug, lev.g, dt, lev.dx, wl.gamma, wl.limiter if limiter is None else limiter,
                    wl.riemann if riemann is None else riemann, ch=sm if ch is None else ch,
                    alpha=wl.alpha if alpha is None else alpha)
    return oracle.interior(r["U"], lev.g), dt, sm, r["counters"]


def random_mhd_level(n=8, npatch=3, seed=11, bamp=0.4):
    """Self-periodic random MHD patches (same recipe as config 2 plus a random B and psi)."""
    gamma = 5.0 / 3.0
    rng = np.random.default_rng([wk.SEED, 99, seed])
    U = np.empty((9, npatch, n, n, n))
    for p in range(npatch):
        g = rng.standard_normal((8, n, n, n))
        rho = np.exp(0.3 * g[0])
        v = 0.5 * g[1:4]
        B = bamp * g[4:7]
        U[:, p] = wk.primitive_to_conserved(rho, v, np.ones_like(rho), gamma, B=B)
        U[8, p] = 0.05 * g[7]
    lev = wk.Level(n=n, g=3, level=0, dx=1.0 / n, origin=np.zeros((npatch, 3), np.int32),
                   domain_cells=(n, n, n), bc=(0,) * 6, self_periodic=True, U=U)
    return lev, wk.Workload("random_mhd", [lev], gamma, True, LIM_MC, RS_HLLD, 0.3, 1)


# ---------------------------------------------------------------- P4 uniform state
@pytest.mark.parametrize("mhd", [False, True])
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_uniform_state_is_preserved_bitwise(oracle, mhd, dtype):
    n = 8
    one = np.ones((n, n, n))
    v = (0.3 * one, -0.7 * one, 0.45 * one)
    B = (0.2 * one, 0.5 * one, -0.3 * one) if mhd else None
    U = wk.primitive_to_conserved(1.3 * one, v, 0.8 * one, 5.0 / 3.0, B=B)[:, None]
    lev = wk.Level(n=n, g=3, level=0, dx=1.0 / n, origin=np.zeros((1, 3), np.int32), domain_cells=(n, n, n),
                   bc=(1, 1, 0, 0, 1, 1), self_periodic=False, U=np.ascontiguousarray(U))
    wl = wk.Workload("uniform", [lev], 5.0 / 3.0, mhd, LIM_MC, RS_HLLD if mhd else RS_HLLC, 0.3, 1)
    for rs in ((RS_HLL, RS_HLLD) if mhd else (RS_HLL, RS_HLLC)):
        out, dt, sm, _ = one_step(oracle, lev, wl, dtype=dtype, riemann=rs)
        assert np.array_equal(out, lev.U.astype(dtype))
    if mhd:  # uniform psi0 != 0: only psi changes, to psi0 exp(-alpha ch dt/dx)
        lev.U[8] = 0.25
        out, dt, sm, _ = one_step(oracle, lev, wl, dtype=dtype)
        assert np.array_equal(out[:8], lev.U[:8].astype(dtype))
        expect = dtype(0.25) * dtype(np.exp(-wl.alpha * sm * dt / lev.dx))
        assert np.allclose(out[8], expect, rtol=4e-7 if dtype == np.float32 else 1e-15, atol=0)


# ---------------------------------------------------------------- P5 conservation
def test_conservation_hydro_periodic_patches(oracle):
    wl = wk.config2_random_patches(npatch=6, n=16)
    lev = wl.levels[0]
    out, dt, sm, cnt = one_step(oracle, lev, wl)
    for p in range(lev.npatch):
        for f in range(5):
            a, b = lev.U[f, p].sum(), out[f, p].sum()
            assert abs(a - b) <= 1e-13 * np.abs(lev.U[f, p]).sum()
    assert np.abs(out - lev.U).max() > 1e-3          # the step did something


def test_conservation_mhd_periodic_grid(oracle):
    wl = wk.config3_orszag_tang(N=32, n=16)
    lev = wl.levels[0]
    r = oracle.advance(lev, wl, 3)
    for f in range(8):                                   # psi (8) is not conserved
        assert abs(r["U"][f].sum() - lev.U[f].sum()) <= 1e-13 * max(np.abs(lev.U[f]).sum(), 1.0)


# ---------------------------------------------------------------- P6 symmetry
def permute_level(lev, perm):
    """New physical axis d' = old axis perm[d'] (axes numbered x=0,y=1,z=2)."""
    U = lev.U
    nf = U.shape[0]
    ax = [2 + (2 - perm[2 - a]) for a in range(3)]        # array axes (k,j,i) of the new array
    V = np.transpose(U, (0, 1) + tuple(ax))
    out = V.copy()
    for d in range(3):
        out[1 + d] = V[1 + perm[d]]
        if nf == 9:
            out[5 + d] = V[5 + perm[d]]
    return np.ascontiguousarray(out)


@pytest.mark.parametrize("mhd", [False, True])
@pytest.mark.parametrize("perm", [(1, 2, 0), (2, 0, 1), (1, 0, 2)])
def test_permutation_symmetry(oracle, mhd, perm):
    if mhd:
        lev, wl = random_mhd_level()
    else:
        wl = wk.config2_random_patches(npatch=2, n=8)
        lev = wl.levels[0]
    out, dt, sm, _ = one_step(oracle, lev, wl)
    lev2 = wk.Level(**{**lev.__dict__, "U": permute_level(lev, perm)})
    out2, dt2, sm2, _ = one_step(oracle, lev2, wl, dt=dt, ch=sm)
    assert sm2 == pytest.approx(sm, rel=1e-15)
    ref = permute_level(wk.Level(**{**lev.__dict__, "U": out}), perm)
    scale = np.abs(ref).max(axis=(1, 2, 3, 4), keepdims=True)
    assert (np.abs(out2 - ref) / scale).max() < 1e-13


@pytest.mark.parametrize("mhd", [False, True])
def test_mirror_symmetry(oracle, mhd):
    """x -> -x with v_x (and B_x, as a true vector) flipped; psi is a scalar."""
    if mhd:
        lev, wl = random_mhd_level(seed=12)
    else:
        wl = wk.config2_random_patches(npatch=2, n=8)
        lev = wl.levels[0]

    def mirror(U):
        V = U[..., ::-1].copy()
        V[1] *= -1
        if U.shape[0] == 9:
            V[5] *= -1
        return np.ascontiguousarray(V)
    out, dt, sm, _ = one_step(oracle, lev, wl)
    lev2 = wk.Level(**{**lev.__dict__, "U": mirror(lev.U)})
    out2, _, _, _ = one_step(oracle, lev2, wl, dt=dt, ch=sm)
    ref = mirror(out)
    scale = np.abs(ref).max(axis=(1, 2, 3, 4), keepdims=True)
    assert (np.abs(out2 - ref) / scale).max() < 1e-13


# ---------------------------------------------------------------- P8 mhd(B=0) == hydro
@pytest.mark.parametrize("rs_pair", [(RS_HLLC, RS_HLLD), (RS_HLL, RS_HLL)])
def test_mhd_step_without_field_equals_hydro_step(oracle, rs_pair):
    wl = wk.config2_random_patches(npatch=2, n=8)
    lev = wl.levels[0]
    out_h, dt, sm, _ = one_step(oracle, lev, wl, riemann=rs_pair[0])
    U9 = np.concatenate([lev.U, np.zeros((4,) + lev.U.shape[1:])])
    lev9 = wk.Level(**{**lev.__dict__, "U": U9})
    out_m, _, _, _ = one_step(oracle, lev9, wl, riemann=rs_pair[1], dt=dt, ch=sm, alpha=0.4)
    assert np.all(out_m[5:] == 0)
    scale = np.abs(out_h).max(axis=(1, 2, 3, 4), keepdims=True)
    assert (np.abs(out_m[:5] - out_h) / scale).max() < 1e-13


# ---------------------------------------------------------------- P9 extruded Orszag-Tang
def test_extruded_orszag_tang_is_z_invariant(oracle):
    wl = wk.config3_orszag_tang(N=32, n=16, eps=0.0)
    lev = wl.levels[0]
    r = oracle.advance(lev, wl, 3)
    G = wk.configs.join_patches(r["U"], lev.origin, (32, 32, 32))
    for f in range(9):
        assert np.array_equal(G[f], np.broadcast_to(G[f, 0:1], G[f].shape)), f
    assert np.all(G[3] == 0) and np.all(G[7] == 0)
    assert np.abs(G[8]).max() > 0                         # psi picked up the discretisation's div B


# ---------------------------------------------------------------- P15 CFL closed form
@pytest.mark.parametrize("mhd", [False, True])
def test_cfl_closed_form(oracle, mhd):
    n = 8
    one = np.ones((n, n, n))
    gamma, rho, p = 5.0 / 3.0, 1.7, 0.9
    v = (0.3, -1.1, 0.45)
    B = (0.2, 0.5, -0.3)
    U = wk.primitive_to_conserved(rho * one, [c * one for c in v], p * one, gamma,
                                  B=[c * one for c in B] if mhd else None)[:, None]
    Ug = oracle.ghosted(np.ascontiguousarray(U), 3)
    sm = oracle.smax(Ug, 3, gamma)
    if not mhd:
        expect = max(abs(c) for c in v) + np.sqrt(gamma * p / rho)
    else:
        B2 = sum(c * c for c in B)
        a = (gamma * p + B2) / rho
        expect = max(abs(v[d]) + np.sqrt(0.5 * (a + np.sqrt(a * a - 4 * gamma * p * B[d] ** 2 / rho ** 2)))
                     for d in range(3))
    assert sm == pytest.approx(expect, rel=1e-14)
    # one extreme cell decides the maximum
    U2 = U.copy()
    U2[1, 0, 2, 3, 4] = rho * 7.0
    U2[4, 0, 2, 3, 4] += 0.5 * rho * (7.0 ** 2 - v[0] ** 2)
    sm2 = oracle.smax(oracle.ghosted(np.ascontiguousarray(U2), 3), 3, gamma)
    assert sm2 > 7.0
    if not mhd:
        assert sm2 == pytest.approx(7.0 + np.sqrt(gamma * p / rho), rel=1e-12)

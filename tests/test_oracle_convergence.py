"""Pins P10, P12: second-order convergence of the oracle on smooth exact
solutions along each axis, and the O3 primitive predictor against Toro's conservative
MUSCL-Hancock predictor (an independent restatement of the same half step)."""
import numpy as np
import pytest

import workloads as wk

LIM_MC = 2


def evolve_to(oracle, wl, t_end):
    lev = wl.levels[0]
    Ug = oracle.ghosted(lev.U, lev.g)
    t = 0.0
    while t < t_end - 1e-14:
        oracle.fill_ghosts(Ug, lev.g, lev.origin, lev.domain_cells, lev.bc, lev.self_periodic)
        sm = oracle.smax(Ug, lev.g, wl.gamma)
        dt = min(wl.cfl * lev.dx / sm, t_end - t)
        Ug = oracle.step(Ug, lev.g, dt, lev.dx, wl.gamma, wl.limiter, wl.riemann, ch=sm, alpha=wl.alpha)["U"]
        t += dt
    return oracle.interior(Ug, lev.g)


@pytest.mark.parametrize("kind,fields", [("density", (0,)), ("alfven", (5, 6, 7, 1, 2, 3))])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_second_order_convergence(oracle, kind, fields, axis):
    """P10: L1 error against the exact translated wave drops by >= 3 per doubling with MC
    (N = 16 -> 32 -> 64), along x, y and z in turn."""
    t_end = 0.2
    errs = []
    for N in (16, 32, 64):
        wl = wk.smooth_wave_patchset(kind, N, axis=axis)
        U = evolve_to(oracle, wl, t_end)
        exact = wk.smooth_wave_patchset(kind, N, axis=axis, t=t_end).levels[0].U
        errs.append(sum(np.mean(np.abs(U[f] - exact[f])) for f in fields))
    assert errs[0] / errs[1] >= 3.0 and errs[1] / errs[2] >= 3.0, errs
    assert errs[2] < 2e-3


def test_alfven_wave_direction(oracle):
    """The v_perp = -B_perp branch of the circularly polarised wave travels towards +axis: the
    numerical solution is closer to the wave shifted by +t than by -t."""
    N, t_end = 32, 0.2
    wl = wk.smooth_wave_patchset("alfven", N, axis=0)
    U = evolve_to(oracle, wl, t_end)
    fwd = wk.smooth_wave_patchset("alfven", N, axis=0, t=t_end).levels[0].U
    bwd = wk.smooth_wave_patchset("alfven", N, axis=0, t=-t_end).levels[0].U
    assert np.abs(U[6] - fwd[6]).mean() < 0.05 * np.abs(U[6] - bwd[6]).mean()


# ------------------------------------------------------------------------------------------
# P12: conservative (Toro) Hancock predictor, written out independently in numpy
# ------------------------------------------------------------------------------------------

def cons_from_prim(W, gamma, mhd):
    r, v, p = W[0], W[1:4], W[4]
    E = p / (gamma - 1) + 0.5 * r * (v ** 2).sum(axis=0)
    out = [r, r * v[0], r * v[1], r * v[2]]
    if mhd:
        B = W[5:8]
        E = E + 0.5 * (B ** 2).sum(axis=0)
        return np.stack(out + [E, B[0], B[1], B[2], W[8]])
    return np.stack(out + [E])


def prim_from_cons(U, gamma, mhd):
    r = U[0]
    v = U[1:4] / r
    e = U[4] - 0.5 * r * (v ** 2).sum(axis=0)
    if mhd:
        e = e - 0.5 * (U[5:8] ** 2).sum(axis=0)
        return np.stack([r, v[0], v[1], v[2], (gamma - 1) * e, U[5], U[6], U[7], U[8]])
    return np.stack([r, v[0], v[1], v[2], (gamma - 1) * e])


def phys_flux(W, d, gamma, mhd, ch):
    """Flux of the conservative (GLM-)MHD / Euler system along axis d, field order of the arena."""
    r, v, p = W[0], W[1:4], W[4]
    U = cons_from_prim(W, gamma, mhd)
    F = np.zeros_like(U)
    if not mhd:
        F[0] = r * v[d]
        for e in range(3):
            F[1 + e] = r * v[d] * v[e] + (p if e == d else 0.0)
        F[4] = (U[4] + p) * v[d]
        return F
    B, psi = W[5:8], W[8]
    pT = p + 0.5 * (B ** 2).sum(axis=0)
    vB = (v * B).sum(axis=0)
    F[0] = r * v[d]
    for e in range(3):
        F[1 + e] = r * v[d] * v[e] - B[d] * B[e] + (pT if e == d else 0.0)
        F[5 + e] = v[d] * B[e] - v[e] * B[d] + (psi if e == d else 0.0)
    F[4] = (U[4] + pT) * v[d] - B[d] * vB
    F[8] = ch * ch * B[d]
    return F


@pytest.mark.parametrize("mhd", [False, True])
def test_predictor_matches_conservative_hancock_to_second_order(oracle, mhd):
    """On smooth 3-D data the oracle's primitive predictor and Toro's conservative one differ by
    O(h^2): the difference in the predicted cell state drops ~4x per doubling."""
    gamma, ch = 5.0 / 3.0, 2.0
    diffs = []
    for N in (8, 16, 32):
        c = (np.arange(N) + 0.5) / N
        Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
        s = lambda a, b, cc: np.sin(2 * np.pi * (a * X + b * Y + cc * Z))
        rho = 1.0 + 0.2 * s(1, 1, 0)
        v = (0.3 * s(0, 1, 1), 0.2 * s(1, 0, 1) + 0.1, -0.25 * s(1, 1, 1))
        p = 1.0 + 0.1 * s(1, 0, 0) * s(0, 1, 0)
        B = (0.3 * s(0, 1, 0) + 0.2, 0.25 * s(1, 0, 1), 0.2 * s(1, 1, 0)) if mhd else None
        U = wk.primitive_to_conserved(rho, v, p, gamma, B=B)
        if mhd:
            U[8] = 0.05 * s(1, 1, 1)
        lev = wk.Level(n=N, g=3, level=0, dx=1.0 / N, origin=np.zeros((1, 3), np.int32),
                       domain_cells=(N, N, N), bc=(0,) * 6, self_periodic=True,
                       U=np.ascontiguousarray(U[:, None]))
        Ug = oracle.ghosted(lev.U, 3)
        oracle.fill_ghosts(Ug, 3, lev.origin, lev.domain_cells, lev.bc, True)
        dt = 0.3 * lev.dx / oracle.smax(Ug, 3, gamma)
        r = oracle.step(Ug, 3, dt, lev.dx, gamma, LIM_MC, 2 if mhd else 1, ch=ch, alpha=0.0,
                        want_face_states=True)
        FS = r["FS"][:, :, :, 0, 3:-3, 3:-3, 3:-3]         # [d, side, field, k, j, i]
        slopes = FS[:, 1] - FS[:, 0]
        Wstar_oracle = 0.5 * (FS[0, 1] + FS[0, 0])
        W = prim_from_cons(lev.U[:, 0], gamma, mhd)
        dU = np.zeros_like(lev.U[:, 0])
        for d in range(3):
            dU -= dt / (2 * lev.dx) * (phys_flux(W + 0.5 * slopes[d], d, gamma, mhd, ch)
                                       - phys_flux(W - 0.5 * slopes[d], d, gamma, mhd, ch))
        Wstar_toro = prim_from_cons(lev.U[:, 0] + dU, gamma, mhd)
        # the three directions must give the same W* in the oracle
        for d in (1, 2):
            assert np.allclose(0.5 * (FS[d, 1] + FS[d, 0]), Wstar_oracle, rtol=0, atol=1e-14)
        diffs.append(np.abs(Wstar_toro - Wstar_oracle).max())
        # and the predictor itself is a first-order-in-dt change, far larger than the discrepancy
        assert np.abs(Wstar_oracle - W).max() > 20 * diffs[-1]
    assert diffs[0] / diffs[1] > 3.0 and diffs[1] / diffs[2] > 3.3, diffs

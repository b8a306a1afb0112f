"""Pin P16: the oracle's array bookkeeping (ghost fill, slope/face-state/flux
indexing, direction rotations, update) against a deliberately naive second routine on a 4^3
self-periodic patch: loop over faces, recompute everything needed for that face from the
conserved data with modulo indexing (no ghost arrays, no stored intermediates).  The single-face
Riemann flux is taken from the oracle's exported solver, which pins P7/P8 cover separately."""
import numpy as np
import pytest

import workloads as wk

N = 4


def prim(U, idx, gamma, mhd):
    i, j, k = (c % N for c in idx)
    u = U[:, k, j, i]
    rho = u[0]
    v = u[1:4] / rho
    e = u[4] - 0.5 * rho * np.dot(v, v)
    if mhd:
        e -= 0.5 * np.dot(u[5:8], u[5:8])
        return np.concatenate([[rho], v, [(gamma - 1) * e], u[5:8], [u[8]]])
    return np.concatenate([[rho], v, [(gamma - 1) * e]])


def mc(a, b):
    if a * b <= 0:
        return 0.0
    return np.sign(a) * min(2 * abs(a), 2 * abs(b), 0.5 * abs(a + b))


def face_states(U, idx, gamma, mhd, s, ch):
    """W^-_d and W^+_d (d = 0..2) of cell idx, straight from SURVEY.md O2-O4."""
    W = prim(U, idx, gamma, mhd)
    nv = W.size
    D = np.zeros((3, nv))
    for d in range(3):
        e = np.zeros(3, int)
        e[d] = 1
        Wm, Wp = prim(U, np.array(idx) - e, gamma, mhd), prim(U, np.array(idx) + e, gamma, mhd)
        for q in range(nv):
            D[d, q] = mc(W[q] - Wm[q], Wp[q] - W[q])
    rho, v, p = W[0], W[1:4], W[4]
    divv = D[0, 1] + D[1, 2] + D[2, 3]
    adv = lambda q: sum(v[d] * D[d, q] for d in range(3))
    Ws = np.zeros(nv)
    Ws[0] = rho - s * (adv(0) + rho * divv)
    if not mhd:
        for e in range(3):
            Ws[1 + e] = v[e] - s * (adv(1 + e) + D[e, 4] / rho)
        Ws[4] = p - s * (adv(4) + gamma * p * divv)
    else:
        B, psi = W[5:8], W[8]
        divB = D[0, 5] + D[1, 6] + D[2, 7]
        Bgrad = lambda q: sum(B[d] * D[d, q] for d in range(3))
        for e in range(3):
            gradPt_e = D[e, 4] + sum(B[c] * D[e, 5 + c] for c in range(3))
            Ws[1 + e] = v[e] - s * (adv(1 + e) + gradPt_e / rho - (Bgrad(5 + e) + B[e] * divB) / rho)
            Ws[5 + e] = B[e] - s * (adv(5 + e) + B[e] * divv - Bgrad(1 + e) - v[e] * divB + D[e, 8])
        Ws[4] = p - s * (adv(4) + gamma * p * divv + (gamma - 1) * (np.dot(v, B) * divB - Bgrad(8)))
        Ws[8] = psi - s * ch * ch * divB
    minus = np.array([Ws - 0.5 * D[d] for d in range(3)])
    plus = np.array([Ws + 0.5 * D[d] for d in range(3)])
    bad = Ws[0] <= 0 or Ws[4] <= 0 or (minus[:, [0, 4]] <= 0).any() or (plus[:, [0, 4]] <= 0).any()
    if bad:
        minus = np.array([W] * 3)
        plus = np.array([W] * 3)
    return minus, plus


def rotate(W, d, mhd):
    t1, t2 = (d + 1) % 3, (d + 2) % 3
    out = [W[0], W[1 + d], W[1 + t1], W[1 + t2], W[4]]
    if mhd:
        out += [W[5 + d], W[5 + t1], W[5 + t2], W[8]]
    return np.array(out)


def unrotate(F, d, mhd):
    t1, t2 = (d + 1) % 3, (d + 2) % 3
    out = np.zeros_like(F)
    out[0], out[4] = F[0], F[4]
    out[1 + d], out[1 + t1], out[1 + t2] = F[1], F[2], F[3]
    if mhd:
        out[5 + d], out[5 + t1], out[5 + t2], out[8] = F[5], F[6], F[7], F[8]
    return out


def naive_step(oracle, U, dt, dx, gamma, mhd, solver, ch, alpha):
    s = dt / (2 * dx)
    out = np.zeros_like(U)
    for k in range(N):
        for j in range(N):
            for i in range(N):
                idx = np.array([i, j, k])
                acc = np.zeros(U.shape[0])
                for d in range(3):
                    e = np.zeros(3, int)
                    e[d] = 1
                    for sign in (+1, -1):       # upper face (+1), lower face (-1)
                        left = idx if sign > 0 else idx - e
                        right = left + e
                        _, plusL = face_states(U, left, gamma, mhd, s, ch)
                        minusR, _ = face_states(U, right, gamma, mhd, s, ch)
                        F, _ = oracle.riemann(rotate(plusL[d], d, mhd), rotate(minusR[d], d, mhd), gamma, solver, ch=ch)
                        acc += sign * unrotate(F, d, mhd)
                out[:, k, j, i] = U[:, k, j, i] - dt / dx * acc
    if mhd:
        out[8] *= np.exp(-alpha * ch * dt / dx)
    return out


@pytest.mark.parametrize("mhd", [False, True])
def test_bruteforce_4cubed(oracle, mhd):
    gamma = 5.0 / 3.0
    rng = np.random.default_rng([wk.SEED, 16, int(mhd)])
    g = rng.standard_normal((8, N, N, N))
    rho = np.exp(0.4 * g[0])
    v = 0.6 * g[1:4]
    p = np.exp(0.2 * g[4] * 0) + 0.3 * np.abs(g[4])
    if mhd:
        U = wk.primitive_to_conserved(rho, v, p, gamma, B=0.5 * g[5:8])
        U[8] = 0.1 * rng.standard_normal((N, N, N))
    else:
        U = wk.primitive_to_conserved(rho, v, p, gamma)
    Ug = oracle.ghosted(np.ascontiguousarray(U[:, None]), 3)
    oracle.fill_ghosts(Ug, 3, np.zeros((1, 3), np.int32), (N, N, N), (0,) * 6, True)
    sm = oracle.smax(Ug, 3, gamma)
    dx = 1.0 / N
    dt = 0.3 * dx / sm
    solver = 2 if mhd else 1
    r = oracle.step(Ug, 3, dt, dx, gamma, 2, solver, ch=sm, alpha=0.4)
    ref = naive_step(oracle, U, dt, dx, gamma, mhd, solver, sm, 0.4)
    got = oracle.interior(r["U"], 3)[:, 0]
    assert np.abs(got - U).max() > 1e-3
    scale = np.abs(ref).max(axis=(1, 2, 3), keepdims=True)
    assert (np.abs(got - ref) / scale).max() < 1e-14

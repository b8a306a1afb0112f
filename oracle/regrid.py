"""CPU oracle of regridding a refinement level between steps ("regridding between steps";
PAPER.md:31 the mesh is "refined ... in space as well as in time", :59 levels are rebuilt and processed in turn).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module; it shares no code with the CUDA path.

Plain numpy, written to be read against the definitions below.  The paper gives no criterion and no transfer
rule (readings):
  * flagging: an aligned (n/2)^3 block of a level's cells is flagged when the maximum of one field over the
    block exceeds a threshold (the rule the workload generator uses for the initial hierarchy, A15);
  * transfer: a patch of the new fine level that existed in the old one (same origin) keeps its data; a new
    patch is filled by the conservative limited linear interpolation of O8 from the coarse level's current
    state: U_f = U_C + sum_d o_d minmod(U_C - U_{C-e_d}, U_{C+e_d} - U_C), o_d = -1/4 (lower child), +1/4
    (upper child) - so the 8 children of a coarse cell average to it and the composite totals do not change.
Which flagged blocks become patches (growth, proper nesting) is geometry policy of the caller
(workloads.select_blocks), not arithmetic.

Pins (tests/test_oracle_regrid.py): children average to the parent; kept patches are bitwise copies; a field
linear in space is reproduced exactly; uniform stays uniform; flags against a hand-made field; composite totals
unchanged by a regrid; at a non-periodic face the stencil sees the clamped cell, not the far side of the domain.
"""
from __future__ import annotations

import numpy as np


def flag_blocks(level, field: int, threshold: float) -> np.ndarray:
    """bool [npatch, 2, 2, 2] (z, y, x halves): max of U[field] over the aligned (n/2)^3 block > threshold."""
    n, h = level.n, level.n // 2
    u = level.U[field].reshape(level.npatch, 2, h, 2, h, 2, h)
    return u.max(axis=(2, 4, 6)) > threshold


def _dense(level, fill=np.nan) -> np.ndarray:
    """The level's interiors laid out on its whole index space [nf, Nz, Ny, Nx]; `fill` where no patch is."""
    n = level.n
    Nx, Ny, Nz = level.domain_cells
    G = np.full((level.nfields, Nz, Ny, Nx), fill, dtype=np.float64)
    for p, (ox, oy, oz) in enumerate(level.origin):
        G[:, oz:oz + n, oy:oy + n, ox:ox + n] = level.U[:, p]
    return G


def minmod(a, b):
    return np.where((a > 0) & (b > 0), np.minimum(a, b), np.where((a < 0) & (b < 0), np.maximum(a, b), 0.0))


def prolong_patch(Gc: np.ndarray, origin_f, n: int, bc=(0,) * 6) -> np.ndarray:
    """The n^3 fine cells of the patch at fine origin `origin_f` from the dense coarse field Gc.  bc = (xlo, xhi, ylo,
    yhi, zlo, zhi) of the level pair, 0 = periodic: a +-1 stencil cell beyond a periodic face is the wrapped cell; beyond
    any other face it is the coarse level's ghost cell there, i.e. the nearest in-domain cell (O0 rule (ii); DESIGN.md
    section 3 "AMR at non-periodic domain faces": never data from the far side of the domain)."""
    nf = Gc.shape[0]
    Nz, Ny, Nx = Gc.shape[1:]
    h = n // 2
    cx = origin_f[0] // 2 + np.arange(h)
    cy = origin_f[1] // 2 + np.arange(h)
    cz = origin_f[2] // 2 + np.arange(h)

    def idx(c, N, lo, hi):
        c = np.asarray(c).copy()
        below, above = c < 0, c >= N
        c[below] = c[below] + N if lo == 0 else 0
        c[above] = c[above] - N if hi == 0 else N - 1
        return c

    def at(dz, dy, dx):
        return Gc[:, idx(cz + dz, Nz, bc[4], bc[5])[:, None, None], idx(cy + dy, Ny, bc[2], bc[3])[None, :, None],
                  idx(cx + dx, Nx, bc[0], bc[1])[None, None, :]]

    U = at(0, 0, 0)
    sx = minmod(U - at(0, 0, -1), at(0, 0, 1) - U)
    sy = minmod(U - at(0, -1, 0), at(0, 1, 0) - U)
    sz = minmod(U - at(-1, 0, 0), at(1, 0, 0) - U)
    out = np.empty((nf, n, n, n))
    for dk in range(2):
        for dj in range(2):
            for di in range(2):
                val = U + (0.25 if di else -0.25) * sx + (0.25 if dj else -0.25) * sy + (0.25 if dk else -0.25) * sz
                out[:, dk::2, dj::2, di::2] = val
    return out


def regrid_fill(coarse, fine_old, origin_new: np.ndarray) -> np.ndarray:
    """Data of the new fine level [nf, np_new, n, n, n]: copy where the old level had the same patch, prolong
    from `coarse` elsewhere.  `fine_old` may be None (a level is born)."""
    n = coarse.n
    Gc = _dense(coarse)
    old = {} if fine_old is None else {tuple(int(v) for v in o): p for p, o in enumerate(fine_old.origin)}
    out = np.empty((coarse.nfields, len(origin_new), n, n, n))
    for p, o in enumerate(origin_new):
        key = tuple(int(v) for v in o)
        if key in old:
            out[:, p] = fine_old.U[:, old[key]]
        else:
            out[:, p] = prolong_patch(Gc, key, n, tuple(coarse.bc))
            assert np.isfinite(out[:, p]).all(), "new patch %d reaches outside the coarse level (not properly nested)" % p
    return out

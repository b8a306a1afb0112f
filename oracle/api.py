"""ctypes binding of the CPU oracle (TEST INFRASTRUCTURE ONLY -- see godunov_oracle.cpp).

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this module.  It never imports the CUDA package.

Arrays are numpy, layout ``U[field, patch, k, j, i]`` WITH ghosts (M = n + 2g per side).
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np

from . import build as _build

_lib = None

CNT_NAMES = ("positivity_fallback_cells", "hll_fallback_faces", "degenerate_D", "nonpositive_rho_after")


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_smax.restype = C.c_double
        _lib.oracle_limited_slope.restype = C.c_double
        _lib.oracle_limited_slope.argtypes = [C.c_double, C.c_double, C.c_int]
    return _lib


def _dt(a: np.ndarray) -> int:
    if a.dtype == np.float64:
        return 1
    if a.dtype == np.float32:
        return 0
    raise TypeError(a.dtype)


def _p(a: Optional[np.ndarray]):
    if a is None:
        return None
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.c_void_p)


def _ip(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


def default_eps(dtype) -> float:
    """HLLD degeneracy threshold (reading A7): 1e-12 in fp64, 1e-6 in fp32."""
    return 1e-12 if np.dtype(dtype) == np.float64 else 1e-6


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(nt: int) -> None:
    """Thread count of the oracle's OpenMP loops over patches (bench.py: 1 core vs all cores)."""
    lib().oracle_set_num_threads(int(nt))


def fill_ghosts(Ug: np.ndarray, g: int, origin, domain_cells, bc, self_periodic: bool) -> np.ndarray:
    """O0 (i)+(ii) in place.  Returns mask[npatch, M, M, M]: 1 = interior or filled, 0 = left for O8."""
    nf, npch, M = Ug.shape[0], Ug.shape[1], Ug.shape[2]
    mask = np.zeros((npch, M, M, M), dtype=np.uint8)
    o, d, b = _ip(origin), _ip(domain_cells), _ip(bc)
    lib().oracle_fill_ghosts(_dt(Ug), _p(Ug), _p(mask), npch, M - 2 * g, g, nf, _p(o), _p(d), _p(b),
                             int(bool(self_periodic)))
    return mask


def step(Ug: np.ndarray, g: int, dt: float, dx: float, gamma: float, limiter: int, riemann: int,
         ch: float = 0.0, alpha: float = 0.0, eps: Optional[float] = None, want_flux: bool = False,
         want_face_states: bool = False):
    """O1..O6 on every patch.  Returns dict(U=ghosted array with updated interiors (ghosts copied
    from the input), counters=..., F=[3, nf, np, M, M, M] or None, FS=[3, 2, nf, np, M, M, M] or None)."""
    nf, npch, M = Ug.shape[0], Ug.shape[1], Ug.shape[2]
    out = Ug.copy()
    F = np.zeros((3,) + Ug.shape, dtype=Ug.dtype) if want_flux else None
    FS = np.zeros((3, 2) + Ug.shape, dtype=Ug.dtype) if want_face_states else None
    cnt = np.zeros(4, dtype=np.int64)
    if eps is None:
        eps = default_eps(Ug.dtype)
    rc = lib().oracle_step(_dt(Ug), _p(Ug), _p(out), _p(F), _p(FS), npch, M - 2 * g, g, nf,
                           C.c_double(dt), C.c_double(dx), C.c_double(gamma), int(limiter), int(riemann),
                           C.c_double(ch), C.c_double(alpha), C.c_double(eps), _p(cnt))
    if rc != 0:
        raise ValueError("oracle_step rejected its arguments")
    return dict(U=out, counters=dict(zip(CNT_NAMES, cnt.tolist())), F=F, FS=FS)


def ppm_parabola(a5) -> tuple:
    """PPM steps P1 + P2 of one cell from its five-point stencil (a_{i-2} .. a_{i+2}): (aL, aR)."""
    a5 = np.ascontiguousarray(a5, dtype=np.float64)
    aL, aR = C.c_double(), C.c_double()
    lib().oracle_ppm_parabola(_p(a5), C.byref(aL), C.byref(aR))
    return float(aL.value), float(aR.value)


def ppm_sweep(Ug: np.ndarray, g: int, d: int, dt: float, dx: float, gamma: float, riemann: int):
    """One PPM sweep (P1..P5) along direction d (0 = x, 1 = y, 2 = z) on every patch; hydro only.  Returns
    dict(U=ghosted array with updated interiors (ghosts copied from the input), counters=...)."""
    nf, npch, M = Ug.shape[0], Ug.shape[1], Ug.shape[2]
    out = Ug.copy()
    cnt = np.zeros(4, dtype=np.int64)
    rc = lib().oracle_ppm_sweep(_dt(Ug), _p(Ug), _p(out), npch, M - 2 * g, g, nf, int(d), C.c_double(dt),
                                C.c_double(dx), C.c_double(gamma), int(riemann), _p(cnt))
    if rc != 0:
        raise ValueError("oracle_ppm_sweep rejected its arguments")
    return dict(U=out, counters=dict(zip(CNT_NAMES, cnt.tolist())))


def smax(Ug: np.ndarray, g: int, gamma: float) -> float:
    """O7: max over interior cells and directions of |v_d| + c_d."""
    nf, npch, M = Ug.shape[0], Ug.shape[1], Ug.shape[2]
    return float(lib().oracle_smax(_dt(Ug), _p(Ug), npch, M - 2 * g, g, nf, C.c_double(gamma)))


def totals(Ug: np.ndarray, g: int) -> np.ndarray:
    nf, npch, M = Ug.shape[0], Ug.shape[1], Ug.shape[2]
    out = np.zeros(nf)
    lib().oracle_totals(_dt(Ug), _p(Ug), npch, M - 2 * g, g, nf, _p(out))
    return out


def riemann(WL, WR, gamma: float, solver: int, ch: float = 1.0, eps: float = 1e-12):
    WL = np.ascontiguousarray(WL, dtype=np.float64)
    WR = np.ascontiguousarray(WR, dtype=np.float64)
    nf = WL.shape[0]
    F = np.zeros(nf)
    cnt = np.zeros(4, dtype=np.int64)
    lib().oracle_riemann(nf, _p(WL), _p(WR), C.c_double(gamma), C.c_double(ch), int(solver),
                         C.c_double(eps), _p(F), _p(cnt))
    return F, dict(zip(CNT_NAMES, cnt.tolist()))


def hlld_states(WL, WR, gamma: float, ch: float, eps: float = 1e-12):
    """HLLD flux plus its intermediate fan: dict(S[5], U[6,7], FL[7], FR[7], ptstar, Bn, path, F[9])."""
    WL = np.ascontiguousarray(WL, dtype=np.float64)
    WR = np.ascontiguousarray(WR, dtype=np.float64)
    F = np.zeros(9)
    out = np.zeros(64)
    lib().oracle_hlld_states(_p(WL), _p(WR), C.c_double(gamma), C.c_double(ch), C.c_double(eps), _p(F), _p(out))
    return dict(S=out[0:5].copy(), U=out[5:47].reshape(6, 7).copy(), FL=out[47:54].copy(),
                FR=out[54:61].copy(), ptstar=out[61], Bn=out[62], path=int(out[63]), F=F)


def limited_slope(a: float, b: float, lim: int) -> float:
    return float(lib().oracle_limited_slope(a, b, lim))


# ----------------------------------------------------------------------------------------------
# drivers (sequencing only; all arithmetic is in the C++ routines above)
# ----------------------------------------------------------------------------------------------

def ghosted(U: np.ndarray, g: int, dtype=np.float64) -> np.ndarray:
    nf, npch, n = U.shape[0], U.shape[1], U.shape[2]
    M = n + 2 * g
    out = np.zeros((nf, npch, M, M, M), dtype=dtype)
    out[:, :, g:g + n, g:g + n, g:g + n] = U.astype(dtype)
    return out


def interior(Ug: np.ndarray, g: int) -> np.ndarray:
    M = Ug.shape[2]
    return np.ascontiguousarray(Ug[:, :, g:M - g, g:M - g, g:M - g])


def advance(level, wl, nsteps: int, dtype=np.float64, dt_fixed: Optional[float] = None,
            limiter: Optional[int] = None, riemann_solver: Optional[int] = None, eps: Optional[float] = None):
    """Single-level evolution exactly as the harness sequences it: every step = O0 ghost fill,
    O7 smax -> dt = cfl dx / smax and c_h = smax, O1..O6.  `level`/`wl` are workloads.Level/Workload
    (read as plain data).  Returns dict(U=final interior, dts=[...], smaxs=[...], counters=[...])."""
    g = level.g
    Ug = ghosted(level.U, g, dtype)
    lim = wl.limiter if limiter is None else limiter
    rs = wl.riemann if riemann_solver is None else riemann_solver
    dts, smaxs, counters = [], [], []
    for _ in range(nsteps):
        fill_ghosts(Ug, g, level.origin, level.domain_cells, level.bc, level.self_periodic)
        sm = smax(Ug, g, wl.gamma)
        dt = dt_fixed if dt_fixed is not None else wl.cfl * level.dx / sm
        r = step(Ug, g, dt, level.dx, wl.gamma, lim, rs, ch=sm, alpha=wl.alpha, eps=eps)
        Ug = r["U"]
        dts.append(dt)
        smaxs.append(sm)
        counters.append(r["counters"])
    return dict(U=interior(Ug, g), dts=dts, smaxs=smaxs, counters=counters)


PPM_ORDERS = ((0, 1, 2), (2, 1, 0))     # sweep order 0: x-y-z, order 1: z-y-x


def ppm_advance(level, wl, nsteps: int, dtype=np.float64, dt_fixed: Optional[float] = None,
                riemann_solver: Optional[int] = None):
    """Single-level PPM evolution as the harness sequences it: every step = O0 ghost fill, O7 smax ->
    dt = cfl dx / smax, then three sweeps in the order x-y-z on even steps and z-y-x on odd steps, the ghost
    cells refilled (O0) before every sweep.  Returns dict(U=final interior, dts, smaxs, counters)."""
    g = level.g
    Ug = ghosted(level.U, g, dtype)
    rs = wl.riemann if riemann_solver is None else riemann_solver
    dts, smaxs, counters = [], [], []
    for step_no in range(nsteps):
        fill_ghosts(Ug, g, level.origin, level.domain_cells, level.bc, level.self_periodic)
        sm = smax(Ug, g, wl.gamma)
        dt = dt_fixed if dt_fixed is not None else wl.cfl * level.dx / sm
        for d in PPM_ORDERS[step_no % 2]:
            fill_ghosts(Ug, g, level.origin, level.domain_cells, level.bc, level.self_periodic)
            r = ppm_sweep(Ug, g, d, dt, level.dx, wl.gamma, rs)
            Ug = r["U"]
            counters.append(r["counters"])
        dts.append(dt)
        smaxs.append(sm)
    return dict(U=interior(Ug, g), dts=dts, smaxs=smaxs, counters=counters)


def _geom_args(level):
    return _ip(level.origin), _ip(level.domain_cells)


def prolong_ghosts(Uf, mask, lf, Ucold, Ucnew, lc, theta: float):
    of, df = _geom_args(lf)
    oc, dc = _geom_args(lc)
    nf, npf, M = Uf.shape[0], Uf.shape[1], Uf.shape[2]
    lib().oracle_prolong_ghosts(_dt(Uf), _p(Uf), _p(mask), npf, lf.n, lf.g, nf, _p(of), _p(df),
                                _p(Ucold), _p(Ucnew), Ucold.shape[1], _p(oc), _p(dc), C.c_double(theta),
                                _p(_ip(lf.bc)))


def restrict(Uf, lf, Uc, lc):
    of, df = _geom_args(lf)
    oc, dc = _geom_args(lc)
    lib().oracle_restrict(_dt(Uf), _p(Uf), Uf.shape[1], lf.n, lf.g, Uf.shape[0], _p(of), _p(df),
                          _p(Uc), Uc.shape[1], _p(oc), _p(dc))


def reflux(Uc, lc, Fc, lf, Ffsum, dt0: float):
    of, df = _geom_args(lf)
    oc, dc = _geom_args(lc)
    lib().oracle_reflux(_dt(Uc), _p(Uc), Uc.shape[1], lc.n, lc.g, Uc.shape[0], _p(oc), _p(dc), _p(Fc),
                        Ffsum.shape[2], _p(of), _p(df), _p(Ffsum), C.c_double(dt0), C.c_double(lc.dx),
                        _p(_ip(lc.bc)))


def composite_totals(Uc, lc, Uf, lf) -> np.ndarray:
    of, df = _geom_args(lf)
    oc, dc = _geom_args(lc)
    out = np.zeros(Uc.shape[0])
    lib().oracle_composite_totals(_dt(Uc), _p(Uc), Uc.shape[1], lc.n, lc.g, Uc.shape[0], _p(oc), _p(dc),
                                  _p(Uf), Uf.shape[1], _p(of), _p(df), C.c_double(lc.dx), _p(out))
    return out


def two_level_step(wl, dtype=np.float64, eps: Optional[float] = None, do_reflux: bool = True):
    """O9: one coarse step with two fine substeps (Berger-Colella order).  Returns dict with the
    final coarse/fine interiors, dt0, smax and the composite totals before/after."""
    lc, lf = wl.levels
    g = lc.g
    Uc = ghosted(lc.U, g, dtype)
    Uf = ghosted(lf.U, g, dtype)
    tot0 = composite_totals(Uc, lc, Uf, lf)
    sm = max(smax(Uc, g, wl.gamma), smax(Uf, g, wl.gamma))                       # (1)
    dt0 = wl.cfl * lc.dx / sm
    fill_ghosts(Uc, g, lc.origin, lc.domain_cells, lc.bc, False)                 # (2)
    rc = step(Uc, g, dt0, lc.dx, wl.gamma, wl.limiter, wl.riemann, ch=sm, alpha=wl.alpha, eps=eps,
              want_flux=True)                                                    # (3)
    Ucnew = rc["U"]
    fill_ghosts(Ucnew, g, lc.origin, lc.domain_cells, lc.bc, False)             # ghosts of U0^{n+1} for theta=1/2
    Ffsum = None
    counters = [rc["counters"]]
    for theta in (0.0, 0.5):                                                     # (4), (5)
        mask = fill_ghosts(Uf, g, lf.origin, lf.domain_cells, lf.bc, False)
        prolong_ghosts(Uf, mask, lf, Uc, Ucnew, lc, theta)
        rf = step(Uf, g, 0.5 * dt0, lf.dx, wl.gamma, wl.limiter, wl.riemann, ch=sm, alpha=wl.alpha,
                  eps=eps, want_flux=True)
        Uf = rf["U"]
        Ffsum = rf["F"] if Ffsum is None else Ffsum + rf["F"]
        counters.append(rf["counters"])
    restrict(Uf, lf, Ucnew, lc)                                                  # (6)
    if do_reflux:
        reflux(Ucnew, lc, rc["F"], lf, Ffsum, dt0)                               # (7)
    tot1 = composite_totals(Ucnew, lc, Uf, lf)
    return dict(Uc=interior(Ucnew, g), Uf=interior(Uf, g), dt0=dt0, smax=sm, totals_before=tot0,
                totals_after=tot1, counters=counters)


def level_totals(U, level) -> np.ndarray:
    """sum over the interiors of one level of U dx^3, per field (fp64)."""
    return totals(U, level.g) * level.dx ** 3


def hierarchy_totals(Us, levels) -> np.ndarray:
    """Composite totals of an L-level hierarchy: every level's cells that no finer level covers.
    composite_totals(c, f) = uncovered(c) + all(f), so the sum telescopes."""
    tot = composite_totals(Us[0], levels[0], Us[1], levels[1])
    for l in range(1, len(levels) - 1):
        tot = tot - level_totals(Us[l], levels[l]) + composite_totals(Us[l], levels[l], Us[l + 1], levels[l + 1])
    return tot


def hierarchy_step(wl, dtype=np.float64, eps: Optional[float] = None, do_reflux: bool = True):
    """one root step of an L-level hierarchy with recursive subcycling (PAPER.md:31
    "the different resolution levels are advanced in time with different time-steps", :59 "once a refinement
    level is completed the solution is corrected ... and the next (coarser) level of refinement is processed").
    O9 applied recursively: advance(l, dt) = step level l by dt; then, if a finer level exists, twice
    { sibling ghosts of l+1, prolong its coarse-fine ghosts from level l's old/new states at theta = 0, 1/2
    (O8), advance(l+1, dt/2) }; restrict l+1 -> l; reflux l with its own fluxes against the time-summed fine
    fluxes.  One dt0 = cfl dx0 / max_l smax_l and one c_h = that maximum for the whole root step; dt_l =
    dt0 / 2^l.  For L = 2 this is two_level_step call for call.  Returns final interiors per level, dt0, smax,
    composite totals before/after, counters in execution order."""
    levels = wl.levels
    L = len(levels)
    g = levels[0].g
    U = [ghosted(lv.U, g, dtype) for lv in levels]
    tot0 = hierarchy_totals(U, levels)
    sm = max(smax(U[l], g, wl.gamma) for l in range(L))
    dt0 = wl.cfl * levels[0].dx / sm
    Uold = [None] * L
    counters = []
    nsteps = [0] * L

    def sibling_ghosts(l):
        lv = levels[l]
        return fill_ghosts(U[l], g, lv.origin, lv.domain_cells, lv.bc, False)

    def advance(l, dt):
        lv = levels[l]
        r = step(U[l], g, dt, lv.dx, wl.gamma, wl.limiter, wl.riemann, ch=sm, alpha=wl.alpha, eps=eps,
                 want_flux=True)
        Uold[l], U[l] = U[l], r["U"]
        counters.append(r["counters"])
        nsteps[l] += 1
        if l + 1 < L:
            sibling_ghosts(l)                       # ghosts of the new level-l state for the theta = 1/2 stencil
            Fsum = None
            for theta in (0.0, 0.5):
                mask = sibling_ghosts(l + 1)
                prolong_ghosts(U[l + 1], mask, levels[l + 1], Uold[l], U[l], lv, theta)
                Ff = advance(l + 1, 0.5 * dt)
                Fsum = Ff if Fsum is None else Fsum + Ff
            restrict(U[l + 1], levels[l + 1], U[l], lv)
            if do_reflux:
                reflux(U[l], lv, r["F"], levels[l + 1], Fsum, dt)
        return r["F"]

    sibling_ghosts(0)
    advance(0, dt0)
    tot1 = hierarchy_totals(U, levels)
    return dict(U=[interior(U[l], g) for l in range(L)], dt0=dt0, smax=sm, totals_before=tot0, totals_after=tot1,
                counters=counters, nsteps=nsteps)

"""Pins P7, P8: the oracle's Riemann solvers against identities that the
mathematics fixes -- consistency, Rankine-Hugoniot closure over the five-wave HLLD fan, the
textbook HLL formula, HLLD(B=0) == HLLC -- plus limiter special cases (O2)."""
import numpy as np
import pytest

RS_HLL, RS_HLLC, RS_HLLD = 0, 1, 2
G = 5.0 / 3.0


def phys_flux_hydro(W, gamma):
    r, u, v, w, p = W
    E = p / (gamma - 1) + 0.5 * r * (u * u + v * v + w * w)
    return np.array([r * u, r * u * u + p, r * u * v, r * u * w, (E + p) * u])


def phys_flux_mhd(W, gamma, ch):
    r, u, v, w, p, bn, b1, b2, psi = W
    B2 = bn * bn + b1 * b1 + b2 * b2
    pT = p + 0.5 * B2
    E = p / (gamma - 1) + 0.5 * r * (u * u + v * v + w * w) + 0.5 * B2
    vB = u * bn + v * b1 + w * b2
    return np.array([r * u, r * u * u + pT - bn * bn, r * u * v - bn * b1, r * u * w - bn * b2,
                     (E + pT) * u - bn * vB, psi, u * b1 - v * bn, u * b2 - w * bn, ch * ch * bn])


def random_hydro_states(rng, nstates, mach=1.0):
    r = np.exp(rng.normal(0, 0.5, nstates))
    p = np.exp(rng.normal(0, 0.5, nstates))
    v = rng.normal(0, mach, (3, nstates))
    return np.stack([r, v[0], v[1], v[2], p], axis=1)


def random_mhd_states(rng, nstates, mach=1.0, bamp=1.0):
    h = random_hydro_states(rng, nstates, mach)
    B = rng.normal(0, bamp, (3, nstates))
    psi = rng.normal(0, 0.1, nstates)
    return np.concatenate([h, B.T, psi[:, None]], axis=1)


def test_consistency_hydro(oracle):
    """F(W, W) = F_phys(W) for HLL and HLLC (to rounding of the star-state algebra)."""
    rng = np.random.default_rng(1)
    for W in random_hydro_states(rng, 200, mach=2.0):
        ref = phys_flux_hydro(W, G)
        for solver in (RS_HLL, RS_HLLC):
            F, _ = oracle.riemann(W, W, G, solver)
            assert np.allclose(F, ref, rtol=0, atol=2e-14 * max(1.0, np.abs(ref).max()))


def test_consistency_mhd(oracle):
    rng = np.random.default_rng(2)
    for W in random_mhd_states(rng, 200, mach=2.0):
        ch = 3.0
        ref = phys_flux_mhd(W, G, ch)
        for solver in (RS_HLL, RS_HLLD):
            F, _ = oracle.riemann(W, W, G, solver, ch=ch)
            assert np.allclose(F, ref, rtol=0, atol=5e-14 * max(1.0, np.abs(ref).max())), (solver, F - ref)


def test_hll_is_textbook_formula(oracle):
    """HLL == (SR FL - SL FR + SL SR (UR-UL))/(SR-SL) with the Davis-type bounds of reading A5,
    and the upwind flux when the fan is one-sided."""
    rng = np.random.default_rng(3)
    Ws = random_hydro_states(rng, 400, mach=1.5)
    nsub = 0
    for WL, WR in zip(Ws[::2], Ws[1::2]):
        cL, cR = np.sqrt(G * WL[4] / WL[0]), np.sqrt(G * WR[4] / WR[0])
        SL = min(WL[1], WR[1]) - max(cL, cR)
        SR = max(WL[1], WR[1]) + max(cL, cR)
        FL, FR = phys_flux_hydro(WL, G), phys_flux_hydro(WR, G)

        def cons(W):
            r, u, v, w, p = W
            return np.array([r, r * u, r * v, r * w, p / (G - 1) + 0.5 * r * (u * u + v * v + w * w)])
        if SL >= 0:
            ref = FL
        elif SR <= 0:
            ref = FR
        else:
            nsub += 1
            ref = (SR * FL - SL * FR + SL * SR * (cons(WR) - cons(WL))) / (SR - SL)
        F, _ = oracle.riemann(WL, WR, G, RS_HLL)
        assert np.allclose(F, ref, rtol=1e-13, atol=1e-13)
    assert nsub > 50


def test_supersonic_upwinding(oracle):
    """Both solvers return the pure upwind flux when all waves move one way."""
    W1 = np.array([1.0, 5.0, 0.3, -0.2, 1.0])
    W2 = np.array([0.8, 4.5, 0.1, 0.2, 0.9])
    for solver in (RS_HLL, RS_HLLC):
        F, _ = oracle.riemann(W1, W2, G, solver)
        assert np.array_equal(F, _c_order(phys_flux_hydro(W1, G), F))
        Wm1, Wm2 = W1.copy(), W2.copy()
        Wm1[1] *= -1
        Wm2[1] *= -1
        F, _ = oracle.riemann(Wm1, Wm2, G, solver)
        assert np.allclose(F, phys_flux_hydro(Wm2, G), rtol=1e-15, atol=0)


def _c_order(ref, F):
    # the oracle evaluates rho*u*u + p as (rho*u)*u + p; allow 1 ulp
    assert np.allclose(ref, F, rtol=4e-16, atol=0)
    return F


def test_hllc_contact_is_exact(oracle):
    """An isolated contact (equal u, p; jump in rho and transverse v) is resolved exactly by HLLC:
    F = upwind physical flux of the side the contact moves away from."""
    for u in (0.3, -0.3, 0.0):
        WL = np.array([1.0, u, 0.5, -0.1, 1.0])
        WR = np.array([0.25, u, -0.2, 0.4, 1.0])
        F, _ = oracle.riemann(WL, WR, G, RS_HLLC)
        ref = phys_flux_hydro(WL if u >= 0 else WR, G)
        assert np.allclose(F, ref, rtol=0, atol=1e-14)
        Fh, _ = oracle.riemann(WL, WR, G, RS_HLL)
        assert abs(Fh[0] - ref[0]) > 1e-2  # HLL smears it: the test can tell the solvers apart


def test_rankine_hugoniot_closure_hlld(oracle):
    """Sum of the jumps across the five HLLD waves equals F_R - F_L (7 components), and the
    star-state normal momentum flux equals rho* SM^2 + pT* - Bn^2."""
    rng = np.random.default_rng(4)
    Ws = random_mhd_states(rng, 4000, mach=0.7, bamp=0.7)
    nfull = 0
    worst = 0.0
    for WL, WR in zip(Ws[::2], Ws[1::2]):
        ch = 2.5
        st = oracle.hlld_states(WL, WR, G, ch)
        if st["path"] in (0, 1, 7):
            continue
        S, U = st["S"], st["U"]
        lhs = (S[0] * (U[1] - U[0]) + S[1] * (U[2] - U[1]) + S[2] * (U[3] - U[2])
               + S[3] * (U[4] - U[3]) + S[4] * (U[5] - U[4]))
        rhs = st["FR"] - st["FL"]
        scale = max(1.0, np.abs(st["FL"]).max(), np.abs(st["FR"]).max(), np.abs(S).max() * np.abs(U).max())
        worst = max(worst, np.abs(lhs - rhs).max() / scale)
        # F*_L normal momentum
        FsL = st["FL"] + S[0] * (U[1] - U[0])
        assert abs(FsL[1] - (U[1][0] * S[2] ** 2 + st["ptstar"] - st["Bn"] ** 2)) < 1e-12 * scale
        # mass flux is continuous across the contact S_M
        assert abs(FsL[0] - U[1][0] * S[2]) < 1e-12 * scale
        if st["path"] in (2, 3, 4, 5):
            nfull += 1
    assert nfull > 500
    assert worst < 1e-13, worst


def test_hlld_wave_ordering_and_selection(oracle):
    """The returned flux is the one of the region that contains xi = 0 (selection chain of O5)."""
    rng = np.random.default_rng(5)
    Ws = random_mhd_states(rng, 2000, mach=1.0, bamp=0.5)
    seen = set()
    for WL, WR in zip(Ws[::2], Ws[1::2]):
        st = oracle.hlld_states(WL, WR, G, 2.0)
        S, U, path = st["S"], st["U"], st["path"]
        seen.add(path)
        FsL = st["FL"] + S[0] * (U[1] - U[0])
        FssL = FsL + S[1] * (U[2] - U[1])
        FsR = st["FR"] + S[4] * (U[4] - U[5])
        FssR = FsR + S[3] * (U[3] - U[4])
        pick = {0: st["FL"], 1: st["FR"], 2: FsL, 3: FssL, 4: FssR, 5: FsR, 8: FsL, 9: FsR}
        if path in pick:
            F7 = st["F"][[0, 1, 2, 3, 4, 6, 7]]
            assert np.allclose(F7, pick[path], rtol=1e-13, atol=1e-13)
        if path == 3:
            assert S[1] < 0 <= S[2]
        if path == 4:
            assert S[2] < 0 <= S[3]
    assert {2, 3, 4, 5} <= seen


def test_glm_prestep(oracle):
    """Flux of Bn is psi* and flux of psi is ch^2 Bn* (2x2 upwind GLM system)."""
    rng = np.random.default_rng(6)
    Ws = random_mhd_states(rng, 100)
    for WL, WR in zip(Ws[::2], Ws[1::2]):
        ch = 1.7
        for solver in (RS_HLL, RS_HLLD):
            F, _ = oracle.riemann(WL, WR, G, solver, ch=ch)
            bn = 0.5 * (WL[5] + WR[5]) - (WR[8] - WL[8]) / (2 * ch)
            ps = 0.5 * (WL[8] + WR[8]) - 0.5 * ch * (WR[5] - WL[5])
            assert abs(F[5] - ps) < 1e-15 and abs(F[8] - ch * ch * bn) < 1e-14


def test_hlld_equals_hllc_without_field(oracle):
    """P8: with B = 0, psi = 0 the HLLD flux equals the HLLC flux (<= 1e-13)."""
    rng = np.random.default_rng(7)
    Ws = random_hydro_states(rng, 2000, mach=1.0)
    worst = 0.0
    for WL, WR in zip(Ws[::2], Ws[1::2]):
        Fh, c1 = oracle.riemann(WL, WR, G, RS_HLLC)
        Fm, c2 = oracle.riemann(np.concatenate([WL, np.zeros(4)]), np.concatenate([WR, np.zeros(4)]),
                                G, RS_HLLD, ch=2.0)
        assert c1["hll_fallback_faces"] == c2["hll_fallback_faces"]
        scale = max(1.0, np.abs(Fh).max())
        worst = max(worst, np.abs(Fm[:5] - Fh).max() / scale)
        assert np.all(Fm[5:] == 0)
    assert worst < 1e-13, worst


def test_negative_star_pressure_falls_back_to_hll(oracle):
    """A7: strongly receding states give p* <= 0 -> the HLL flux, counted."""
    WL = np.array([1.0, -10.0, 0.0, 0.0, 0.01])
    WR = np.array([1.0, 10.0, 0.0, 0.0, 0.01])
    Fc, c = oracle.riemann(WL, WR, G, RS_HLLC)
    Fh, _ = oracle.riemann(WL, WR, G, RS_HLL)
    assert c["hll_fallback_faces"] == 1 and np.array_equal(Fc, Fh)
    Fd, c = oracle.riemann(np.concatenate([WL, [0.1, 0.1, 0.0, 0.0]]), np.concatenate([WR, [0.1, 0.1, 0.0, 0.0]]),
                           G, RS_HLLD, ch=1.0)
    Fdh, _ = oracle.riemann(np.concatenate([WL, [0.1, 0.1, 0.0, 0.0]]), np.concatenate([WR, [0.1, 0.1, 0.0, 0.0]]),
                            G, RS_HLL, ch=1.0)
    assert c["hll_fallback_faces"] == 1 and np.array_equal(Fd, Fdh)


@pytest.mark.parametrize("lim", [1, 2])
def test_limiter_special_cases(oracle, lim):
    """O2: zero at extrema, symmetric under sign flip and argument swap, central difference on
    smooth data (MC) / smaller difference (minmod), never steeper than 2x either one-sided slope."""
    f = oracle.limited_slope
    assert f(1.0, -1.0, lim) == 0.0 and f(-2.0, 3.0, lim) == 0.0 and f(0.0, 1.0, lim) == 0.0
    rng = np.random.default_rng(8)
    for a, b in np.abs(rng.normal(size=(200, 2))) + 1e-3:
        s = f(a, b, lim)
        assert s == f(b, a, lim) and f(-a, -b, lim) == -s
        if lim == 1:
            assert s == min(a, b)
        else:
            assert s == min(2 * a, 2 * b, 0.5 * (a + b))
            if max(a, b) <= 3 * min(a, b):
                assert s == 0.5 * (a + b)
    assert f(1.0, 1.0, lim) == 1.0
    assert oracle.limited_slope(1.0, 1.0, 0) == 0.0

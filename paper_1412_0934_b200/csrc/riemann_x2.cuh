// O5 for two faces at a time (packed fp32 pairs, pair_math.cuh): branch-free HLLC (hydro) and GLM + HLLD
// (MHD, Miyoshi & Kusano 2005) with the readings of DESIGN.md §3 (A5 wave speeds, A7 selection chain and
// degeneracies, A8 GLM).  The two faces of a pair generally lie in different regions of the Riemann fan,
// so nothing branches on the region: the side K the interface lies in is picked with selects, the star
// and double-star increments are multiplied by S_K / S*_K or by 0, and the only branches are the rare
// events (HLL fallback when p* <= 0, degenerate D), taken when either half needs them.
//   F = F_K + [fan] S_K (U*_K - U_K) + [double star] S*_K (U**_K - U*_K)
// Everything a masked increment touches is kept finite (the one divisor that can vanish outside the
// fan, S_K - S_M, is replaced by 1 there), so that 0 * increment == 0.
#pragma once
#include "pair_math.cuh"
#include "scalar_math_d.cuh"

namespace amr {
namespace x2 {

enum { X2_RS_HLL = 0, X2_RS_HLLC = 1, X2_RS_HLLD = 2 };
enum { X2_CNT_HLL_FALLBACK = 1, X2_CNT_DEGENERATE_D = 2 };

template <class S>
struct RCT {
  S gamma, igm1, ch2, half_ch, half_ich, eps;
};
using RC2 = RCT<float>;    // packed fp32 pairs (value F2, mask B2)
using RCD = RCT<double>;   // one fp64 value per thread (value double, mask bool)

// (S_R F_L - S_L F_R + S_L S_R (U_R - U_L)) / (S_R - S_L)
template <class V>
__device__ __forceinline__ V hll_mix(V fl, V fr, V ul, V ur, V SL, V SR, V SLSR, V idS) {
  return fma(SLSR, ur - ul, fms(SR, fl, SL * fr)) * idS;
}

// hydro.  W = (rho, u, v, w, p) in the rotated order (n, t1, t2); F for (rho, m_n, m_t1, m_t2, E).
// valid: which halves are real faces (event counting only).
template <int RS, class V, class M, class S>
__device__ __forceinline__ void riemann_hydro2(const V* WL, const V* WR, const RCT<S>& C, V* F, M valid,
                                               int* s_cnt) {
  const V rL = WL[0], uL = WL[1], vL = WL[2], wL = WL[3], pL = WL[4];
  const V rR = WR[0], uR = WR[1], vR = WR[2], wR = WR[3], pR = WR[4];
  // max(c_L, c_R) = sqrt(max(c_L^2, c_R^2)): one square root instead of two (the root is monotone)
  const V cmax = sqrt2(max2((C.gamma * pL) * rcp2(rL), (C.gamma * pR) * rcp2(rR)));
  const V SL = min2(uL, uR) - cmax, SR = max2(uL, uR) + cmax;
  const V EL = fma(pL, C.igm1, (0.5f * rL) * fma(uL, uL, fma(vL, vL, wL * wL)));
  const V ER = fma(pR, C.igm1, (0.5f * rR) * fma(uR, uR, fma(vR, vR, wR * wR)));
  const M fan = lt(SL, 0.f) & gt(SR, 0.f);
  const V mL = rL * (SL - uL), mR = rR * (SR - uR);
  V Ss = 0.f;
  M star = false, need_hll = fan;
  if (RS == X2_RS_HLLC) {
    Ss = (fma(mL, uL, pR - pL) - mR * uR) * rcp2(mL - mR);
    const V ps = fma(mL, Ss - uL, pL);
    star = fan & gt(ps, 0.f);
    need_hll = fan & !star;
  }
  const M left = ge(SL, 0.f) | (star & ge(Ss, 0.f));
  const V rK = sel(left, rL, rR), uK = sel(left, uL, uR), vK = sel(left, vL, vR), wK = sel(left, wL, wR);
  const V pK = sel(left, pL, pR), EK = sel(left, EL, ER);
  const V mnK = rK * uK;
  V f0 = mnK, f1 = fma(mnK, uK, pK), f2 = mnK * vK, f3 = mnK * wK, f4 = (EK + pK) * uK;
  if (RS == X2_RS_HLLC) {
    const V SK = sel(left, SL, SR), mK = sel(left, mL, mR);
    const V cK = sel(star, SK, 0.f);
    const V idS = rcp2(sel(star, SK - Ss, 1.f));
    const V fac = mK * idS;  // rho*_K
    // E*_K = [(S_K-u_K) E_K + (S*-u_K)(m_K S* + p_K)] / (S_K - S*)
    const V Es = fma(SK - uK, EK, (Ss - uK) * fma(mK, Ss, pK)) * idS;
    const V cdr = cK * (fac - rK);
    f0 = f0 + cdr;
    f1 = fma(cK, fms(fac, Ss, mnK), f1);
    f2 = fma(cdr, vK, f2);
    f3 = fma(cdr, wK, f3);
    f4 = fma(cK, Es - EK, f4);
  }
  if (RS == X2_RS_HLL ? any(need_hll) : X2_UNLIKELY(any(need_hll))) {  // HLL: the requested solver, or the fallback for p* <= 0 (A7)
    const V idS = rcp2(SR - SL), SLSR = SL * SR;
    const V mnL = rL * uL, mnR = rR * uR;
    const V h0 = hll_mix(mnL, mnR, rL, rR, SL, SR, SLSR, idS);
    const V h1 = hll_mix(fma(mnL, uL, pL), fma(mnR, uR, pR), mnL, mnR, SL, SR, SLSR, idS);
    const V h2 = hll_mix(mnL * vL, mnR * vR, rL * vL, rR * vR, SL, SR, SLSR, idS);
    const V h3 = hll_mix(mnL * wL, mnR * wR, rL * wL, rR * wR, SL, SR, SLSR, idS);
    const V h4 = hll_mix((EL + pL) * uL, (ER + pR) * uR, EL, ER, SL, SR, SLSR, idS);
    f0 = sel(need_hll, h0, f0); f1 = sel(need_hll, h1, f1); f2 = sel(need_hll, h2, f2);
    f3 = sel(need_hll, h3, f3); f4 = sel(need_hll, h4, f4);
    if (RS == X2_RS_HLLC) {
      const int c = count_true(need_hll & valid);
      if (c) atomicAdd(&s_cnt[X2_CNT_HLL_FALLBACK], c);
    }
  }
  F[0] = f0; F[1] = f1; F[2] = f2; F[3] = f3; F[4] = f4;
}

// MHD: GLM 2x2 upwind pre-step for (B_n, psi), then HLL or HLLD on the 7-component system with
// B_n = B_n* on both sides.  W = (rho,u,v,w,p,Bn,Bt1,Bt2,psi); F for (rho,m_n,m_t1,m_t2,E,Bn,Bt1,Bt2,psi).
template <int RS, class V, class M, class S>
__device__ __forceinline__ void riemann_mhd2(const V* WL, const V* WR, const RCT<S>& C, V* F, M valid,
                                             int* s_cnt) {
  const V Bn = fma(WL[8] - WR[8], C.half_ich, 0.5f * (WL[5] + WR[5]));
  F[5] = fma(WL[5] - WR[5], C.half_ch, 0.5f * (WL[8] + WR[8]));
  F[8] = C.ch2 * Bn;
  const V Bn2 = Bn * Bn;

  const V rL = WL[0], uL = WL[1], vL = WL[2], wL = WL[3], pL = WL[4], b1L = WL[6], b2L = WL[7];
  const V rR = WR[0], uR = WR[1], vR = WR[2], wR = WR[3], pR = WR[4], b1R = WR[6], b2R = WR[7];
  const V B2L = fma(b1L, b1L, fma(b2L, b2L, Bn2)), B2R = fma(b1R, b1R, fma(b2R, b2R, Bn2));
  const V pTL = fma(B2L, 0.5f, pL), pTR = fma(B2R, 0.5f, pR);
  const V EL = fma(fma(rL, fma(uL, uL, fma(vL, vL, wL * wL)), B2L), 0.5f, pL * C.igm1);
  const V ER = fma(fma(rR, fma(uR, uR, fma(vR, vR, wR * wR)), B2R), 0.5f, pR * C.igm1);
  const V vBL = fma(uL, Bn, fma(vL, b1L, wL * b2L)), vBR = fma(uR, Bn, fma(vR, b1R, wR * b2R));
  const V irL = rcp2(rL), irR = rcp2(rR);
  const V gpL = C.gamma * pL, gpR = C.gamma * pR;
  const V aL = (gpL + B2L) * irL, aR = (gpR + B2R) * irR;
  // fast speed along n: c_f^2 = (a + sqrt(max(a^2 - 4 gamma p Bn^2 / rho^2, 0))) / 2
  const V dL = max2(fma((gpL * irL) * (Bn2 * irL), -4.f, aL * aL), 0.f);
  const V dR = max2(fma((gpR * irR) * (Bn2 * irR), -4.f, aR * aR), 0.f);
  // max(c_fL, c_fR) = sqrt(max(c_fL^2, c_fR^2)): one outer square root instead of two (the root is monotone)
  const V cmax = sqrt2(0.5f * max2(aL + sqrt2(dL), aR + sqrt2(dR)));
  const V SL = min2(uL, uR) - cmax, SR = max2(uL, uR) + cmax;
  const M fan = lt(SL, 0.f) & gt(SR, 0.f);

  const V sl = SL - uL, sr = SR - uR;
  const V mL = rL * sl, mR = rR * sr;
  V SM = 0.f, pTs = 0.f;
  M star = false, need_hll = fan;
  if (RS == X2_RS_HLLD) {
    const V iden = rcp2(mR - mL);
    SM = fnma(mL, uL, fma(mR, uR, pTL - pTR)) * iden;
    pTs = fma(mL * mR, uR - uL, fnma(mL, pTR, mR * pTL)) * iden;
    star = fan & gt(pTs, 0.f);
    need_hll = fan & !star;
  }
  const M left = ge(SL, 0.f) | (star & ge(SM, 0.f));
  const V rK = sel(left, rL, rR), uK = sel(left, uL, uR), vK = sel(left, vL, vR), wK = sel(left, wL, wR);
  const V b1K = sel(left, b1L, b1R), b2K = sel(left, b2L, b2R);
  const V pTK = sel(left, pTL, pTR), EK = sel(left, EL, ER), vBK = sel(left, vBL, vBR);
  const V mnK = rK * uK;
  V f0 = mnK;
  V f1 = fma(mnK, uK, pTK - Bn2);
  V f2 = fnma(Bn, b1K, mnK * vK);
  V f3 = fnma(Bn, b2K, mnK * wK);
  V f4 = fnma(Bn, vBK, (EK + pTK) * uK);
  V f6 = fnma(vK, Bn, uK * b1K);
  V f7 = fnma(wK, Bn, uK * b2K);
  if (RS == X2_RS_HLLD) {
    // star-state tangential components on both sides (the ** state needs both)
    V vs[2], ws[2], b1s[2], b2s[2], rs[2], idSM[2];
    M degc = false;
#pragma unroll
    for (int K = 0; K < 2; ++K) {
      const V m = K ? mR : mL, sk = K ? sr : sl, SKk = K ? SR : SL, u = K ? uR : uL;
      const V v = K ? vR : vL, w = K ? wR : wL, b1 = K ? b1R : b1L, b2 = K ? b2R : b2L;
      const V dSM = sel(star, SKk - SM, 1.f);
      idSM[K] = rcp2(dSM);
      rs[K] = m * idSM[K];
      const V msk = m * sk;
      const V D = fms(m, dSM, Bn2);
      const M deg = lt(abs2(D), C.eps * msk);
      degc = degc | (deg & star);
      const V iD = sel(deg, 0.f, rcp2(D));
      const V fv = (Bn * (SM - u)) * iD;
      const V g = sel(deg, 1.f, (msk - Bn2) * iD);
      vs[K] = fnma(b1, fv, v);
      ws[K] = fnma(b2, fv, w);
      b1s[K] = b1 * g;
      b2s[K] = b2 * g;
    }
    if (X2_UNLIKELY(any(degc))) {
      const int c = count_true(degc & valid);
      if (c) atomicAdd(&s_cnt[X2_CNT_DEGENERATE_D], c);
    }
    const V SK = sel(left, SL, SR), skK = sel(left, sl, sr);
    const V rsK = sel(left, rs[0], rs[1]), vsK = sel(left, vs[0], vs[1]), wsK = sel(left, ws[0], ws[1]);
    const V b1sK = sel(left, b1s[0], b1s[1]), b2sK = sel(left, b2s[0], b2s[1]);
    const V idK = sel(left, idSM[0], idSM[1]);
    const V vBsK = fma(SM, Bn, fma(vsK, b1sK, wsK * b2sK));
    const V EsK = fma(Bn, vBK - vBsK, fma(pTs, SM, fms(skK, EK, pTK * uK))) * idK;
    const V cK = sel(star, SK, 0.f);
    f0 = fma(cK, rsK - rK, f0);
    f1 = fma(cK, fms(rsK, SM, mnK), f1);
    f2 = fma(cK, fms(rsK, vsK, rK * vK), f2);
    f3 = fma(cK, fms(rsK, wsK, rK * wK), f3);
    f4 = fma(cK, EsK - EK, f4);
    f6 = fma(cK, b1sK - b1K, f6);
    f7 = fma(cK, b2sK - b2K, f7);
    // rotational waves: S*_K = S_M -+ |Bn| / sqrt(rho*_K); skipped when Bn^2 < eps pT* (A7)
    const V sqL = sqrt2(abs2(rs[0])), sqR = sqrt2(abs2(rs[1]));
    const V sqK = sel(left, sqL, sqR);
    const V sgnK = sel(left, -1.f, 1.f);
    const V SsK = fma(sgnK * abs2(Bn), rcp2(sqK), SM);
    const M rot = !lt(Bn2, C.eps * pTs);
    const M dstar = star & rot & ((left & lt(SsK, 0.f)) | (!left & ge(SsK, 0.f)));
    const V sg = sel(gt(Bn, 0.f), 1.f, -1.f);
    const V iSig = rcp2(sqL + sqR);
    const V sqLR = sqL * sqR;
    const V vss = fma(b1s[1] - b1s[0], sg, fma(sqL, vs[0], sqR * vs[1])) * iSig;
    const V wss = fma(b2s[1] - b2s[0], sg, fma(sqL, ws[0], sqR * ws[1])) * iSig;
    const V b1ss = fma(sqLR * (vs[1] - vs[0]), sg, fma(sqL, b1s[1], sqR * b1s[0])) * iSig;
    const V b2ss = fma(sqLR * (ws[1] - ws[0]), sg, fma(sqL, b2s[1], sqR * b2s[0])) * iSig;
    const V vBss = fma(SM, Bn, fma(vss, b1ss, wss * b2ss));
    // E**_L = E*_L - sqrt(rho*_L)(vB*_L - vB**) sg ;  E**_R = E*_R + sqrt(rho*_R)(vB*_R - vB**) sg
    const V dE = (sgnK * sg) * (sqK * (vBsK - vBss));
    const V cS = sel(dstar, SsK, 0.f);
    const V cSr = cS * rsK;
    f2 = fma(cSr, vss - vsK, f2);
    f3 = fma(cSr, wss - wsK, f3);
    f4 = fma(cS, dE, f4);
    f6 = fma(cS, b1ss - b1sK, f6);
    f7 = fma(cS, b2ss - b2sK, f7);
  }
  if (RS == X2_RS_HLL ? any(need_hll) : X2_UNLIKELY(any(need_hll))) {  // HLL: the requested solver, or the fallback for pT* <= 0 (A7)
    const V idS = rcp2(SR - SL), SLSR = SL * SR;
    const V mnL = rL * uL, mnR = rR * uR;
    const V h0 = hll_mix(mnL, mnR, rL, rR, SL, SR, SLSR, idS);
    const V h1 = hll_mix(fma(mnL, uL, pTL - Bn2), fma(mnR, uR, pTR - Bn2), mnL, mnR, SL, SR, SLSR, idS);
    const V h2 = hll_mix(fnma(Bn, b1L, mnL * vL), fnma(Bn, b1R, mnR * vR), rL * vL, rR * vR, SL, SR, SLSR, idS);
    const V h3 = hll_mix(fnma(Bn, b2L, mnL * wL), fnma(Bn, b2R, mnR * wR), rL * wL, rR * wR, SL, SR, SLSR, idS);
    const V h4 = hll_mix(fnma(Bn, vBL, (EL + pTL) * uL), fnma(Bn, vBR, (ER + pTR) * uR), EL, ER, SL, SR, SLSR, idS);
    const V h6 = hll_mix(fnma(vL, Bn, uL * b1L), fnma(vR, Bn, uR * b1R), b1L, b1R, SL, SR, SLSR, idS);
    const V h7 = hll_mix(fnma(wL, Bn, uL * b2L), fnma(wR, Bn, uR * b2R), b2L, b2R, SL, SR, SLSR, idS);
    f0 = sel(need_hll, h0, f0); f1 = sel(need_hll, h1, f1); f2 = sel(need_hll, h2, f2);
    f3 = sel(need_hll, h3, f3); f4 = sel(need_hll, h4, f4); f6 = sel(need_hll, h6, f6);
    f7 = sel(need_hll, h7, f7);
    if (RS == X2_RS_HLLD) {
      const int c = count_true(need_hll & valid);
      if (c) atomicAdd(&s_cnt[X2_CNT_HLL_FALLBACK], c);
    }
  }
  F[0] = f0; F[1] = f1; F[2] = f2; F[3] = f3; F[4] = f4; F[6] = f6; F[7] = f7;
}

template <int NF, int RS, class V, class M, class S>
__device__ __forceinline__ void riemann2(const V* WL, const V* WR, const RCT<S>& C, V* F, M valid, int* s_cnt) {
  if (NF == 5) riemann_hydro2<RS, V, M, S>(WL, WR, C, F, valid, s_cnt);
  else riemann_mhd2<RS, V, M, S>(WL, WR, C, F, valid, s_cnt);
}

}  // namespace x2
}  // namespace amr

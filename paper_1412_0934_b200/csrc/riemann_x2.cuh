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

namespace amr {
namespace x2 {

enum { X2_RS_HLL = 0, X2_RS_HLLC = 1, X2_RS_HLLD = 2 };
enum { X2_CNT_HLL_FALLBACK = 1, X2_CNT_DEGENERATE_D = 2 };

struct RC2 {
  float gamma, igm1, ch2, half_ch, half_ich, eps;
};

// (S_R F_L - S_L F_R + S_L S_R (U_R - U_L)) / (S_R - S_L)
__device__ __forceinline__ F2 hll_mix(F2 fl, F2 fr, F2 ul, F2 ur, F2 SL, F2 SR, F2 SLSR, F2 idS) {
  return fma(SLSR, ur - ul, fms(SR, fl, SL * fr)) * idS;
}

// hydro.  W = (rho, u, v, w, p) in the rotated order (n, t1, t2); F for (rho, m_n, m_t1, m_t2, E).
// valid: which halves are real faces (event counting only).
template <int RS>
__device__ __forceinline__ void riemann_hydro2(const F2* WL, const F2* WR, const RC2& C, F2* F, B2 valid,
                                               int* s_cnt) {
  const F2 rL = WL[0], uL = WL[1], vL = WL[2], wL = WL[3], pL = WL[4];
  const F2 rR = WR[0], uR = WR[1], vR = WR[2], wR = WR[3], pR = WR[4];
  const F2 cL = sqrt2((C.gamma * pL) * rcp2(rL)), cR = sqrt2((C.gamma * pR) * rcp2(rR));
  const F2 cmax = max2(cL, cR);
  const F2 SL = min2(uL, uR) - cmax, SR = max2(uL, uR) + cmax;
  const F2 EL = fma(pL, C.igm1, (0.5f * rL) * fma(uL, uL, fma(vL, vL, wL * wL)));
  const F2 ER = fma(pR, C.igm1, (0.5f * rR) * fma(uR, uR, fma(vR, vR, wR * wR)));
  const B2 fan = lt(SL, 0.f) & gt(SR, 0.f);
  const F2 mL = rL * (SL - uL), mR = rR * (SR - uR);
  F2 Ss = 0.f;
  B2 star = false, need_hll = fan;
  if (RS == X2_RS_HLLC) {
    Ss = (fma(mL, uL, pR - pL) - mR * uR) * rcp2(mL - mR);
    const F2 ps = fma(mL, Ss - uL, pL);
    star = fan & gt(ps, 0.f);
    need_hll = fan & !star;
  }
  const B2 left = ge(SL, 0.f) | (star & ge(Ss, 0.f));
  const F2 rK = sel(left, rL, rR), uK = sel(left, uL, uR), vK = sel(left, vL, vR), wK = sel(left, wL, wR);
  const F2 pK = sel(left, pL, pR), EK = sel(left, EL, ER);
  const F2 mnK = rK * uK;
  F2 f0 = mnK, f1 = fma(mnK, uK, pK), f2 = mnK * vK, f3 = mnK * wK, f4 = (EK + pK) * uK;
  if (RS == X2_RS_HLLC) {
    const F2 SK = sel(left, SL, SR), mK = sel(left, mL, mR);
    const F2 cK = sel(star, SK, 0.f);
    const F2 idS = rcp2(sel(star, SK - Ss, 1.f));
    const F2 fac = mK * idS;  // rho*_K
    // E*_K = [(S_K-u_K) E_K + (S*-u_K)(m_K S* + p_K)] / (S_K - S*)
    const F2 Es = fma(SK - uK, EK, (Ss - uK) * fma(mK, Ss, pK)) * idS;
    const F2 cdr = cK * (fac - rK);
    f0 = f0 + cdr;
    f1 = fma(cK, fms(fac, Ss, mnK), f1);
    f2 = fma(cdr, vK, f2);
    f3 = fma(cdr, wK, f3);
    f4 = fma(cK, Es - EK, f4);
  }
  if (RS == X2_RS_HLL ? any(need_hll) : X2_UNLIKELY(any(need_hll))) {  // HLL: the requested solver, or the fallback for p* <= 0 (A7)
    const F2 idS = rcp2(SR - SL), SLSR = SL * SR;
    const F2 mnL = rL * uL, mnR = rR * uR;
    const F2 h0 = hll_mix(mnL, mnR, rL, rR, SL, SR, SLSR, idS);
    const F2 h1 = hll_mix(fma(mnL, uL, pL), fma(mnR, uR, pR), mnL, mnR, SL, SR, SLSR, idS);
    const F2 h2 = hll_mix(mnL * vL, mnR * vR, rL * vL, rR * vR, SL, SR, SLSR, idS);
    const F2 h3 = hll_mix(mnL * wL, mnR * wR, rL * wL, rR * wR, SL, SR, SLSR, idS);
    const F2 h4 = hll_mix((EL + pL) * uL, (ER + pR) * uR, EL, ER, SL, SR, SLSR, idS);
    f0 = sel(need_hll, h0, f0); f1 = sel(need_hll, h1, f1); f2 = sel(need_hll, h2, f2);
    f3 = sel(need_hll, h3, f3); f4 = sel(need_hll, h4, f4);
    if (RS == X2_RS_HLLC) {
      const int c = (int)(need_hll.x && valid.x) + (int)(need_hll.y && valid.y);
      if (c) atomicAdd(&s_cnt[X2_CNT_HLL_FALLBACK], c);
    }
  }
  F[0] = f0; F[1] = f1; F[2] = f2; F[3] = f3; F[4] = f4;
}

// MHD: GLM 2x2 upwind pre-step for (B_n, psi), then HLL or HLLD on the 7-component system with
// B_n = B_n* on both sides.  W = (rho,u,v,w,p,Bn,Bt1,Bt2,psi); F for (rho,m_n,m_t1,m_t2,E,Bn,Bt1,Bt2,psi).
template <int RS>
__device__ __forceinline__ void riemann_mhd2(const F2* WL, const F2* WR, const RC2& C, F2* F, B2 valid,
                                             int* s_cnt) {
  const F2 Bn = fma(WL[8] - WR[8], C.half_ich, 0.5f * (WL[5] + WR[5]));
  F[5] = fma(WL[5] - WR[5], C.half_ch, 0.5f * (WL[8] + WR[8]));
  F[8] = C.ch2 * Bn;
  const F2 Bn2 = Bn * Bn;

  const F2 rL = WL[0], uL = WL[1], vL = WL[2], wL = WL[3], pL = WL[4], b1L = WL[6], b2L = WL[7];
  const F2 rR = WR[0], uR = WR[1], vR = WR[2], wR = WR[3], pR = WR[4], b1R = WR[6], b2R = WR[7];
  const F2 B2L = fma(b1L, b1L, fma(b2L, b2L, Bn2)), B2R = fma(b1R, b1R, fma(b2R, b2R, Bn2));
  const F2 pTL = fma(B2L, 0.5f, pL), pTR = fma(B2R, 0.5f, pR);
  const F2 EL = fma(fma(rL, fma(uL, uL, fma(vL, vL, wL * wL)), B2L), 0.5f, pL * C.igm1);
  const F2 ER = fma(fma(rR, fma(uR, uR, fma(vR, vR, wR * wR)), B2R), 0.5f, pR * C.igm1);
  const F2 vBL = fma(uL, Bn, fma(vL, b1L, wL * b2L)), vBR = fma(uR, Bn, fma(vR, b1R, wR * b2R));
  const F2 irL = rcp2(rL), irR = rcp2(rR);
  const F2 gpL = C.gamma * pL, gpR = C.gamma * pR;
  const F2 aL = (gpL + B2L) * irL, aR = (gpR + B2R) * irR;
  // fast speed along n: c_f^2 = (a + sqrt(max(a^2 - 4 gamma p Bn^2 / rho^2, 0))) / 2
  const F2 dL = max2(fma((gpL * irL) * (Bn2 * irL), -4.f, aL * aL), 0.f);
  const F2 dR = max2(fma((gpR * irR) * (Bn2 * irR), -4.f, aR * aR), 0.f);
  const F2 cfL = sqrt2(0.5f * (aL + sqrt2(dL))), cfR = sqrt2(0.5f * (aR + sqrt2(dR)));
  const F2 cmax = max2(cfL, cfR);
  const F2 SL = min2(uL, uR) - cmax, SR = max2(uL, uR) + cmax;
  const B2 fan = lt(SL, 0.f) & gt(SR, 0.f);

  const F2 sl = SL - uL, sr = SR - uR;
  const F2 mL = rL * sl, mR = rR * sr;
  F2 SM = 0.f, pTs = 0.f;
  B2 star = false, need_hll = fan;
  if (RS == X2_RS_HLLD) {
    const F2 iden = rcp2(mR - mL);
    SM = fnma(mL, uL, fma(mR, uR, pTL - pTR)) * iden;
    pTs = fma(mL * mR, uR - uL, fnma(mL, pTR, mR * pTL)) * iden;
    star = fan & gt(pTs, 0.f);
    need_hll = fan & !star;
  }
  const B2 left = ge(SL, 0.f) | (star & ge(SM, 0.f));
  const F2 rK = sel(left, rL, rR), uK = sel(left, uL, uR), vK = sel(left, vL, vR), wK = sel(left, wL, wR);
  const F2 b1K = sel(left, b1L, b1R), b2K = sel(left, b2L, b2R);
  const F2 pTK = sel(left, pTL, pTR), EK = sel(left, EL, ER), vBK = sel(left, vBL, vBR);
  const F2 mnK = rK * uK;
  F2 f0 = mnK;
  F2 f1 = fma(mnK, uK, pTK - Bn2);
  F2 f2 = fnma(Bn, b1K, mnK * vK);
  F2 f3 = fnma(Bn, b2K, mnK * wK);
  F2 f4 = fnma(Bn, vBK, (EK + pTK) * uK);
  F2 f6 = fnma(vK, Bn, uK * b1K);
  F2 f7 = fnma(wK, Bn, uK * b2K);
  if (RS == X2_RS_HLLD) {
    // star-state tangential components on both sides (the ** state needs both)
    F2 vs[2], ws[2], b1s[2], b2s[2], rs[2], idSM[2];
    B2 degc = false;
#pragma unroll
    for (int K = 0; K < 2; ++K) {
      const F2 m = K ? mR : mL, sk = K ? sr : sl, SKk = K ? SR : SL, u = K ? uR : uL;
      const F2 v = K ? vR : vL, w = K ? wR : wL, b1 = K ? b1R : b1L, b2 = K ? b2R : b2L;
      const F2 dSM = sel(star, SKk - SM, 1.f);
      idSM[K] = rcp2(dSM);
      rs[K] = m * idSM[K];
      const F2 msk = m * sk;
      const F2 D = fms(m, dSM, Bn2);
      const B2 deg = lt(abs2(D), C.eps * msk);
      degc = degc | (deg & star);
      const F2 iD = sel(deg, 0.f, rcp2(D));
      const F2 fv = (Bn * (SM - u)) * iD;
      const F2 g = sel(deg, 1.f, (msk - Bn2) * iD);
      vs[K] = fnma(b1, fv, v);
      ws[K] = fnma(b2, fv, w);
      b1s[K] = b1 * g;
      b2s[K] = b2 * g;
    }
    if (X2_UNLIKELY(any(degc))) {
      const int c = (int)(degc.x && valid.x) + (int)(degc.y && valid.y);
      if (c) atomicAdd(&s_cnt[X2_CNT_DEGENERATE_D], c);
    }
    const F2 SK = sel(left, SL, SR), skK = sel(left, sl, sr);
    const F2 rsK = sel(left, rs[0], rs[1]), vsK = sel(left, vs[0], vs[1]), wsK = sel(left, ws[0], ws[1]);
    const F2 b1sK = sel(left, b1s[0], b1s[1]), b2sK = sel(left, b2s[0], b2s[1]);
    const F2 idK = sel(left, idSM[0], idSM[1]);
    const F2 vBsK = fma(SM, Bn, fma(vsK, b1sK, wsK * b2sK));
    const F2 EsK = fma(Bn, vBK - vBsK, fma(pTs, SM, fms(skK, EK, pTK * uK))) * idK;
    const F2 cK = sel(star, SK, 0.f);
    f0 = fma(cK, rsK - rK, f0);
    f1 = fma(cK, fms(rsK, SM, mnK), f1);
    f2 = fma(cK, fms(rsK, vsK, rK * vK), f2);
    f3 = fma(cK, fms(rsK, wsK, rK * wK), f3);
    f4 = fma(cK, EsK - EK, f4);
    f6 = fma(cK, b1sK - b1K, f6);
    f7 = fma(cK, b2sK - b2K, f7);
    // rotational waves: S*_K = S_M -+ |Bn| / sqrt(rho*_K); skipped when Bn^2 < eps pT* (A7)
    const F2 sqL = sqrt2(abs2(rs[0])), sqR = sqrt2(abs2(rs[1]));
    const F2 sqK = sel(left, sqL, sqR);
    const F2 sgnK = sel(left, -1.f, 1.f);
    const F2 SsK = fma(sgnK * abs2(Bn), rcp2(sqK), SM);
    const B2 rot = !lt(Bn2, C.eps * pTs);
    const B2 dstar = star & rot & ((left & lt(SsK, 0.f)) | (!left & ge(SsK, 0.f)));
    const F2 sg = sel(gt(Bn, 0.f), 1.f, -1.f);
    const F2 iSig = rcp2(sqL + sqR);
    const F2 sqLR = sqL * sqR;
    const F2 vss = fma(b1s[1] - b1s[0], sg, fma(sqL, vs[0], sqR * vs[1])) * iSig;
    const F2 wss = fma(b2s[1] - b2s[0], sg, fma(sqL, ws[0], sqR * ws[1])) * iSig;
    const F2 b1ss = fma(sqLR * (vs[1] - vs[0]), sg, fma(sqL, b1s[1], sqR * b1s[0])) * iSig;
    const F2 b2ss = fma(sqLR * (ws[1] - ws[0]), sg, fma(sqL, b2s[1], sqR * b2s[0])) * iSig;
    const F2 vBss = fma(SM, Bn, fma(vss, b1ss, wss * b2ss));
    // E**_L = E*_L - sqrt(rho*_L)(vB*_L - vB**) sg ;  E**_R = E*_R + sqrt(rho*_R)(vB*_R - vB**) sg
    const F2 dE = (sgnK * sg) * (sqK * (vBsK - vBss));
    const F2 cS = sel(dstar, SsK, 0.f);
    const F2 cSr = cS * rsK;
    f2 = fma(cSr, vss - vsK, f2);
    f3 = fma(cSr, wss - wsK, f3);
    f4 = fma(cS, dE, f4);
    f6 = fma(cS, b1ss - b1sK, f6);
    f7 = fma(cS, b2ss - b2sK, f7);
  }
  if (RS == X2_RS_HLL ? any(need_hll) : X2_UNLIKELY(any(need_hll))) {  // HLL: the requested solver, or the fallback for pT* <= 0 (A7)
    const F2 idS = rcp2(SR - SL), SLSR = SL * SR;
    const F2 mnL = rL * uL, mnR = rR * uR;
    const F2 h0 = hll_mix(mnL, mnR, rL, rR, SL, SR, SLSR, idS);
    const F2 h1 = hll_mix(fma(mnL, uL, pTL - Bn2), fma(mnR, uR, pTR - Bn2), mnL, mnR, SL, SR, SLSR, idS);
    const F2 h2 = hll_mix(fnma(Bn, b1L, mnL * vL), fnma(Bn, b1R, mnR * vR), rL * vL, rR * vR, SL, SR, SLSR, idS);
    const F2 h3 = hll_mix(fnma(Bn, b2L, mnL * wL), fnma(Bn, b2R, mnR * wR), rL * wL, rR * wR, SL, SR, SLSR, idS);
    const F2 h4 = hll_mix(fnma(Bn, vBL, (EL + pTL) * uL), fnma(Bn, vBR, (ER + pTR) * uR), EL, ER, SL, SR, SLSR, idS);
    const F2 h6 = hll_mix(fnma(vL, Bn, uL * b1L), fnma(vR, Bn, uR * b1R), b1L, b1R, SL, SR, SLSR, idS);
    const F2 h7 = hll_mix(fnma(wL, Bn, uL * b2L), fnma(wR, Bn, uR * b2R), b2L, b2R, SL, SR, SLSR, idS);
    f0 = sel(need_hll, h0, f0); f1 = sel(need_hll, h1, f1); f2 = sel(need_hll, h2, f2);
    f3 = sel(need_hll, h3, f3); f4 = sel(need_hll, h4, f4); f6 = sel(need_hll, h6, f6);
    f7 = sel(need_hll, h7, f7);
    if (RS == X2_RS_HLLD) {
      const int c = (int)(need_hll.x && valid.x) + (int)(need_hll.y && valid.y);
      if (c) atomicAdd(&s_cnt[X2_CNT_HLL_FALLBACK], c);
    }
  }
  F[0] = f0; F[1] = f1; F[2] = f2; F[3] = f3; F[4] = f4; F[6] = f6; F[7] = f7;
}

template <int NF, int RS>
__device__ __forceinline__ void riemann2(const F2* WL, const F2* WR, const RC2& C, F2* F, B2 valid, int* s_cnt) {
  if (NF == 5) riemann_hydro2<RS>(WL, WR, C, F, valid, s_cnt);
  else riemann_mhd2<RS>(WL, WR, C, F, valid, s_cnt);
}

}  // namespace x2
}  // namespace amr

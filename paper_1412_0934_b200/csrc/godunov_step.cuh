// Fused per-tile Godunov step for sm_100a: halo assembly (O0) -> primitives (O1) -> limited slopes
// (O2) -> MUSCL-Hancock predictor (O3) -> face states (O4) -> Riemann flux (O5) -> conservative
// update (O6) -> max signal speed of the new state (O7), one pass, nothing but U_old read from and
// U_new written to HBM.  Formulas: DESIGN.md §3; PAPER.md:43, 57, 58, 76 name the pieces.
//
// Work decomposition: one CTA owns a TX x TY column of one patch and marches along z
// (2.5-D streaming).  One thread per cell of the tile grown by one layer in x/y (no corners).  Shared
// memory is array-of-structs (all NF components of a cell contiguous, padded to a bank-conflict-free
// stride) so that a cell moves with 128-bit LDS/STS:
//   ring   three planes of primitives on the tile + radius-2 halo; the raw conserved plane k+2 arrives by
//          cp.async (LDGSTS) into the slot plane k-1 vacates and is converted in place by the thread
//          that issued the copies
//   XP/YP  W^+_x / W^+_y of the left / lower neighbour of every x / y face of the current plane
//   FX/FY  the x / y face fluxes of the current plane
// Per plane, two barriers:
//   1  slopes, predictor, positivity; publish W^+_x, W^+_y; keep W^-_x, W^-_y in registers; the z face
//      (left state = this thread's W^+_z of the previous plane) is solved here and the previous plane
//      is updated, stored and its signal speed reduced                                   | barrier
//   2  issue the copies of plane k+2; x and y Riemann problems at this cell's lower faces (the upper
//      ring solves the tile's last face); convert plane k+2 to primitives                | barrier
//   3  (Fx+ - Fx-) + (Fy+ - Fy-) of this plane -> registers; falls through into 1 of the next plane
// Every face flux is computed once per tile by one position-independent routine, so a face shared by
// two tiles/patches gets bitwise the same flux on both sides (conservation to round-off).
//
// fp32 arithmetic uses the SFU approximations (rcp/sqrt/rsqrt .approx.ftz, <= 2 ulp) instead of the
// IEEE sequences (12 issue slots each, measured): DESIGN.md §3 "arithmetic freedom"; fp64 is IEEE.
#pragma once
#include <cstdio>
#include <cuda_runtime.h>
#include <math_constants.h>

#include "amr_internal.hpp"
#include "signal_speed.cuh"

namespace amr {

enum { LIM_NONE = 0, LIM_MINMOD = 1, LIM_MC = 2 };
enum { RS_HLL = 0, RS_HLLC = 1, RS_HLLD = 2 };
enum { CNT_POSITIVITY = 0, CNT_HLL_FALLBACK = 1, CNT_DEGENERATE_D = 2, CNT_NEG_STATE = 3 };

__device__ __forceinline__ float rmin(float a, float b) { return fminf(a, b); }
// fp64: fmin / fmax expand to DSETP + six moves/selects each (NaN-propagation rules); a compare-select is three
// instructions and equal for the finite operands the limiter and the solvers see (profiles/r1c)
__device__ __forceinline__ double rmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ float rmax(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ double rmax(double a, double b) { return a > b ? a : b; }
// three-input min / max: one FMNMX3 on sm_100a for fp32
__device__ __forceinline__ float rmin3(float a, float b, float c) {
  float r;
  asm("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
  return r;
}
__device__ __forceinline__ float rmax3(float a, float b, float c) {
  float r;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
  return r;
}
__device__ __forceinline__ double rmin3(double a, double b, double c) { return rmin(rmin(a, b), c); }
__device__ __forceinline__ double rmax3(double a, double b, double c) { return rmax(rmax(a, b), c); }
__device__ __forceinline__ float rsqrt_(float a) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
  return r;
}
__device__ __forceinline__ double rsqrt_(double a) { return fast_sqrt(a); }
__device__ __forceinline__ double rrcp(double a) { return fast_rcp(a); }
__device__ __forceinline__ float rabs(float a) { return fabsf(a); }
__device__ __forceinline__ double rabs(double a) { return fabs(a); }
__device__ __forceinline__ float rrcp(float a) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
  return r;
}
// 1/sqrt(x) given x and sq = sqrt(x)
__device__ __forceinline__ float rinvsqrt(float x, float) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ double rinvsqrt(double, double sq) { return rrcp(sq); }
template <class T> __device__ __forceinline__ T rinf();
template <> __device__ __forceinline__ float rinf<float>() { return CUDART_INF_F; }
template <> __device__ __forceinline__ double rinf<double>() { return CUDART_INF; }

// O2, as HALF slopes h = Delta/2 (the face states are W* +- h, the predictor uses (dt/dx) h).
// a = W_c - W_{c-1}, b = W_{c+1} - W_c (undivided).  Branch-free forms that return exactly the value of
// the sign-test definition (x = min of the candidates, y = max of them: x > 0 -> x, y < 0 -> y, else 0):
//   minmod: Delta/2 = max(x, min(y, 0)) with candidates a/2, b/2
//   MC    : Delta/2 = max(x, min(y, 0)) with candidates a, b, (a+b)/4
template <class T, int LIM>
__device__ __forceinline__ T half_slope(T a, T b) {
  if (LIM == LIM_NONE) return T(0);
  if constexpr (sizeof(T) == 8) {
    // fp64 has no min/max instruction (a compare-select is DSETP + 2 selects), so the sign-test definition
    // itself is cheaper than the min/max form: smallest magnitude of the candidates, sign of a, zero unless
    // a and b have the same sign (equal sign bits; if either is zero the smallest magnitude is zero anyway)
    const bool same = (__double2hiint(a) ^ __double2hiint(b)) >= 0;
    const double aa = fabs(a), ab = fabs(b);
    double m = aa < ab ? aa : ab;
    if (LIM == LIM_MC) {
      const double aq = fabs(T(0.25) * (a + b));
      m = m < aq ? m : aq;
    } else {
      m = T(0.5) * m;
    }
    return same ? copysign(m, a) : T(0);
  } else {
    if (LIM == LIM_MINMOD) {
      const T ha = T(0.5) * a, hb = T(0.5) * b;
      return rmax(rmin(ha, hb), rmin(rmax(ha, hb), T(0)));
    }
    const T q = T(0.25) * (a + b);
    return rmax(rmin3(a, b, q), rmin(rmax3(a, b, q), T(0)));
  }
}

template <class T>
struct RiemannConst {
  T gamma, igm1, ch2, half_ch, half_ich, eps;
};

// O5, hydro.  W = (rho, u, v, w, p) in the rotated order (n, t1, t2); F for (rho, m_n, m_t1, m_t2, E).
// One-sided evaluation: pick the side K the interface lies in, build F_K, add S_K (U*_K - U_K) when
// the interface is inside the fan.  p* <= 0 falls back to HLL (A7).
template <class T, int RS>
__device__ __forceinline__ void riemann_hydro(const T* WL, const T* WR, const RiemannConst<T>& C, T* F,
                                              int* s_cnt) {
  const T rL = WL[0], uL = WL[1], pL = WL[4];
  const T rR = WR[0], uR = WR[1], pR = WR[4];
  const T cL = rsqrt_(C.gamma * pL * rrcp(rL)), cR = rsqrt_(C.gamma * pR * rrcp(rR));
  const T cmax = rmax(cL, cR);
  const T SL = rmin(uL, uR) - cmax, SR = rmax(uL, uR) + cmax;
  const T EL = pL * C.igm1 + T(0.5) * rL * (uL * uL + WL[2] * WL[2] + WL[3] * WL[3]);
  const T ER = pR * C.igm1 + T(0.5) * rR * (uR * uR + WR[2] * WR[2] + WR[3] * WR[3]);
  const bool fan = (SL < T(0)) && (SR > T(0));
  const T mL = rL * (SL - uL), mR = rR * (SR - uR);
  T Ss = T(0);
  bool star = false;
  if (RS == RS_HLLC) {
    Ss = (pR - pL + mL * uL - mR * uR) * rrcp(mL - mR);
    const T ps = pL + mL * (Ss - uL);
    star = fan;
    if (fan && !(ps > T(0))) {
      star = false;
      atomicAdd(&s_cnt[CNT_HLL_FALLBACK], 1);
    }
  }
  if (fan && !star) {  // HLL (requested, or fallback)
    const T UL[5] = {rL, rL * uL, rL * WL[2], rL * WL[3], EL};
    const T UR[5] = {rR, rR * uR, rR * WR[2], rR * WR[3], ER};
    const T FL[5] = {UL[1], UL[1] * uL + pL, UL[1] * WL[2], UL[1] * WL[3], (EL + pL) * uL};
    const T FR[5] = {UR[1], UR[1] * uR + pR, UR[1] * WR[2], UR[1] * WR[3], (ER + pR) * uR};
    const T idS = rrcp(SR - SL);
#pragma unroll
    for (int q = 0; q < 5; ++q) F[q] = (SR * FL[q] - SL * FR[q] + SL * SR * (UR[q] - UL[q])) * idS;
    return;
  }
  const bool left = (SL >= T(0)) || (star && Ss >= T(0));
  const T rK = left ? rL : rR, uK = left ? uL : uR, vK = left ? WL[2] : WR[2], wK = left ? WL[3] : WR[3];
  const T pK = left ? pL : pR, EK = left ? EL : ER;
  const T mnK = rK * uK;
  F[0] = mnK;
  F[1] = mnK * uK + pK;
  F[2] = mnK * vK;
  F[3] = mnK * wK;
  F[4] = (EK + pK) * uK;
  if (star) {
    const T SK = left ? SL : SR, mK = left ? mL : mR;
    const T idS = rrcp(SK - Ss);
    const T fac = mK * idS;  // rho*_K
    // E*_K = fac (E_K/rho_K + (S*-u_K)(S* + p_K/m_K)) = [(S_K-u_K) E_K + (S*-u_K)(m_K S* + p_K)]/(S_K-S*)
    const T Es = ((SK - uK) * EK + (Ss - uK) * (mK * Ss + pK)) * idS;
    F[0] += SK * (fac - rK);
    F[1] += SK * (fac * Ss - mnK);
    F[2] += SK * (fac * vK - rK * vK);
    F[3] += SK * (fac * wK - rK * wK);
    F[4] += SK * (Es - EK);
  }
}

// O5, MHD: GLM 2x2 upwind pre-step for (B_n, psi), then HLL or HLLD (Miyoshi & Kusano 2005) on the
// 7-component system with B_n = B_n* on both sides.  W = (rho,u,v,w,p,Bn,Bt1,Bt2,psi);
// F for (rho, m_n, m_t1, m_t2, E, Bn, Bt1, Bt2, psi).
template <class T, int RS>
__device__ __forceinline__ void riemann_mhd(const T* WL, const T* WR, const RiemannConst<T>& C, T* F,
                                            int* s_cnt) {
  const T Bn = T(0.5) * (WL[5] + WR[5]) - (WR[8] - WL[8]) * C.half_ich;
  F[5] = T(0.5) * (WL[8] + WR[8]) - C.half_ch * (WR[5] - WL[5]);
  F[8] = C.ch2 * Bn;
  const T Bn2 = Bn * Bn;

  const T rL = WL[0], uL = WL[1], vL = WL[2], wL = WL[3], pL = WL[4], b1L = WL[6], b2L = WL[7];
  const T rR = WR[0], uR = WR[1], vR = WR[2], wR = WR[3], pR = WR[4], b1R = WR[6], b2R = WR[7];
  const T B2L = Bn2 + b1L * b1L + b2L * b2L, B2R = Bn2 + b1R * b1R + b2R * b2R;
  const T pTL = pL + T(0.5) * B2L, pTR = pR + T(0.5) * B2R;
  const T EL = pL * C.igm1 + T(0.5) * rL * (uL * uL + vL * vL + wL * wL) + T(0.5) * B2L;
  const T ER = pR * C.igm1 + T(0.5) * rR * (uR * uR + vR * vR + wR * wR) + T(0.5) * B2R;
  const T vBL = uL * Bn + vL * b1L + wL * b2L, vBR = uR * Bn + vR * b1R + wR * b2R;
  const T irL = rrcp(rL), irR = rrcp(rR);
  const T aL = (C.gamma * pL + B2L) * irL, aR = (C.gamma * pR + B2R) * irR;
  const T dL = rmax(aL * aL - T(4) * C.gamma * pL * Bn2 * irL * irL, T(0));
  const T dR = rmax(aR * aR - T(4) * C.gamma * pR * Bn2 * irR * irR, T(0));
  const T cfL = rsqrt_(T(0.5) * (aL + rsqrt_(dL))), cfR = rsqrt_(T(0.5) * (aR + rsqrt_(dR)));
  const T cmax = rmax(cfL, cfR);
  const T SL = rmin(uL, uR) - cmax, SR = rmax(uL, uR) + cmax;
  const bool fan = (SL < T(0)) && (SR > T(0));

  const T sl = SL - uL, sr = SR - uR;
  const T mL = rL * sl, mR = rR * sr;
  T SM = T(0), pTs = T(0);
  bool star = false;
  if (RS == RS_HLLD) {
    const T iden = rrcp(mR - mL);
    SM = (mR * uR - mL * uL - pTR + pTL) * iden;
    pTs = (mR * pTL - mL * pTR + mL * mR * (uR - uL)) * iden;
    star = fan;
    if (fan && !(pTs > T(0))) {
      star = false;
      atomicAdd(&s_cnt[CNT_HLL_FALLBACK], 1);
    }
  }
  if (fan && !star) {  // HLL (requested, or fallback)
    const T UL[7] = {rL, rL * uL, rL * vL, rL * wL, EL, b1L, b2L};
    const T UR[7] = {rR, rR * uR, rR * vR, rR * wR, ER, b1R, b2R};
    const T FL[7] = {UL[1], UL[1] * uL + pTL - Bn2, UL[1] * vL - Bn * b1L, UL[1] * wL - Bn * b2L,
                     (EL + pTL) * uL - Bn * vBL, uL * b1L - vL * Bn, uL * b2L - wL * Bn};
    const T FR[7] = {UR[1], UR[1] * uR + pTR - Bn2, UR[1] * vR - Bn * b1R, UR[1] * wR - Bn * b2R,
                     (ER + pTR) * uR - Bn * vBR, uR * b1R - vR * Bn, uR * b2R - wR * Bn};
    const T idS = rrcp(SR - SL);
    T f7[7];
#pragma unroll
    for (int q = 0; q < 7; ++q) f7[q] = (SR * FL[q] - SL * FR[q] + SL * SR * (UR[q] - UL[q])) * idS;
    F[0] = f7[0]; F[1] = f7[1]; F[2] = f7[2]; F[3] = f7[3]; F[4] = f7[4]; F[6] = f7[5]; F[7] = f7[6];
    return;
  }

  const bool left = (SL >= T(0)) || (star && SM >= T(0));
  const T rK = left ? rL : rR, uK = left ? uL : uR, vK = left ? vL : vR, wK = left ? wL : wR;
  const T b1K = left ? b1L : b1R, b2K = left ? b2L : b2R;
  const T pTK = left ? pTL : pTR, EK = left ? EL : ER, vBK = left ? vBL : vBR;
  const T mnK = rK * uK;
  T f0 = mnK;
  T f1 = mnK * uK + pTK - Bn2;
  T f2 = mnK * vK - Bn * b1K;
  T f3 = mnK * wK - Bn * b2K;
  T f4 = (EK + pTK) * uK - Bn * vBK;
  T f6 = uK * b1K - vK * Bn;
  T f7 = uK * b2K - wK * Bn;
  if (star) {
    // star-state tangential components on both sides (the ** state needs both)
    T vs[2], ws[2], b1s[2], b2s[2], rs[2], idSM[2];
#pragma unroll
    for (int K = 0; K < 2; ++K) {
      const T m = K ? mR : mL, sk = K ? sr : sl, SKk = K ? SR : SL, u = K ? uR : uL;
      const T v = K ? vR : vL, w = K ? wR : wL, b1 = K ? b1R : b1L, b2 = K ? b2R : b2L;
      const T dSM = SKk - SM;
      idSM[K] = rrcp(dSM);
      rs[K] = m * idSM[K];
      const T D = m * dSM - Bn2;
      const bool deg = rabs(D) < C.eps * m * sk;
      if (deg) atomicAdd(&s_cnt[CNT_DEGENERATE_D], 1);
      const T iD = deg ? T(0) : rrcp(D);
      const T fv = Bn * (SM - u) * iD;
      const T g = deg ? T(1) : (m * sk - Bn2) * iD;
      vs[K] = v - b1 * fv;
      ws[K] = w - b2 * fv;
      b1s[K] = b1 * g;
      b2s[K] = b2 * g;
    }
    const T SK = left ? SL : SR, skK = left ? sl : sr;
    const T rsK = left ? rs[0] : rs[1], vsK = left ? vs[0] : vs[1], wsK = left ? ws[0] : ws[1];
    const T b1sK = left ? b1s[0] : b1s[1], b2sK = left ? b2s[0] : b2s[1];
    const T vBsK = SM * Bn + vsK * b1sK + wsK * b2sK;
    const T EsK = (skK * EK - pTK * uK + pTs * SM + Bn * (vBK - vBsK)) * (left ? idSM[0] : idSM[1]);
    f0 += SK * (rsK - rK);
    f1 += SK * (rsK * SM - mnK);
    f2 += SK * (rsK * vsK - rK * vK);
    f3 += SK * (rsK * wsK - rK * wK);
    f4 += SK * (EsK - EK);
    f6 += SK * (b1sK - b1K);
    f7 += SK * (b2sK - b2K);
    if (!(Bn2 < C.eps * pTs)) {  // rotational waves present
      const T sqL = rsqrt_(rs[0]), sqR = rsqrt_(rs[1]);
      const T aBn = rabs(Bn);
      const T sqK = left ? sqL : sqR;
      const T SsK = SM + (left ? -aBn : aBn) * rinvsqrt(rsK, sqK);
      const bool dstar = left ? (SsK < T(0)) : (SsK >= T(0));
      if (dstar) {
        const T sg = (Bn > T(0)) ? T(1) : T(-1);
        const T iSig = rrcp(sqL + sqR);
        const T vss = (sqL * vs[0] + sqR * vs[1] + (b1s[1] - b1s[0]) * sg) * iSig;
        const T wss = (sqL * ws[0] + sqR * ws[1] + (b2s[1] - b2s[0]) * sg) * iSig;
        const T b1ss = (sqL * b1s[1] + sqR * b1s[0] + sqL * sqR * (vs[1] - vs[0]) * sg) * iSig;
        const T b2ss = (sqL * b2s[1] + sqR * b2s[0] + sqL * sqR * (ws[1] - ws[0]) * sg) * iSig;
        const T vBss = SM * Bn + vss * b1ss + wss * b2ss;
        // E**_L = E*_L - sqrt(rho*_L)(vB*_L - vB**) sg ;  E**_R = E*_R + sqrt(rho*_R)(vB*_R - vB**) sg
        const T EssK = left ? (EsK - sqK * (vBsK - vBss) * sg) : (EsK + sqK * (vBsK - vBss) * sg);
        f2 += SsK * (rsK * vss - rsK * vsK);
        f3 += SsK * (rsK * wss - rsK * wsK);
        f4 += SsK * (EssK - EsK);
        f6 += SsK * (b1ss - b1sK);
        f7 += SsK * (b2ss - b2sK);
      }
    }
  }
  F[0] = f0; F[1] = f1; F[2] = f2; F[3] = f3; F[4] = f4; F[6] = f6; F[7] = f7;
}

template <class T, int NF, int RS>
__device__ __forceinline__ void riemann(const T* WL, const T* WR, const RiemannConst<T>& C, T* F, int* s_cnt) {
  if (NF == 5) riemann_hydro<T, RS>(WL, WR, C, F, s_cnt);
  else riemann_mhd<T, RS>(WL, WR, C, F, s_cnt);
}

template <class T> __device__ __forceinline__ void atomic_max_bits(void* slot, T v);
template <> __device__ __forceinline__ void atomic_max_bits<float>(void* slot, float v) {
  atomicMax(reinterpret_cast<unsigned int*>(slot), __float_as_uint(v));
}
template <> __device__ __forceinline__ void atomic_max_bits<double>(void* slot, double v) {
  atomicMax(reinterpret_cast<unsigned long long*>(slot), (unsigned long long)__double_as_longlong(v));
}

// ---- shared-memory cell records (array of structs) -------------------------------------------------
// FS = record stride in elements: a multiple of the vector width VW, chosen so that the 128-bit (64-bit
// for fp32 hydro) accesses of consecutive lanes to consecutive records touch every bank once per phase:
//   fp32 MHD  9 -> 12 (float4, float4, float)     fp32 hydro 5 -> 6 (float2, float2, float)
//   fp64 MHD  9 -> 10 (4 x double2, double)       fp64 hydro 5 -> 6 (2 x double2, double)
template <class T, int NF>
struct Aos {
  static constexpr int VW = (sizeof(T) == 4 && NF == 9) ? 4 : 2;
  static constexpr int FS = sizeof(T) == 4 ? (NF == 9 ? 12 : 6) : (NF == 9 ? 10 : 6);
};
template <class T, int VW> struct Vec;
template <> struct Vec<float, 4> { using type = float4; };
template <> struct Vec<float, 2> { using type = float2; };
template <> struct Vec<double, 2> { using type = double2; };

template <class T, int NF>
__device__ __forceinline__ void lds_cell(const T* p, T* w) {
  constexpr int VW = Aos<T, NF>::VW;
  using V = typename Vec<T, VW>::type;
#pragma unroll
  for (int q = 0; q + VW <= NF; q += VW) {
    const V v = *reinterpret_cast<const V*>(p + q);
    w[q] = v.x;
    w[q + 1] = v.y;
    if constexpr (VW == 4) { w[q + 2] = v.z; w[q + 3] = v.w; }
  }
#pragma unroll
  for (int q = (NF / VW) * VW; q < NF; ++q) w[q] = p[q];
}
template <class T, int NF>
__device__ __forceinline__ void sts_cell(T* p, const T* w) {
  constexpr int VW = Aos<T, NF>::VW;
  using V = typename Vec<T, VW>::type;
#pragma unroll
  for (int q = 0; q + VW <= NF; q += VW) {
    V v;
    v.x = w[q];
    v.y = w[q + 1];
    if constexpr (VW == 4) { v.z = w[q + 2]; v.w = w[q + 3]; }
    *reinterpret_cast<V*>(p + q) = v;
  }
#pragma unroll
  for (int q = (NF / VW) * VW; q < NF; ++q) p[q] = w[q];
}

// LDGSTS: one element, global -> shared, asynchronously
template <class T>
__device__ __forceinline__ void cp_async_elem(T* smem_dst, const T* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  if constexpr (sizeof(T) == 4) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
  else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <class T, int NF, int TX, int TY>
struct TileGeom {
  static constexpr int FS = Aos<T, NF>::FS;
  static constexpr int RW = TX + 4, RH = TY + 4, RP = RW * RH;   // ring plane (tile + radius-2 halo)
  static constexpr int NXF = (TX + 1) * TY, NYF = TX * (TY + 1);  // x / y faces per plane
  static constexpr int NCELL = TX * TY;
  static constexpr int NBC = NCELL + 2 * TY + 2 * TX;             // cells that need the predictor
  static constexpr int NSLOT = 4;                                 // ring planes: k-1, k, k+1 and k+2 in flight
  static constexpr size_t smem_elems = (size_t)FS * (NSLOT * RP + NXF + NYF) + (size_t)2 * 4 * NCELL;
  static constexpr size_t smem_bytes = smem_elems * sizeof(T);
};

// rotated component order handed to the 1-D Riemann routine: x -> (x,y,z), y -> (y,z,x), z -> (z,x,y)
template <class T, int NF, int D>
__device__ __forceinline__ void rotate_in(const T* w, T* r) {
  constexpr int qn = 1 + D, q1 = 1 + (D + 1) % 3, q2 = 1 + (D + 2) % 3;
  r[0] = w[0]; r[1] = w[qn]; r[2] = w[q1]; r[3] = w[q2]; r[4] = w[4];
  if (NF == 9) { r[5] = w[4 + qn]; r[6] = w[4 + q1]; r[7] = w[4 + q2]; r[8] = w[8]; }
}
template <class T, int NF, int D>
__device__ __forceinline__ void rotate_out(const T* r, T* f) {
  constexpr int qn = 1 + D, q1 = 1 + (D + 1) % 3, q2 = 1 + (D + 2) % 3;
  f[0] = r[0]; f[qn] = r[1]; f[q1] = r[2]; f[q2] = r[3]; f[4] = r[4];
  if (NF == 9) { f[4 + qn] = r[5]; f[4 + q1] = r[6]; f[4 + q2] = r[7]; f[8] = r[8]; }
}

template <class T, int NF, int LIM, int RS, int TX, int TY, int NT, int MAXR>
__global__ void __maxnreg__(MAXR) godunov_step_kernel(const __grid_constant__ StepParams<T> P) {
  using G = TileGeom<T, NF, TX, TY>;
  constexpr int FS = G::FS, RW = G::RW, RP = G::RP, NXF = G::NXF, NYF = G::NYF, NCELL = G::NCELL, NBC = G::NBC;
  constexpr int LC = (RP + NT - 1) / NT;  // ring cells per thread in the plane loader
  static_assert(NT >= NBC, "one thread per predictor cell");
  static_assert(NT % 32 == 0, "whole warps");
  static_assert(LC <= 8, "loader masks");

  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* const ring = reinterpret_cast<T*>(smem_raw);  // [4][RP][FS]   primitives (raw U while in flight)
  T* const XF = ring + G::NSLOT * RP * FS;         // [NXF][FS]     W^+_x of the cell left of the face, then the x flux
  T* const YF = XF + NXF * FS;                     // [NYF][FS]     W^+_y of the cell below the face, then the y flux
  T* const UO = YF + NYF * FS;                     // [2][NCELL][4] (m_x, m_y, m_z, E) of the cell awaiting its update
  __shared__ int s_nbr[27];
  __shared__ int s_cnt[4];
  __shared__ T s_red[NT / 32];

  const int tid = threadIdx.x;
  const int n = P.n;
  int bb = blockIdx.x;
  const int tpp = P.ntx * P.nty * P.ntz;
  const int p = bb / tpp;
  bb -= p * tpp;
  const int tz = bb / (P.ntx * P.nty);
  bb -= tz * (P.ntx * P.nty);
  const int ty = bb / P.ntx, tx = bb - ty * P.ntx;
  const int x0 = tx * TX, y0 = ty * TY, z0 = tz * P.zc, zc = P.zc;

  if (tid < 27) s_nbr[tid] = P.nbr[p * 27 + tid];
  if (tid < 4) s_cnt[tid] = 0;
  __syncthreads();

  const int n2 = n * n;
  const int n3 = n2 * n;                     // host guarantees np * (n+2g)^3 < 2^31
  const size_t fs_int = (size_t)P.np * n3;
  const int M = n + 2 * P.g;
  const int M2 = M * M;
  const size_t fs_halo = (size_t)P.np * M2 * M;

  RiemannConst<T> RC;
  RC.gamma = P.gamma; RC.igm1 = P.igm1; RC.ch2 = P.ch2; RC.half_ch = T(0.5) * P.ch; RC.half_ich = P.half_ich;
  RC.eps = P.eps;

  // ---- plane loader (O0): raw U of plane lz -> ring slot, asynchronously ----------------------------
  // ring cell c = ry*RW + rx  <->  patch-local (lx, ly) = (x0 + rx - 2, y0 + ry - 2); cells outside the
  // stencil footprint (corners) are never touched.  Per z region (below / inside / above the patch) the
  // source of a cell is fixed up to the z term, so its offset is resolved once per region:
  //   goff[l]  element offset of (source patch, z = 0, sy, sx)      hmask  source is the prolongation halo
  //   zmask    the z index is clamped (outflow)
  unsigned lmask = 0;  // bit l: this thread's l-th loader cell exists
#pragma unroll
  for (int l = 0; l < LC; ++l) {
    const int c = tid + l * NT;
    if (c < RP) {
      const int ry = c / RW, rx = c - ry * RW;
      const int hx = rx < 2 ? 2 - rx : (rx >= TX + 2 ? rx - (TX + 1) : 0);
      const int hy = ry < 2 ? 2 - ry : (ry >= TY + 2 ? ry - (TY + 1) : 0);
      if (hx + hy <= 2) lmask |= 1u << l;
    }
  }
  int goff[LC];
  unsigned hmask = 0, zmask = 0;
  int cur_rz = -1;
  auto setup_region = [&](int rz) {
    hmask = 0; zmask = 0;
#pragma unroll
    for (int l = 0; l < LC; ++l) {
      goff[l] = 0;
      if (lmask & (1u << l)) {
        const int c = tid + l * NT;
        const int ry = c / RW, rx = c - ry * RW;
        const int lx = x0 + rx - 2, ly = y0 + ry - 2;
        const int gx = lx < 0 ? 0 : (lx >= n ? 2 : 1), gy = ly < 0 ? 0 : (ly >= n ? 2 : 1);
        const int e = s_nbr[rz * 9 + gy * 3 + gx];
        if (e >= 0) {
          const int sp = e & NBR_PATCH_MASK, md = e >> NBR_MODE_SHIFT;
          const int sx = (gx != 1 && (md & 1)) ? (gx == 0 ? 0 : n - 1) : lx - (gx - 1) * n;
          const int sy = (gy != 1 && (md & 2)) ? (gy == 0 ? 0 : n - 1) : ly - (gy - 1) * n;
          if (rz != 1 && (md & 4)) zmask |= 1u << l;
          goff[l] = sp * n3 + sy * n + sx;
        } else {
          hmask |= 1u << l;
          goff[l] = p * (M2 * M) + (ly + P.g) * M + (lx + P.g);
        }
      }
    }
    cur_rz = rz;
  };
  auto issue_plane = [&](int lz, T* dst) {
    const int rz = lz < 0 ? 0 : (lz >= n ? 2 : 1);
    if (rz != cur_rz) setup_region(rz);
    const int zt_int = (lz - (rz - 1) * n) * n2;
    const int zt_clamp = (rz == 0 ? 0 : n - 1) * n2;
    const int zt_halo = (lz + P.g) * M2;
#pragma unroll
    for (int l = 0; l < LC; ++l) {
      if (lmask & (1u << l)) {
        const bool fh = hmask & (1u << l);
        const int off = goff[l] + (fh ? zt_halo : ((zmask & (1u << l)) ? zt_clamp : zt_int));
        const T* src = (fh ? P.halo : P.Uin) + off;
        const size_t fs = fh ? fs_halo : fs_int;
        T* d = dst + (tid + l * NT) * FS;
#pragma unroll
        for (int q = 0; q < NF; ++q) cp_async_elem<T>(d + q, src + q * fs);
      }
    }
  };
  // O1 in place: conserved -> primitive, each thread on the cells it copied
  auto convert_plane = [&](T* dst) {
#pragma unroll
    for (int l = 0; l < LC; ++l) {
      if (lmask & (1u << l)) {
        T* d = dst + (tid + l * NT) * FS;
        T u[NF];
        lds_cell<T, NF>(d, u);
        const T ir = rrcp(u[0]);
        const T vx = u[1] * ir, vy = u[2] * ir, vz = u[3] * ir;
        T e_int = u[4] - T(0.5) * u[0] * (vx * vx + vy * vy + vz * vz);
        if (NF == 9) e_int -= T(0.5) * (u[5] * u[5] + u[6] * u[6] + u[7] * u[7]);
        u[1] = vx; u[2] = vy; u[3] = vz; u[4] = P.gm1 * e_int;
        sts_cell<T, NF>(d, u);
      }
    }
  };

  // ---- per-thread role: one cell (bi, bj) of the tile grown by one layer, no corners ----------------
  //   [0, NCELL)            interior cell: predictor, lower x/y/z faces, update
  //   + TY, + TX            upper ring (bi = TX | bj = TY): predictor, the tile's last x | y face
  //   + TY, + TX            lower ring (bi = -1 | bj = -1): predictor, publishes W^+_x | W^+_y
  int bi, bj;
  if (tid < NCELL) { bj = tid / TX; bi = tid - bj * TX; }
  else if (tid < NCELL + TY) { bi = TX; bj = tid - NCELL; }
  else if (tid < NCELL + TY + TX) { bi = tid - (NCELL + TY); bj = TY; }
  else if (tid < NCELL + 2 * TY + TX) { bi = -1; bj = tid - (NCELL + TY + TX); }
  else { bi = tid - (NCELL + 2 * TY + TX); bj = -1; }
  const bool interior = tid < NCELL;
  const bool pred = tid < NBC;
  const bool in_x = bi >= 0 && bi < TX, in_y = bj >= 0 && bj < TY;
  const bool pub_x = pred && in_y && bi < TX;     // W^+_x feeds face bi+1 of row bj
  const bool pub_y = pred && in_x && bj < TY;     // W^+_y feeds face bj+1 of column bi
  const bool do_x = pred && in_y && bi >= 0;      // solves x face bi of row bj (interior, or bi = TX)
  const bool do_y = pred && in_x && bj >= 0;      // solves y face bj of column bi
  const int bc = pred ? (bj + 2) * RW + (bi + 2) : 0;
  T* const xfp = XF + (do_x ? bj * (TX + 1) + bi : 0) * FS;   // x face to the left of this cell
  T* const yfp = YF + (do_y ? bj * TX + bi : 0) * FS;         // y face below this cell
  const int cell0 = interior ? p * n3 + (y0 + bj) * n + (x0 + bi) : 0;
  T* const uo = UO + (interior ? tid * 4 : 0);

  T zl[NF];     // W^+_z of the previous plane (left state of the next z face)
  T dU[NF];     // flux sum of the plane whose update is pending: ((Fx+ - Fx-) + (Fy+ - Fy-)) - Fz-
  T wmx[NF];    // W^-_x of the current plane (right state of this cell's lower x face), then its x flux
  T wmy[NF];    // W^-_y, then the y flux
  T smax_loc = T(0);
#pragma unroll
  for (int q = 0; q < NF; ++q) { zl[q] = T(0); dU[q] = T(0); wmx[q] = T(0); wmy[q] = T(0); }

  T* Wm = ring;
  T* Wc = ring + RP * FS;
  T* Wp = ring + 2 * RP * FS;
  T* Wn = ring + 3 * RP * FS;
  issue_plane(z0 - 2, Wm);
  issue_plane(z0 - 1, Wc);
  issue_plane(z0, Wp);
  cp_async_commit();
  issue_plane(z0 + 1, Wn);
  cp_async_commit();
  cp_async_wait_group<1>();
  convert_plane(Wm);
  convert_plane(Wc);
  convert_plane(Wp);
  __syncthreads();

  const int blk = (P.fblk != nullptr) ? P.fblk_of[p] : -1;  // flux-register block of this patch
  // flux blocks: [block][direction][field][3 face planes: index 0, n/2, n along the normal][n^2 in-plane, the
  // lower remaining axis fastest]
  const size_t fsz = (size_t)3 * n2;

  for (int t = 0; t <= zc + 1; ++t) {
    const int kk = z0 - 1 + t;               // plane being predicted
    const bool mid = (t >= 1) && (t <= zc);  // kk is a plane of this tile (x/y fluxes needed)

    // ---- phase 1: slopes, predictor, face states; z face; update of plane kk-1 ---------------------
    if (mid ? pred : interior) {
      T w[NF], hx[NF], hy[NF], hz[NF];
      {
        const T* cc = Wc + bc * FS;
        T a[NF], b[NF];
        lds_cell<T, NF>(cc, w);
        lds_cell<T, NF>(cc - FS, a);
        lds_cell<T, NF>(cc + FS, b);
#pragma unroll
        for (int q = 0; q < NF; ++q) hx[q] = half_slope<T, LIM>(w[q] - a[q], b[q] - w[q]);
        lds_cell<T, NF>(cc - RW * FS, a);
        lds_cell<T, NF>(cc + RW * FS, b);
#pragma unroll
        for (int q = 0; q < NF; ++q) hy[q] = half_slope<T, LIM>(w[q] - a[q], b[q] - w[q]);
        lds_cell<T, NF>(Wm + bc * FS, a);
        lds_cell<T, NF>(Wp + bc * FS, b);
#pragma unroll
        for (int q = 0; q < NF; ++q) hz[q] = half_slope<T, LIM>(w[q] - a[q], b[q] - w[q]);
      }
      // O3 predictor with half slopes: W* = W - (dt/dx) sum_d A_d h_d
      const T s = P.dtdx;
      const T rho = w[0], pr = w[4];
      const T ir = rrcp(rho);
      T ws[NF];
#define ADV(q) (w[1] * hx[q] + w[2] * hy[q] + w[3] * hz[q])
      const T divv = hx[1] + hy[2] + hz[3];
      ws[0] = rho - s * (ADV(0) + rho * divv);
      if (NF == 5) {
        ws[1] = w[1] - s * (ADV(1) + hx[4] * ir);
        ws[2] = w[2] - s * (ADV(2) + hy[4] * ir);
        ws[3] = w[3] - s * (ADV(3) + hz[4] * ir);
        ws[4] = pr - s * (ADV(4) + P.gamma * pr * divv);
      } else {
#define BGRAD(q) (w[5] * hx[q] + w[6] * hy[q] + w[7] * hz[q])
        const T divB = hx[5] + hy[6] + hz[7];
        const T vB = w[1] * w[5] + w[2] * w[6] + w[3] * w[7];
        const T BdBx = w[5] * hx[5] + w[6] * hx[6] + w[7] * hx[7];
        const T BdBy = w[5] * hy[5] + w[6] * hy[6] + w[7] * hy[7];
        const T BdBz = w[5] * hz[5] + w[6] * hz[6] + w[7] * hz[7];
        ws[1] = w[1] - s * (ADV(1) + ((hx[4] + BdBx) - (BGRAD(5) + w[5] * divB)) * ir);
        ws[2] = w[2] - s * (ADV(2) + ((hy[4] + BdBy) - (BGRAD(6) + w[6] * divB)) * ir);
        ws[3] = w[3] - s * (ADV(3) + ((hz[4] + BdBz) - (BGRAD(7) + w[7] * divB)) * ir);
        ws[5] = w[5] - s * (ADV(5) + w[5] * divv - BGRAD(1) - w[1] * divB + hx[8]);
        ws[6] = w[6] - s * (ADV(6) + w[6] * divv - BGRAD(2) - w[2] * divB + hy[8]);
        ws[7] = w[7] - s * (ADV(7) + w[7] * divv - BGRAD(3) - w[3] * divB + hz[8]);
        ws[4] = pr - s * (ADV(4) + P.gamma * pr * divv + P.gm1 * (vB * divB - BGRAD(8)));
        ws[8] = w[8] - s * P.ch2 * divB;
#undef BGRAD
      }
#undef ADV
      // O4 positivity: the smallest/largest of the six face values of rho and p
      const T hr = rmax3(rabs(hx[0]), rabs(hy[0]), rabs(hz[0]));
      const T hp = rmax3(rabs(hx[4]), rabs(hy[4]), rabs(hz[4]));
      const bool ok = (ws[0] - hr > T(0)) && (ws[4] - hp > T(0)) && (ws[0] + hr < rinf<T>()) &&
                      (ws[4] + hp < rinf<T>());
      if (!ok) {
        atomicAdd(&s_cnt[CNT_POSITIVITY], 1);
#pragma unroll
        for (int q = 0; q < NF; ++q) { ws[q] = w[q]; hx[q] = T(0); hy[q] = T(0); hz[q] = T(0); }
      }
      if (mid) {
        T fs_[NF];
        if (pub_x) {
#pragma unroll
          for (int q = 0; q < NF; ++q) fs_[q] = ws[q] + hx[q];
          sts_cell<T, NF>(XF + (bj * (TX + 1) + bi + 1) * FS, fs_);
        }
        if (pub_y) {
#pragma unroll
          for (int q = 0; q < NF; ++q) fs_[q] = ws[q] + hy[q];
          sts_cell<T, NF>(YF + ((bj + 1) * TX + bi) * FS, fs_);
        }
#pragma unroll
        for (int q = 0; q < NF; ++q) { wmx[q] = ws[q] - hx[q]; wmy[q] = ws[q] - hy[q]; }
      }
      if (interior) {
        T wr[NF], zn[NF];
#pragma unroll
        for (int q = 0; q < NF; ++q) { wr[q] = ws[q] - hz[q]; zn[q] = ws[q] + hz[q]; }
        if (t >= 1) {  // z face between planes kk-1 and kk
          T fz[NF];
          {
            T WL[NF], WR[NF], Fr[NF];
            rotate_in<T, NF, 2>(zl, WL);
            rotate_in<T, NF, 2>(wr, WR);
            riemann<T, NF, RS>(WL, WR, RC, Fr, s_cnt);
            rotate_out<T, NF, 2>(Fr, fz);
          }
          // only the face planes a link can read (index 0, n/2, n along the normal) are recorded
          if (blk >= 0 && (t <= zc || z0 + zc == n) && (kk == 0 || kk == (n >> 1) || kk == n)) {
            T* dstF = P.fblk + ((size_t)blk * 3 + 2) * NF * fsz + ((size_t)((kk) == 0 ? 0 : ((kk) == n ? 2 : 1)) * n2 + (size_t)((y0 + bj) * n + (x0 + bi)));
#pragma unroll
            for (int q = 0; q < NF; ++q) atomicAdd(dstF + (size_t)q * fsz, fz[q]);
          }
          if (t >= 2) {  // O6 for plane kk-1, GLM damping, O7 of the new state
            // U_old: rho, B, psi are the ring record of plane kk-1 (conversion leaves them untouched),
            // m and E were staged two iterations ago
            T un[NF];
            const T* om = Wm + bc * FS;
            un[0] = om[0];
            if (NF == 9) { un[5] = om[5]; un[6] = om[6]; un[7] = om[7]; un[8] = om[8]; }
            {
              const T* ou = uo + ((t & 1) ? 4 * NCELL : 0);
              using V = typename Vec<T, Aos<T, 9>::VW>::type;
              if constexpr (sizeof(T) == 4) {
                const V v = *reinterpret_cast<const V*>(ou);
                un[1] = v.x; un[2] = v.y; un[3] = v.z; un[4] = v.w;
              } else {
                const V v0 = *reinterpret_cast<const V*>(ou), v1 = *reinterpret_cast<const V*>(ou + 2);
                un[1] = v0.x; un[2] = v0.y; un[3] = v1.x; un[4] = v1.y;
              }
            }
#pragma unroll
            for (int q = 0; q < NF; ++q) un[q] = un[q] - P.dtdx * (dU[q] + fz[q]);
            if (NF == 9) un[8] *= P.damp;
            T* out = P.Uout + (cell0 + (kk - 1) * n2);
#pragma unroll
            for (int q = 0; q < NF; ++q) out[q * fs_int] = un[q];
            if (!(un[0] > T(0))) atomicAdd(&s_cnt[CNT_NEG_STATE], 1);
            smax_loc = rmax(signal_speed<T, NF>(un, P.gamma, P.gm1), smax_loc);  // a NaN speed is dropped
          }
#pragma unroll
          for (int q = 0; q < NF; ++q) dU[q] = -fz[q];
        }
#pragma unroll
        for (int q = 0; q < NF; ++q) zl[q] = zn[q];
      }
    }
    if (t == zc + 1) break;
    __syncthreads();

    // ---- phase 2: copies of plane kk+3 and of (m, E) of plane kk+1; x / y Riemann problems of plane kk;
    //      convert plane kk+2 (its copies were issued one iteration ago) ---------------------------------
    if (t <= zc - 1) {
      issue_plane(kk + 3, Wm);
      if (interior) {
        const T* src = P.Uin + (cell0 + (kk + 1) * n2);
        T* d = uo + ((t & 1) ? 4 * NCELL : 0);
#pragma unroll
        for (int q = 0; q < 4; ++q) cp_async_elem<T>(d + q, src + (q + 1) * fs_int);
      }
    }
    cp_async_commit();
    if (mid) {
      if (do_x) {
        T wl[NF], WL[NF], WR[NF], Fr[NF];
        lds_cell<T, NF>(xfp, wl);
        rotate_in<T, NF, 0>(wl, WL);
        rotate_in<T, NF, 0>(wmx, WR);
        riemann<T, NF, RS>(WL, WR, RC, Fr, s_cnt);
        rotate_out<T, NF, 0>(Fr, wmx);
        sts_cell<T, NF>(xfp, wmx);
        if (blk >= 0 && (bi < TX || x0 + TX == n) && (x0 + bi == 0 || x0 + bi == (n >> 1) || x0 + bi == n)) {  // record the flux for the reflux
          T* dstF = P.fblk + ((size_t)blk * 3 + 0) * NF * fsz + ((size_t)((x0 + bi) == 0 ? 0 : ((x0 + bi) == n ? 2 : 1)) * n2 + (size_t)(kk * n + (y0 + bj)));
#pragma unroll
          for (int q = 0; q < NF; ++q) atomicAdd(dstF + (size_t)q * fsz, wmx[q]);
        }
      }
      if (do_y) {
        T wl[NF], WL[NF], WR[NF], Fr[NF];
        lds_cell<T, NF>(yfp, wl);
        rotate_in<T, NF, 1>(wl, WL);
        rotate_in<T, NF, 1>(wmy, WR);
        riemann<T, NF, RS>(WL, WR, RC, Fr, s_cnt);
        rotate_out<T, NF, 1>(Fr, wmy);
        sts_cell<T, NF>(yfp, wmy);
        if (blk >= 0 && (bj < TY || y0 + TY == n) && (y0 + bj == 0 || y0 + bj == (n >> 1) || y0 + bj == n)) {
          T* dstF = P.fblk + ((size_t)blk * 3 + 1) * NF * fsz + ((size_t)((y0 + bj) == 0 ? 0 : ((y0 + bj) == n ? 2 : 1)) * n2 + (size_t)(kk * n + (x0 + bi)));
#pragma unroll
          for (int q = 0; q < NF; ++q) atomicAdd(dstF + (size_t)q * fsz, wmy[q]);
        }
      }
    }
    cp_async_wait_group<1>();
    convert_plane(Wn);
    __syncthreads();

    // ---- phase 3: x/y flux differences of plane kk -> registers ------------------------------------
    // (own fluxes are in wmx / wmy; the upper ones are read from the slots this very thread overwrites
    // with its W^+ in the next phase 1, so no barrier is needed before that)
    if (interior && mid) {
      T b[NF], d[NF];
      lds_cell<T, NF>(xfp + FS, b);
      lds_cell<T, NF>(yfp + TX * FS, d);
#pragma unroll
      for (int q = 0; q < NF; ++q) dU[q] = ((b[q] - wmx[q]) + (d[q] - wmy[q])) + dU[q];
    }
    T* tmp = Wm; Wm = Wc; Wc = Wp; Wp = Wn; Wn = tmp;
  }

  // ---- epilogue: max signal speed of the new state (O7), event counters -----------------------
  // NaN-safe: rmax(x, m) keeps m when x is NaN; a NaN state shows up in the NEG_STATE counter instead.
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) smax_loc = rmax(smax_loc, __shfl_xor_sync(0xffffffffu, smax_loc, o));
  if ((tid & 31) == 0) s_red[tid >> 5] = smax_loc;
  __syncthreads();
  if (tid == 0) {
    T m = s_red[0];
#pragma unroll
    for (int wv = 1; wv < NT / 32; ++wv) m = rmax(m, s_red[wv]);
    atomic_max_bits<T>(P.smax, m);
  }
  if (tid < 4 && s_cnt[tid] != 0) atomicAdd(P.counters + tid, (unsigned long long)s_cnt[tid]);
}

// host-side launcher for one (T, NF, TX, TY, NT, MAXR) tile configuration
template <class T, int NF, int LIM, int RS, int TX, int TY, int NT, int MAXR>
cudaError_t launch_variant(const StepParams<T>& P, cudaStream_t s) {
  using G = TileGeom<T, NF, TX, TY>;
  auto kern = godunov_step_kernel<T, NF, LIM, RS, TX, TY, NT, MAXR>;
  static std::atomic<unsigned long long> configured{0};  // per instantiation, one bit per device
  {
    cudaError_t e = ensure_dynamic_smem((const void*)kern, (int)G::smem_bytes, configured);
    if (e != cudaSuccess) return e;
  }
  const long long grid = (long long)P.np_active * P.ntx * P.nty * P.ntz;
  kern<<<(unsigned)grid, NT, G::smem_bytes, s>>>(P);
  cudaError_t le = cudaGetLastError();
  if (le != cudaSuccess) {
    cudaFuncAttributes fa;
    if (cudaFuncGetAttributes(&fa, kern) == cudaSuccess)
      fprintf(stderr, "amr: step kernel launch failed: %d threads, %d regs/thread, %zu B dynamic + %zu B static smem, maxThreadsPerBlock %d\n",
              NT, fa.numRegs, (size_t)G::smem_bytes, fa.sharedSizeBytes, fa.maxThreadsPerBlock);
  }
  return le;
}

template <class T, int NF, int TX, int TY, int NT, int MAXR>
cudaError_t launch_dispatch(const StepParams<T>& P, int limiter, int riemann, cudaStream_t s) {
  constexpr int RSX = (NF == 5) ? RS_HLLC : RS_HLLD;
#define AMR_CASE(L, R) \
  if (limiter == L && riemann == R) return launch_variant<T, NF, L, R, TX, TY, NT, MAXR>(P, s);
  AMR_CASE(LIM_NONE, RS_HLL)
  AMR_CASE(LIM_MINMOD, RS_HLL)
  AMR_CASE(LIM_MC, RS_HLL)
  AMR_CASE(LIM_NONE, RSX)
  AMR_CASE(LIM_MINMOD, RSX)
  AMR_CASE(LIM_MC, RSX)
#undef AMR_CASE
  return cudaErrorInvalidValue;
}

}  // namespace amr

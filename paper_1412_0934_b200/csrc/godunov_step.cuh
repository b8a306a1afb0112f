// Fused per-tile Godunov step for sm_100a: halo assembly (O0) -> primitives (O1) -> limited slopes
// (O2) -> MUSCL-Hancock predictor (O3) -> face states (O4) -> Riemann flux (O5) -> conservative
// update (O6) -> max signal speed of the new state (O7), one pass, nothing but U_old read from and
// U_new written to HBM.  Formulas: DESIGN.md §3; PAPER.md:43, 57, 58, 76 name the pieces.
//
// Work decomposition: one CTA owns a TX x TY column of one patch and marches along z
// (2.5-D streaming).  A ring of three primitive planes (tile + radius-2 halo) lives in shared memory.
// Per plane:  A  load U of plane k+1 through the neighbour table, convert, store to the ring
//             B  one thread per cell of the tile grown by one layer in x/y: slopes, predictor, face
//                states; x/y face states go to shared memory, z face states stay in registers and the
//                z flux is solved here
//             C  one thread per x/y face: Riemann flux -> shared memory
//             D  one thread per interior cell: gather the six fluxes, update, store, signal speed
// Every face flux is computed once per tile by one position-independent routine, so a face shared by
// two tiles/patches gets bitwise the same flux on both sides (conservation to round-off).
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>

#include "amr_internal.hpp"
#include "signal_speed.cuh"

namespace amr {

enum { LIM_NONE = 0, LIM_MINMOD = 1, LIM_MC = 2 };
enum { RS_HLL = 0, RS_HLLC = 1, RS_HLLD = 2 };
enum { CNT_POSITIVITY = 0, CNT_HLL_FALLBACK = 1, CNT_DEGENERATE_D = 2, CNT_NEG_STATE = 3 };

template <class T> __device__ __forceinline__ T rmin(T a, T b) { return a < b ? a : b; }
template <> __device__ __forceinline__ float rmin<float>(float a, float b) { return fminf(a, b); }
template <> __device__ __forceinline__ double rmin<double>(double a, double b) { return fmin(a, b); }
template <class T> __device__ __forceinline__ T rmax(T a, T b) { return a > b ? a : b; }
template <> __device__ __forceinline__ float rmax<float>(float a, float b) { return fmaxf(a, b); }
template <> __device__ __forceinline__ double rmax<double>(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float rsqrt_(float a) { return sqrtf(a); }
__device__ __forceinline__ double rsqrt_(double a) { return sqrt(a); }
__device__ __forceinline__ float rabs(float a) { return fabsf(a); }
__device__ __forceinline__ double rabs(double a) { return fabs(a); }
__device__ __forceinline__ float rrcp(float a) { return 1.0f / a; }
__device__ __forceinline__ double rrcp(double a) { return 1.0 / a; }
template <class T> __device__ __forceinline__ T rinf();
template <> __device__ __forceinline__ float rinf<float>() { return CUDART_INF_F; }
template <> __device__ __forceinline__ double rinf<double>() { return CUDART_INF; }

// O2.  a = W_c - W_{c-1}, b = W_{c+1} - W_c (undivided).  Branch-free forms that return exactly
// the value of the sign-test definition:
//   minmod: max(min(a,b),0) + min(max(a,b),0)
//   MC    : 2*( max(min(a,b,q),0) + min(max(a,b,q),0) ),  q = (a+b)/4
template <class T, int LIM>
__device__ __forceinline__ T limited_slope(T a, T b) {
  if (LIM == LIM_NONE) return T(0);
  const T lo = rmin(a, b), hi = rmax(a, b);
  if (LIM == LIM_MINMOD) return rmax(lo, T(0)) + rmin(hi, T(0));
  const T q = T(0.25) * (a + b);
  return T(2) * (rmax(rmin(lo, q), T(0)) + rmin(rmax(hi, q), T(0)));
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
    T vs[2], ws[2], b1s[2], b2s[2], rs[2];
#pragma unroll
    for (int K = 0; K < 2; ++K) {
      const T m = K ? mR : mL, sk = K ? sr : sl, SKk = K ? SR : SL, u = K ? uR : uL;
      const T v = K ? vR : vL, w = K ? wR : wL, b1 = K ? b1R : b1L, b2 = K ? b2R : b2L;
      const T dSM = SKk - SM;
      rs[K] = m * rrcp(dSM);
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
    const T EsK = (skK * EK - pTK * uK + pTs * SM + Bn * (vBK - vBsK)) * rrcp(SK - SM);
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
      const T SsK = left ? (SM - aBn * rrcp(sqL)) : (SM + aBn * rrcp(sqR));
      const bool dstar = left ? (SsK < T(0)) : (SsK >= T(0));
      if (dstar) {
        const T sg = (Bn > T(0)) ? T(1) : T(-1);
        const T iSig = rrcp(sqL + sqR);
        const T vss = (sqL * vs[0] + sqR * vs[1] + (b1s[1] - b1s[0]) * sg) * iSig;
        const T wss = (sqL * ws[0] + sqR * ws[1] + (b2s[1] - b2s[0]) * sg) * iSig;
        const T b1ss = (sqL * b1s[1] + sqR * b1s[0] + sqL * sqR * (vs[1] - vs[0]) * sg) * iSig;
        const T b2ss = (sqL * b2s[1] + sqR * b2s[0] + sqL * sqR * (ws[1] - ws[0]) * sg) * iSig;
        const T vBss = SM * Bn + vss * b1ss + wss * b2ss;
        const T sqK = left ? sqL : sqR;
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

template <class T, int NF, int TX, int TY>
struct TileGeom {
  static constexpr int RW = TX + 4, RH = TY + 4, RP = RW * RH;   // ring plane (tile + radius-2 halo)
  static constexpr int NXF = (TX + 1) * TY, NYF = TX * (TY + 1);  // x / y faces per plane
  static constexpr int NCELL = TX * TY;
  static constexpr int NBC = NCELL + 2 * TY + 2 * TX;             // cells that need face states
  static constexpr size_t smem_elems = (size_t)3 * NF * RP + (size_t)3 * NF * NXF + (size_t)3 * NF * NYF;
  static constexpr size_t smem_bytes = smem_elems * sizeof(T);
};

template <class T, int NF, int LIM, int RS, int TX, int TY, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) godunov_step_kernel(const __grid_constant__ StepParams<T> P) {
  using G = TileGeom<T, NF, TX, TY>;
  constexpr int RW = G::RW, RP = G::RP, NXF = G::NXF, NYF = G::NYF, NCELL = G::NCELL, NBC = G::NBC;
  static_assert(NT >= NBC, "one thread per predictor cell");
  static_assert(NT % 32 == 0, "whole warps");

  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* ring = reinterpret_cast<T*>(smem_raw);          // [3][NF][RP]
  T* XL = ring + 3 * NF * RP;                        // [NF][NXF]  W^+_x of the cell left of the face
  T* XR = XL + NF * NXF;                             // [NF][NXF]  W^-_x of the cell right of the face
  T* FX = XR + NF * NXF;                             // [NF][NXF]
  T* YL = FX + NF * NXF;                             // [NF][NYF]
  T* YR = YL + NF * NYF;
  T* FY = YR + NF * NYF;
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

  const size_t n3 = (size_t)n * n * n;
  const size_t fs_int = (size_t)P.np * n3;
  const int M = n + 2 * P.g;
  const size_t fs_halo = (size_t)P.np * M * M * M;

  RiemannConst<T> RC;
  RC.gamma = P.gamma; RC.igm1 = P.igm1; RC.ch2 = P.ch2; RC.half_ch = T(0.5) * P.ch; RC.half_ich = P.half_ich;
  RC.eps = P.eps;

  // ---- phase A: one plane of U -> primitives -> ring slot -----------------------------------
  auto load_plane = [&](int lz, int slot) {
    const int rz = lz < 0 ? 0 : (lz >= n ? 2 : 1);
    T* dst = ring + (size_t)slot * NF * RP;
    for (int c = tid; c < RP; c += NT) {
      const int ry = c / RW, rx = c - ry * RW;
      const int hx = rx < 2 ? 2 - rx : (rx >= TX + 2 ? rx - (TX + 1) : 0);
      const int hy = ry < 2 ? 2 - ry : (ry >= TY + 2 ? ry - (TY + 1) : 0);
      if (hx + hy > 2) continue;  // outside the stencil footprint
      const int lx = x0 + rx - 2, ly = y0 + ry - 2;
      const int gx = lx < 0 ? 0 : (lx >= n ? 2 : 1), gy = ly < 0 ? 0 : (ly >= n ? 2 : 1);
      const int e = s_nbr[rz * 9 + gy * 3 + gx];
      const T* src;
      size_t fs;
      if (e >= 0) {
        const int sp = e & NBR_PATCH_MASK, md = e >> NBR_MODE_SHIFT;
        const int sx = (gx != 1 && (md & 1)) ? (gx == 0 ? 0 : n - 1) : lx - (gx - 1) * n;
        const int sy = (gy != 1 && (md & 2)) ? (gy == 0 ? 0 : n - 1) : ly - (gy - 1) * n;
        const int sz = (rz != 1 && (md & 4)) ? (rz == 0 ? 0 : n - 1) : lz - (rz - 1) * n;
        src = P.Uin + (size_t)sp * n3 + ((size_t)sz * n + sy) * n + sx;
        fs = fs_int;
      } else {
        src = P.halo + (size_t)p * M * M * M + ((size_t)(lz + P.g) * M + (ly + P.g)) * M + (lx + P.g);
        fs = fs_halo;
      }
      T u[NF];
#pragma unroll
      for (int q = 0; q < NF; ++q) u[q] = __ldg(src + q * fs);
      const T ir = rrcp(u[0]);
      const T vx = u[1] * ir, vy = u[2] * ir, vz = u[3] * ir;
      T e_int = u[4] - T(0.5) * u[0] * (vx * vx + vy * vy + vz * vz);
      if (NF == 9) e_int -= T(0.5) * (u[5] * u[5] + u[6] * u[6] + u[7] * u[7]);
      dst[0 * RP + c] = u[0];
      dst[1 * RP + c] = vx;
      dst[2 * RP + c] = vy;
      dst[3 * RP + c] = vz;
      dst[4 * RP + c] = P.gm1 * e_int;
      if (NF == 9) {
        dst[5 * RP + c] = u[5]; dst[6 * RP + c] = u[6]; dst[7 * RP + c] = u[7]; dst[8 * RP + c] = u[8];
      }
    }
  };

  // per-thread role in phase B
  const bool interior_thread = tid < NCELL;
  int bi, bj;  // tile-local cell coordinates of this thread's predictor cell
  if (tid < NCELL) { bj = tid / TX; bi = tid - bj * TX; }
  else if (tid < NCELL + 2 * TY) { const int r = tid - NCELL; bj = r >> 1; bi = (r & 1) ? TX : -1; }
  else { const int r = tid - NCELL - 2 * TY; bi = r >> 1; bj = (r & 1) ? TY : -1; }
  const int bc = (bj + 2) * RW + (bi + 2);

  T zl[NF];    // W^+_z of the previous plane (left state of the next z face)
  T fz[NF];    // flux through the lower z face of the current plane
  T fzlo[NF];  // flux through the lower z face of the plane being accumulated
  T acc[NF];   // (Fx+ - Fx-) + (Fy+ - Fy-) of the plane being accumulated
  T smax_loc = T(0);
#pragma unroll
  for (int q = 0; q < NF; ++q) { zl[q] = T(0); fz[q] = T(0); fzlo[q] = T(0); acc[q] = T(0); }

  load_plane(z0 - 2, 0);
  load_plane(z0 - 1, 1);

  for (int t = 0; t <= zc + 1; ++t) {
    const int kk = z0 - 1 + t;  // plane being predicted
    const bool mid = (t >= 1) && (t <= zc);  // kk is a plane of this tile (x/y fluxes needed)
    load_plane(kk + 1, (t + 2) % 3);
    __syncthreads();

    // ---- phase B ---------------------------------------------------------------------------
    if (tid < (mid ? NBC : NCELL)) {
      const T* Wm = ring + (size_t)(t % 3) * NF * RP;
      const T* Wc = ring + (size_t)((t + 1) % 3) * NF * RP;
      const T* Wp = ring + (size_t)((t + 2) % 3) * NF * RP;
      T w[NF], Dx[NF], Dy[NF], Dz[NF];
#pragma unroll
      for (int q = 0; q < NF; ++q) {
        const T c0 = Wc[q * RP + bc];
        w[q] = c0;
        Dx[q] = limited_slope<T, LIM>(c0 - Wc[q * RP + bc - 1], Wc[q * RP + bc + 1] - c0);
        Dy[q] = limited_slope<T, LIM>(c0 - Wc[q * RP + bc - RW], Wc[q * RP + bc + RW] - c0);
        Dz[q] = limited_slope<T, LIM>(c0 - Wm[q * RP + bc], Wp[q * RP + bc] - c0);
      }
      // O3 predictor
      const T s = P.hdtdx;
      const T rho = w[0], pr = w[4];
      const T ir = rrcp(rho);
      T ws[NF];
#define ADV(q) (w[1] * Dx[q] + w[2] * Dy[q] + w[3] * Dz[q])
      const T divv = Dx[1] + Dy[2] + Dz[3];
      ws[0] = rho - s * (ADV(0) + rho * divv);
      if (NF == 5) {
        ws[1] = w[1] - s * (ADV(1) + Dx[4] * ir);
        ws[2] = w[2] - s * (ADV(2) + Dy[4] * ir);
        ws[3] = w[3] - s * (ADV(3) + Dz[4] * ir);
        ws[4] = pr - s * (ADV(4) + P.gamma * pr * divv);
      } else {
#define BGRAD(q) (w[5] * Dx[q] + w[6] * Dy[q] + w[7] * Dz[q])
        const T divB = Dx[5] + Dy[6] + Dz[7];
        const T vB = w[1] * w[5] + w[2] * w[6] + w[3] * w[7];
        const T BdBx = w[5] * Dx[5] + w[6] * Dx[6] + w[7] * Dx[7];
        const T BdBy = w[5] * Dy[5] + w[6] * Dy[6] + w[7] * Dy[7];
        const T BdBz = w[5] * Dz[5] + w[6] * Dz[6] + w[7] * Dz[7];
        ws[1] = w[1] - s * (ADV(1) + ((Dx[4] + BdBx) - (BGRAD(5) + w[5] * divB)) * ir);
        ws[2] = w[2] - s * (ADV(2) + ((Dy[4] + BdBy) - (BGRAD(6) + w[6] * divB)) * ir);
        ws[3] = w[3] - s * (ADV(3) + ((Dz[4] + BdBz) - (BGRAD(7) + w[7] * divB)) * ir);
        ws[5] = w[5] - s * (ADV(5) + w[5] * divv - BGRAD(1) - w[1] * divB + Dx[8]);
        ws[6] = w[6] - s * (ADV(6) + w[6] * divv - BGRAD(2) - w[2] * divB + Dy[8]);
        ws[7] = w[7] - s * (ADV(7) + w[7] * divv - BGRAD(3) - w[3] * divB + Dz[8]);
        ws[4] = pr - s * (ADV(4) + P.gamma * pr * divv + P.gm1 * (vB * divB - BGRAD(8)));
        ws[8] = w[8] - s * P.ch2 * divB;
#undef BGRAD
      }
#undef ADV
      // O4 positivity: the smallest/largest of the six face values of rho and p
      const T hr = T(0.5) * rmax(rmax(rabs(Dx[0]), rabs(Dy[0])), rabs(Dz[0]));
      const T hp = T(0.5) * rmax(rmax(rabs(Dx[4]), rabs(Dy[4])), rabs(Dz[4]));
      const bool ok = (ws[0] - hr > T(0)) && (ws[4] - hp > T(0)) && (ws[0] + hr < rinf<T>()) &&
                      (ws[4] + hp < rinf<T>());
      if (!ok) {
        atomicAdd(&s_cnt[CNT_POSITIVITY], 1);
#pragma unroll
        for (int q = 0; q < NF; ++q) { ws[q] = w[q]; Dx[q] = T(0); Dy[q] = T(0); Dz[q] = T(0); }
      }
      if (mid) {
        // publish x / y face states: face fi lies between cells fi-1 and fi
        if (bj >= 0 && bj < TY) {
          const int row = bj * (TX + 1);
#pragma unroll
          for (int q = 0; q < NF; ++q) {
            if (bi < TX) XL[q * NXF + row + bi + 1] = ws[q] + T(0.5) * Dx[q];
            if (bi >= 0) XR[q * NXF + row + bi] = ws[q] - T(0.5) * Dx[q];
          }
        }
        if (bi >= 0 && bi < TX) {
#pragma unroll
          for (int q = 0; q < NF; ++q) {
            if (bj < TY) YL[q * NYF + (bj + 1) * TX + bi] = ws[q] + T(0.5) * Dy[q];
            if (bj >= 0) YR[q * NYF + bj * TX + bi] = ws[q] - T(0.5) * Dy[q];
          }
        }
      }
      if (interior_thread) {
        if (t >= 1) {  // z face between planes kk-1 and kk; rotated order (z, x, y)
          T WL[NF], WR[NF], Fr[NF];
          WL[0] = zl[0]; WL[1] = zl[3]; WL[2] = zl[1]; WL[3] = zl[2]; WL[4] = zl[4];
          WR[0] = ws[0] - T(0.5) * Dz[0]; WR[1] = ws[3] - T(0.5) * Dz[3]; WR[2] = ws[1] - T(0.5) * Dz[1];
          WR[3] = ws[2] - T(0.5) * Dz[2]; WR[4] = ws[4] - T(0.5) * Dz[4];
          if (NF == 9) {
            WL[5] = zl[7]; WL[6] = zl[5]; WL[7] = zl[6]; WL[8] = zl[8];
            WR[5] = ws[7] - T(0.5) * Dz[7]; WR[6] = ws[5] - T(0.5) * Dz[5]; WR[7] = ws[6] - T(0.5) * Dz[6];
            WR[8] = ws[8] - T(0.5) * Dz[8];
          }
          riemann<T, NF, RS>(WL, WR, RC, Fr, s_cnt);
          fz[0] = Fr[0]; fz[3] = Fr[1]; fz[1] = Fr[2]; fz[2] = Fr[3]; fz[4] = Fr[4];
          if (NF == 9) { fz[7] = Fr[5]; fz[5] = Fr[6]; fz[6] = Fr[7]; fz[8] = Fr[8]; }
        }
#pragma unroll
        for (int q = 0; q < NF; ++q) zl[q] = ws[q] + T(0.5) * Dz[q];
      }
    }
    __syncthreads();

    // ---- phase C: x and y faces of plane kk -----------------------------------------------
    if (mid) {
      for (int f = tid; f < NXF + NYF; f += NT) {
        const int d = f >= NXF ? 1 : 0;
        const int ff = f - d * NXF;
        const int stride = d ? NYF : NXF;
        const T* L = d ? YL : XL;
        const T* R = d ? YR : XR;
        T* Fo = d ? FY : FX;
        const int qn = 1 + d, q1 = 1 + (d + 1) % 3, q2 = 1 + (d + 2) % 3;
        T WL[NF], WR[NF], Fr[NF];
        WL[0] = L[ff]; WR[0] = R[ff];
        WL[1] = L[qn * stride + ff]; WR[1] = R[qn * stride + ff];
        WL[2] = L[q1 * stride + ff]; WR[2] = R[q1 * stride + ff];
        WL[3] = L[q2 * stride + ff]; WR[3] = R[q2 * stride + ff];
        WL[4] = L[4 * stride + ff]; WR[4] = R[4 * stride + ff];
        if (NF == 9) {
          WL[5] = L[(4 + qn) * stride + ff]; WR[5] = R[(4 + qn) * stride + ff];
          WL[6] = L[(4 + q1) * stride + ff]; WR[6] = R[(4 + q1) * stride + ff];
          WL[7] = L[(4 + q2) * stride + ff]; WR[7] = R[(4 + q2) * stride + ff];
          WL[8] = L[8 * stride + ff]; WR[8] = R[8 * stride + ff];
        }
        riemann<T, NF, RS>(WL, WR, RC, Fr, s_cnt);
        Fo[ff] = Fr[0];
        Fo[qn * stride + ff] = Fr[1];
        Fo[q1 * stride + ff] = Fr[2];
        Fo[q2 * stride + ff] = Fr[3];
        Fo[4 * stride + ff] = Fr[4];
        if (NF == 9) {
          Fo[(4 + qn) * stride + ff] = Fr[5];
          Fo[(4 + q1) * stride + ff] = Fr[6];
          Fo[(4 + q2) * stride + ff] = Fr[7];
          Fo[8 * stride + ff] = Fr[8];
        }
        if (P.fblk != nullptr) {  // record x / y face fluxes for the reflux
          const int blk = P.fblk_of[p];
          if (blk >= 0) {
            const int a = d ? ff % TX : ff % (TX + 1), b = d ? ff / TX : ff / (TX + 1);
            // a,b: tile-local (face or cell) coordinates along x and y
            const bool owned = d ? (b < TY || y0 + TY == n) : (a < TX || x0 + TX == n);
            if (owned) {
              const size_t fsz = (size_t)n * n * (n + 1);
              const size_t off = d ? (((size_t)kk * (n + 1) + (y0 + b)) * n + (x0 + a))
                                   : (((size_t)kk * n + (y0 + b)) * (n + 1) + (x0 + a));
              T* dstF = P.fblk + ((size_t)blk * 3 + d) * NF * fsz + off;
              dstF[0] += Fr[0];
              dstF[(size_t)qn * fsz] += Fr[1];
              dstF[(size_t)q1 * fsz] += Fr[2];
              dstF[(size_t)q2 * fsz] += Fr[3];
              dstF[(size_t)4 * fsz] += Fr[4];
              if (NF == 9) {
                dstF[(size_t)(4 + qn) * fsz] += Fr[5];
                dstF[(size_t)(4 + q1) * fsz] += Fr[6];
                dstF[(size_t)(4 + q2) * fsz] += Fr[7];
                dstF[(size_t)8 * fsz] += Fr[8];
              }
            }
          }
        }
      }
    }
    __syncthreads();

    // ---- phase D: finish plane kk-1, start accumulating plane kk ----------------------------
    if (interior_thread) {
      if (t >= 1 && P.fblk != nullptr) {  // z face flux (lower face of plane kk)
        const int blk = P.fblk_of[p];
        if (blk >= 0 && (t <= zc || z0 + zc == n)) {
          const size_t fsz = (size_t)n * n * (n + 1);
          T* dstF = P.fblk + ((size_t)blk * 3 + 2) * NF * fsz + ((size_t)kk * n + (y0 + bj)) * n + (x0 + bi);
#pragma unroll
          for (int q = 0; q < NF; ++q) dstF[(size_t)q * fsz] += fz[q];
        }
      }
      if (t >= 2) {
        const size_t cell = (size_t)p * n3 + ((size_t)(kk - 1) * n + (y0 + bj)) * n + (x0 + bi);
        T un[NF];
#pragma unroll
        for (int q = 0; q < NF; ++q) {
          const T u = __ldg(P.Uin + q * fs_int + cell);
          un[q] = u - P.dtdx * (acc[q] + (fz[q] - fzlo[q]));
        }
        if (NF == 9) un[8] *= P.damp;
#pragma unroll
        for (int q = 0; q < NF; ++q) P.Uout[q * fs_int + cell] = un[q];
        if (!(un[0] > T(0))) atomicAdd(&s_cnt[CNT_NEG_STATE], 1);
        smax_loc = rmax(smax_loc, signal_speed<T, NF>(un, P.gamma, P.gm1));
      }
      if (mid) {
        const int xr = bj * (TX + 1) + bi, yr = bj * TX + bi;
#pragma unroll
        for (int q = 0; q < NF; ++q) {
          acc[q] = (FX[q * NXF + xr + 1] - FX[q * NXF + xr]) + (FY[q * NYF + yr + TX] - FY[q * NYF + yr]);
          fzlo[q] = fz[q];
        }
      }
    }
    // no barrier needed here: the next writers of FX/FY (phase C) and of the ring slot read by this
    // iteration's phase B sit behind the barrier that follows the next load_plane
  }

  // ---- epilogue: max signal speed of the new state (O7), event counters -----------------------
  // NaN-safe: fmax drops NaNs; a NaN state shows up in the NEG_STATE counter instead.
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

// host-side launcher for one (T, NF, TX, TY, NT, MINB) tile configuration
template <class T, int NF, int LIM, int RS, int TX, int TY, int NT, int MINB>
cudaError_t launch_variant(const StepParams<T>& P, cudaStream_t s) {
  using G = TileGeom<T, NF, TX, TY>;
  auto kern = godunov_step_kernel<T, NF, LIM, RS, TX, TY, NT, MINB>;
  static bool configured = false;  // per instantiation; attribute is per device function
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem_bytes);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  const long long grid = (long long)P.np * P.ntx * P.nty * P.ntz;
  kern<<<(unsigned)grid, NT, G::smem_bytes, s>>>(P);
  return cudaGetLastError();
}

template <class T, int NF, int TX, int TY, int NT, int MINB>
cudaError_t launch_dispatch(const StepParams<T>& P, int limiter, int riemann, cudaStream_t s) {
  constexpr int RSX = (NF == 5) ? RS_HLLC : RS_HLLD;
#define AMR_CASE(L, R) \
  if (limiter == L && riemann == R) return launch_variant<T, NF, L, R, TX, TY, NT, MINB>(P, s);
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

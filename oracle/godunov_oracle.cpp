// CPU ORACLE -- TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, step-by-step implementation of the per-patch second-order Godunov hydro / MHD
// update named by BASELINE.json:north_star (MUSCL-Hancock PLM + limiter -> HLL/HLLC or
// GLM + HLL/HLLD flux -> conservative update -> CFL reduction), plus the ghost fill and the
// two-level operators (prolongation, restriction, reflux).  It follows SURVEY.md §8(c) steps
// O0..O9 in that order and notation (the paper, only NAMES these
// pieces; the formulas are the readings listed in DESIGN.md §3).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load this library.  It shares no code, header, table or helper with the CUDA path in
// paper_1412_0934_b200/csrc.  No blocking, fusion or reordering: every intermediate (primitives,
// slopes, face states, fluxes) is a full array.  OpenMP is used over patches only.
//
// Pins (tests/test_oracle_*.py): P1/P2 exact Sod solution, P3 j/k invariance, P4 uniform state,
// P5 conservation, P6 permutation/mirror symmetry, P7 Riemann identities (consistency,
// Rankine-Hugoniot closure), P8 HLLD(B=0) == HLLC and mhd(B=0) == hydro, P9 extruded
// Orszag-Tang, P10 second-order convergence (density wave, circularly polarised Alfven wave),
// P11 first-order limit, P12 predictor cross-check, P13 composite conservation, P14 prolongation
// identities, P15 closed-form CFL, P16 brute force on a 4^3 patch; round 2: the outflow clamp across sibling
// patches against numpy.pad(mode='edge') and Sod tiled 2x2x2 bitwise (test_oracle_sod.py), fine patches on
// non-periodic faces (boundary pressure force, clamped halo cells; test_oracle_amr.py), PPM (test_oracle_ppm.py).
// Parity unpinned: long-time MHD behaviour (no printed values exist in PAPER.md).
//
// Array layout (host): U[field][patch][k][j][i] with ghosts, M = n + 2g per side, i fastest.
// Field order: rho, m_x, m_y, m_z, E [, B_x, B_y, B_z, psi]  (mu_0 = 1).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum { LIM_NONE = 0, LIM_MINMOD = 1, LIM_MC = 2 };
enum { RS_HLL = 0, RS_HLLC = 1, RS_HLLD = 2 };
enum { BC_PERIODIC = 0, BC_OUTFLOW = 1 };
enum { CNT_POSITIVITY = 0, CNT_HLL_FALLBACK = 1, CNT_DEGENERATE_D = 2, CNT_NEG_STATE = 3 };

struct Geom {
  int np, n, g, nf, M;
  const int* origin;  // [np][3] (x, y, z), level-cell units
  int dom[3];
  int bc[6];
  int selfp;
  size_t M3() const { return (size_t)M * M * M; }
  size_t cell(int i, int j, int k) const { return ((size_t)(k + g) * M + (j + g)) * M + (i + g); }
  size_t fld(int f, int p) const { return ((size_t)f * np + p) * M3(); }
};

// Dense map (patch-grid coordinates) -> patch index, -1 where no patch exists.
struct PatchMap {
  int dims[3];
  std::vector<int> idx;
  explicit PatchMap(const Geom& G) {
    for (int d = 0; d < 3; ++d) dims[d] = G.dom[d] / G.n;
    idx.assign((size_t)dims[0] * dims[1] * dims[2], -1);
    if (G.selfp) return;
    for (int p = 0; p < G.np; ++p) {
      int a = G.origin[3 * p] / G.n, b = G.origin[3 * p + 1] / G.n, c = G.origin[3 * p + 2] / G.n;
      idx[((size_t)c * dims[1] + b) * dims[0] + a] = p;
    }
  }
  int at(int gx, int gy, int gz, int n) const {  // gx.. are in-domain cell indices
    int a = gx / n, b = gy / n, c = gz / n;
    return idx[((size_t)c * dims[1] + b) * dims[0] + a];
  }
};

// ------------------------------------------------------------------------------------------
// O2. limited slope of one primitive component (undivided differences a = W_c - W_{c-1},
// b = W_{c+1} - W_c).  Sign tests, not a*b > 0.
// ------------------------------------------------------------------------------------------
template <class T>
T limited_slope(T a, T b, int lim) {
  if (lim == LIM_NONE) return T(0);
  if (lim == LIM_MINMOD) {
    if (a > 0 && b > 0) return std::min(a, b);
    if (a < 0 && b < 0) return std::max(a, b);
    return T(0);
  }
  // MC: magnitude min(2|a|, 2|b|, |a+b|/2), sign of a
  if (a > 0 && b > 0) return std::min(std::min(T(2) * a, T(2) * b), T(0.5) * (a + b));
  if (a < 0 && b < 0) return -std::min(std::min(T(2) * (-a), T(2) * (-b)), T(0.5) * (-(a + b)));
  return T(0);
}

// ------------------------------------------------------------------------------------------
// O5. Riemann solvers.  1-D states are in the rotated order (n, t1, t2):
//   hydro W = (rho, u, v, w, p);  MHD W = (rho, u, v, w, p, Bn, Bt1, Bt2, psi).
// Returned fluxes are for (rho, m_n, m_t1, m_t2, E [, Bn, Bt1, Bt2, psi]).
// ------------------------------------------------------------------------------------------
template <class T>
void riemann_hydro(const T* WL, const T* WR, T gamma, int solver, T* F, long long* cnt) {
  const T rL = WL[0], uL = WL[1], vL = WL[2], wL = WL[3], pL = WL[4];
  const T rR = WR[0], uR = WR[1], vR = WR[2], wR = WR[3], pR = WR[4];
  const T EL = pL / (gamma - 1) + T(0.5) * rL * (uL * uL + vL * vL + wL * wL);
  const T ER = pR / (gamma - 1) + T(0.5) * rR * (uR * uR + vR * vR + wR * wR);
  const T cL = std::sqrt(gamma * pL / rL), cR = std::sqrt(gamma * pR / rR);
  const T SL = std::min(uL, uR) - std::max(cL, cR);
  const T SR = std::max(uL, uR) + std::max(cL, cR);
  const T UL[5] = {rL, rL * uL, rL * vL, rL * wL, EL};
  const T UR[5] = {rR, rR * uR, rR * vR, rR * wR, ER};
  const T FL[5] = {rL * uL, rL * uL * uL + pL, rL * uL * vL, rL * uL * wL, (EL + pL) * uL};
  const T FR[5] = {rR * uR, rR * uR * uR + pR, rR * uR * vR, rR * uR * wR, (ER + pR) * uR};
  if (SL >= 0) { for (int q = 0; q < 5; ++q) F[q] = FL[q]; return; }
  if (SR <= 0) { for (int q = 0; q < 5; ++q) F[q] = FR[q]; return; }
  bool use_hll = (solver == RS_HLL);
  T Ss = 0;
  if (!use_hll) {
    Ss = (pR - pL + rL * uL * (SL - uL) - rR * uR * (SR - uR)) / (rL * (SL - uL) - rR * (SR - uR));
    const T ps = pL + rL * (SL - uL) * (Ss - uL);
    if (!(ps > 0)) { use_hll = true; if (cnt) cnt[CNT_HLL_FALLBACK]++; }
  }
  if (use_hll) {
    for (int q = 0; q < 5; ++q)
      F[q] = (SR * FL[q] - SL * FR[q] + SL * SR * (UR[q] - UL[q])) / (SR - SL);
    return;
  }
  // HLLC star state of side K
  const bool left = (Ss >= 0);
  const T rK = left ? rL : rR, uK = left ? uL : uR, vK = left ? vL : vR, wK = left ? wL : wR;
  const T pK = left ? pL : pR, EK = left ? EL : ER, SK = left ? SL : SR;
  const T* UK = left ? UL : UR;
  const T* FK = left ? FL : FR;
  const T fac = rK * (SK - uK) / (SK - Ss);
  const T Us[5] = {fac, fac * Ss, fac * vK, fac * wK,
                   fac * (EK / rK + (Ss - uK) * (Ss + pK / (rK * (SK - uK))))};
  for (int q = 0; q < 5; ++q) F[q] = FK[q] + SK * (Us[q] - UK[q]);
}

template <class T>
struct HlldDebug {  // intermediate states for pin P7 (7 components: rho, mn, mt1, mt2, E, Bt1, Bt2)
  T S[5];           // SL, SL*, SM, SR*, SR
  T U[6][7];        // UL, UL*, UL**, UR**, UR*, UR
  T FL[7], FR[7];
  T ptstar, Bn;
  int path;         // 0 FL,1 FR,2 FL*,3 FL**,4 FR**,5 FR*, 6 HLL(requested), 7 HLL fallback, 8/9 star w/o ** (L/R)
};

template <class T>
void riemann_mhd(const T* WL_in, const T* WR_in, T gamma, T ch, int solver, T eps, T* F,
                 long long* cnt, HlldDebug<T>* dbg) {
  // GLM pre-step: 2x2 upwind system for (Bn, psi)
  const T BnL = WL_in[5], BnR = WR_in[5], psL = WL_in[8], psR = WR_in[8];
  const T Bn = T(0.5) * (BnL + BnR) - (psR - psL) / (T(2) * ch);
  const T psis = T(0.5) * (psL + psR) - T(0.5) * ch * (BnR - BnL);
  F[5] = psis;
  F[8] = ch * ch * Bn;
  if (dbg) dbg->Bn = Bn;

  struct Side { T r, u, v, w, p, b1, b2, B2, pT, E, vB, cf; T U[7], Fl[7]; };
  Side sd[2];
  const T* Win[2] = {WL_in, WR_in};
  for (int K = 0; K < 2; ++K) {
    Side& s = sd[K];
    const T* W = Win[K];
    s.r = W[0]; s.u = W[1]; s.v = W[2]; s.w = W[3]; s.p = W[4]; s.b1 = W[6]; s.b2 = W[7];
    s.B2 = Bn * Bn + s.b1 * s.b1 + s.b2 * s.b2;
    s.pT = s.p + T(0.5) * s.B2;
    s.E = s.p / (gamma - 1) + T(0.5) * s.r * (s.u * s.u + s.v * s.v + s.w * s.w) + T(0.5) * s.B2;
    s.vB = s.u * Bn + s.v * s.b1 + s.w * s.b2;
    const T a = (gamma * s.p + s.B2) / s.r;
    const T disc = std::max(a * a - T(4) * gamma * s.p * Bn * Bn / (s.r * s.r), T(0));
    s.cf = std::sqrt(T(0.5) * (a + std::sqrt(disc)));
    s.U[0] = s.r; s.U[1] = s.r * s.u; s.U[2] = s.r * s.v; s.U[3] = s.r * s.w; s.U[4] = s.E;
    s.U[5] = s.b1; s.U[6] = s.b2;
    s.Fl[0] = s.r * s.u;
    s.Fl[1] = s.r * s.u * s.u + s.pT - Bn * Bn;
    s.Fl[2] = s.r * s.u * s.v - Bn * s.b1;
    s.Fl[3] = s.r * s.u * s.w - Bn * s.b2;
    s.Fl[4] = (s.E + s.pT) * s.u - Bn * s.vB;
    s.Fl[5] = s.u * s.b1 - s.v * Bn;
    s.Fl[6] = s.u * s.b2 - s.w * Bn;
  }
  const Side &L = sd[0], &R = sd[1];
  const T SL = std::min(L.u, R.u) - std::max(L.cf, R.cf);
  const T SR = std::max(L.u, R.u) + std::max(L.cf, R.cf);
  static const int map7[7] = {0, 1, 2, 3, 4, 6, 7};  // 7-vector slot -> 9-flux slot
  auto put = [&](const T* f7) { for (int q = 0; q < 7; ++q) F[map7[q]] = f7[q]; };
  if (dbg) {
    dbg->S[0] = SL; dbg->S[4] = SR; dbg->S[1] = dbg->S[2] = dbg->S[3] = 0; dbg->ptstar = 0;
    for (int q = 0; q < 7; ++q) { dbg->U[0][q] = L.U[q]; dbg->U[5][q] = R.U[q]; dbg->FL[q] = L.Fl[q]; dbg->FR[q] = R.Fl[q]; }
  }
  if (SL >= 0) { put(L.Fl); if (dbg) dbg->path = 0; return; }
  if (SR <= 0) { put(R.Fl); if (dbg) dbg->path = 1; return; }
  auto hll = [&]() {
    T f7[7];
    for (int q = 0; q < 7; ++q)
      f7[q] = (SR * L.Fl[q] - SL * R.Fl[q] + SL * SR * (R.U[q] - L.U[q])) / (SR - SL);
    put(f7);
  };
  if (solver == RS_HLL) { hll(); if (dbg) dbg->path = 6; return; }

  // HLLD (Miyoshi & Kusano 2005), Bn == Bn* on both sides
  const T sl = SL - L.u, sr = SR - R.u;
  const T den = sr * R.r - sl * L.r;
  const T SM = (sr * R.r * R.u - sl * L.r * L.u - R.pT + L.pT) / den;
  const T pTs = (sr * R.r * L.pT - sl * L.r * R.pT + L.r * R.r * sr * sl * (R.u - L.u)) / den;
  if (dbg) { dbg->S[2] = SM; dbg->ptstar = pTs; }
  if (!(pTs > 0)) { hll(); if (cnt) cnt[CNT_HLL_FALLBACK]++; if (dbg) dbg->path = 7; return; }
  T rs[2], vs[2], ws[2], b1s[2], b2s[2], vBs[2], Es[2], Us[2][7], Fs[2][7];
  const T SK[2] = {SL, SR};
  for (int K = 0; K < 2; ++K) {
    const Side& s = sd[K];
    const T sk = SK[K] - s.u;
    rs[K] = s.r * sk / (SK[K] - SM);
    const T D = s.r * sk * (SK[K] - SM) - Bn * Bn;
    if (std::fabs(D) < eps * s.r * sk * sk) {
      vs[K] = s.v; ws[K] = s.w; b1s[K] = s.b1; b2s[K] = s.b2;
      if (cnt) cnt[CNT_DEGENERATE_D]++;
    } else {
      vs[K] = s.v - Bn * s.b1 * (SM - s.u) / D;
      ws[K] = s.w - Bn * s.b2 * (SM - s.u) / D;
      b1s[K] = s.b1 * (s.r * sk * sk - Bn * Bn) / D;
      b2s[K] = s.b2 * (s.r * sk * sk - Bn * Bn) / D;
    }
    vBs[K] = SM * Bn + vs[K] * b1s[K] + ws[K] * b2s[K];
    Es[K] = (sk * s.E - s.pT * s.u + pTs * SM + Bn * (s.vB - vBs[K])) / (SK[K] - SM);
    Us[K][0] = rs[K]; Us[K][1] = rs[K] * SM; Us[K][2] = rs[K] * vs[K]; Us[K][3] = rs[K] * ws[K];
    Us[K][4] = Es[K]; Us[K][5] = b1s[K]; Us[K][6] = b2s[K];
    for (int q = 0; q < 7; ++q) Fs[K][q] = s.Fl[q] + SK[K] * (Us[K][q] - s.U[q]);
  }
  if (dbg) for (int q = 0; q < 7; ++q) { dbg->U[1][q] = Us[0][q]; dbg->U[4][q] = Us[1][q]; }
  if (Bn * Bn < eps * pTs) {  // no rotational waves: two-state (HLLC-like) fan
    if (dbg) {
      dbg->S[1] = dbg->S[3] = SM;
      for (int q = 0; q < 7; ++q) { dbg->U[2][q] = Us[0][q]; dbg->U[3][q] = Us[1][q]; }
    }
    if (SM >= 0) { put(Fs[0]); if (dbg) dbg->path = 8; } else { put(Fs[1]); if (dbg) dbg->path = 9; }
    return;
  }
  const T sqL = std::sqrt(rs[0]), sqR = std::sqrt(rs[1]);
  const T SsL = SM - std::fabs(Bn) / sqL, SsR = SM + std::fabs(Bn) / sqR;
  const T sg = (Bn > 0) ? T(1) : T(-1);
  const T Sig = sqL + sqR;
  const T vss = (sqL * vs[0] + sqR * vs[1] + (b1s[1] - b1s[0]) * sg) / Sig;
  const T wss = (sqL * ws[0] + sqR * ws[1] + (b2s[1] - b2s[0]) * sg) / Sig;
  const T b1ss = (sqL * b1s[1] + sqR * b1s[0] + sqL * sqR * (vs[1] - vs[0]) * sg) / Sig;
  const T b2ss = (sqL * b2s[1] + sqR * b2s[0] + sqL * sqR * (ws[1] - ws[0]) * sg) / Sig;
  const T vBss = SM * Bn + vss * b1ss + wss * b2ss;
  const T EssL = Es[0] - sqL * (vBs[0] - vBss) * sg;
  const T EssR = Es[1] + sqR * (vBs[1] - vBss) * sg;
  T Uss[2][7], Fss[2][7];
  const T Ess[2] = {EssL, EssR};
  const T SsK[2] = {SsL, SsR};
  for (int K = 0; K < 2; ++K) {
    Uss[K][0] = rs[K]; Uss[K][1] = rs[K] * SM; Uss[K][2] = rs[K] * vss; Uss[K][3] = rs[K] * wss;
    Uss[K][4] = Ess[K]; Uss[K][5] = b1ss; Uss[K][6] = b2ss;
    for (int q = 0; q < 7; ++q) Fss[K][q] = Fs[K][q] + SsK[K] * (Uss[K][q] - Us[K][q]);
  }
  if (dbg) {
    dbg->S[1] = SsL; dbg->S[3] = SsR;
    for (int q = 0; q < 7; ++q) { dbg->U[2][q] = Uss[0][q]; dbg->U[3][q] = Uss[1][q]; }
  }
  if (SsL >= 0) { put(Fs[0]); if (dbg) dbg->path = 2; }
  else if (SM >= 0) { put(Fss[0]); if (dbg) dbg->path = 3; }
  else if (SsR >= 0) { put(Fss[1]); if (dbg) dbg->path = 4; }
  else { put(Fs[1]); if (dbg) dbg->path = 5; }
}

// ------------------------------------------------------------------------------------------
// O1..O6 on one patch.  Scratch arrays are full ghosted cubes, one per intermediate.
// ------------------------------------------------------------------------------------------
template <class T>
struct StepParams {
  T dt, dx, gamma, ch, alpha, eps;
  int limiter, riemann;
};

template <class T>
struct Scratch {
  std::vector<T> W, dW, Wm, Wp, F;
  void init(int nf, size_t M3) {
    W.assign(nf * M3, T(0));
    dW.assign(3 * nf * M3, T(0));
    Wm.assign(3 * nf * M3, T(0));
    Wp.assign(3 * nf * M3, T(0));
    F.assign(3 * nf * M3, T(0));
  }
};

// O1: primitives W = (rho, v, p [, B, psi]) on every cell including ghosts.
template <class T>
void primitives(const T* U, const Geom& G, int p, T gamma, T* W) {
  const size_t M3 = G.M3();
  const int nf = G.nf;
  for (size_t c = 0; c < M3; ++c) {
    const T rho = U[G.fld(0, p) + c];
    const T vx = U[G.fld(1, p) + c] / rho, vy = U[G.fld(2, p) + c] / rho, vz = U[G.fld(3, p) + c] / rho;
    const T E = U[G.fld(4, p) + c];
    T pr;
    if (nf == 9) {
      const T bx = U[G.fld(5, p) + c], by = U[G.fld(6, p) + c], bz = U[G.fld(7, p) + c];
      pr = (gamma - 1) * (E - T(0.5) * rho * (vx * vx + vy * vy + vz * vz) - T(0.5) * (bx * bx + by * by + bz * bz));
      W[5 * M3 + c] = bx; W[6 * M3 + c] = by; W[7 * M3 + c] = bz; W[8 * M3 + c] = U[G.fld(8, p) + c];
    } else {
      pr = (gamma - 1) * (E - T(0.5) * rho * (vx * vx + vy * vy + vz * vz));
    }
    W[0 * M3 + c] = rho; W[1 * M3 + c] = vx; W[2 * M3 + c] = vy; W[3 * M3 + c] = vz; W[4 * M3 + c] = pr;
  }
}

template <class T>
void step_patch(const T* Uin, T* Uout, T* Fout, T* FSout, const Geom& G, int p,
                const StepParams<T>& P, Scratch<T>& S, long long* cnt) {
  const int n = G.n, nf = G.nf, M = G.M;
  const size_t M3 = G.M3();
  const size_t str[3] = {1, (size_t)M, (size_t)M * M};
  T* W = S.W.data();
  auto dWp = [&](int d, int q) { return S.dW.data() + ((size_t)d * nf + q) * M3; };
  auto Wmp = [&](int d, int q) { return S.Wm.data() + ((size_t)d * nf + q) * M3; };
  auto Wpp = [&](int d, int q) { return S.Wp.data() + ((size_t)d * nf + q) * M3; };
  auto Fp = [&](int d, int q) { return S.F.data() + ((size_t)d * nf + q) * M3; };

  primitives(Uin, G, p, P.gamma, W);  // O1

  // O2: slopes on the interior grown by one layer
  for (int k = -1; k <= n; ++k)
    for (int j = -1; j <= n; ++j)
      for (int i = -1; i <= n; ++i) {
        const size_t c = G.cell(i, j, k);
        for (int d = 0; d < 3; ++d)
          for (int q = 0; q < nf; ++q) {
            const T* w = W + q * M3;
            const T a = w[c] - w[c - str[d]];
            const T b = w[c + str[d]] - w[c];
            dWp(d, q)[c] = limited_slope(a, b, P.limiter);
          }
      }

  // O3 + O4: half-step predictor and the six face states
  const T s = P.dt / (T(2) * P.dx);
  for (int k = -1; k <= n; ++k)
    for (int j = -1; j <= n; ++j)
      for (int i = -1; i <= n; ++i) {
        const size_t c = G.cell(i, j, k);
        T w[9], D[3][9], ws[9];
        for (int q = 0; q < nf; ++q) {
          w[q] = W[q * M3 + c];
          for (int d = 0; d < 3; ++d) D[d][q] = dWp(d, q)[c];
        }
        const T rho = w[0], pr = w[4];
        const T* v = w + 1;
        auto adv = [&](int q) { return v[0] * D[0][q] + v[1] * D[1][q] + v[2] * D[2][q]; };
        const T divv = D[0][1] + D[1][2] + D[2][3];
        ws[0] = rho - s * (adv(0) + rho * divv);
        if (nf == 5) {
          for (int e = 0; e < 3; ++e) ws[1 + e] = v[e] - s * (adv(1 + e) + D[e][4] / rho);
          ws[4] = pr - s * (adv(4) + P.gamma * pr * divv);
        } else {
          const T* B = w + 5;
          const T divB = D[0][5] + D[1][6] + D[2][7];
          auto Bgrad = [&](int q) { return B[0] * D[0][q] + B[1] * D[1][q] + B[2] * D[2][q]; };
          const T vB = v[0] * B[0] + v[1] * B[1] + v[2] * B[2];
          for (int e = 0; e < 3; ++e) {
            const T BdB = B[0] * D[e][5] + B[1] * D[e][6] + B[2] * D[e][7];
            ws[1 + e] = v[e] - s * (adv(1 + e) + (D[e][4] + BdB) / rho - (Bgrad(5 + e) + B[e] * divB) / rho);
            ws[5 + e] = B[e] - s * (adv(5 + e) + B[e] * divv - Bgrad(1 + e) - v[e] * divB + D[e][8]);
          }
          ws[4] = pr - s * (adv(4) + P.gamma * pr * divv + (P.gamma - 1) * (vB * divB - Bgrad(8)));
          ws[8] = w[8] - s * P.ch * P.ch * divB;
        }
        // O4 with positivity fallback
        bool ok = (ws[0] > 0) && (ws[4] > 0) && std::isfinite(ws[0]) && std::isfinite(ws[4]);
        T fm[3][9], fp[3][9];
        for (int d = 0; d < 3; ++d)
          for (int q = 0; q < nf; ++q) {
            fm[d][q] = ws[q] - T(0.5) * D[d][q];
            fp[d][q] = ws[q] + T(0.5) * D[d][q];
          }
        for (int d = 0; d < 3; ++d)
          ok = ok && (fm[d][0] > 0) && (fm[d][4] > 0) && (fp[d][0] > 0) && (fp[d][4] > 0) &&
               std::isfinite(fm[d][0]) && std::isfinite(fm[d][4]) && std::isfinite(fp[d][0]) &&
               std::isfinite(fp[d][4]);
        if (!ok) {
          // count only cells whose face states are actually consumed (interior + face neighbours)
          const int outside = (i < 0 || i >= n) + (j < 0 || j >= n) + (k < 0 || k >= n);
          if (cnt && outside <= 1) cnt[CNT_POSITIVITY]++;
          for (int d = 0; d < 3; ++d)
            for (int q = 0; q < nf; ++q) fm[d][q] = fp[d][q] = w[q];
        }
        for (int d = 0; d < 3; ++d)
          for (int q = 0; q < nf; ++q) { Wmp(d, q)[c] = fm[d][q]; Wpp(d, q)[c] = fp[d][q]; }
      }

  // O5: one flux per face; F[d] at cell c is the flux through the LOWER d-face of c
  for (int d = 0; d < 3; ++d) {
    const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
    int lo[3] = {0, 0, 0}, hi[3] = {n - 1, n - 1, n - 1};
    hi[d] = n;
    for (int k = lo[2]; k <= hi[2]; ++k)
      for (int j = lo[1]; j <= hi[1]; ++j)
        for (int i = lo[0]; i <= hi[0]; ++i) {
          const size_t c = G.cell(i, j, k), cl = c - str[d];
          T WL[9], WR[9], Fr[9];
          WL[0] = Wpp(d, 0)[cl]; WR[0] = Wmp(d, 0)[c];
          WL[1] = Wpp(d, 1 + d)[cl]; WR[1] = Wmp(d, 1 + d)[c];
          WL[2] = Wpp(d, 1 + t1)[cl]; WR[2] = Wmp(d, 1 + t1)[c];
          WL[3] = Wpp(d, 1 + t2)[cl]; WR[3] = Wmp(d, 1 + t2)[c];
          WL[4] = Wpp(d, 4)[cl]; WR[4] = Wmp(d, 4)[c];
          if (nf == 9) {
            WL[5] = Wpp(d, 5 + d)[cl]; WR[5] = Wmp(d, 5 + d)[c];
            WL[6] = Wpp(d, 5 + t1)[cl]; WR[6] = Wmp(d, 5 + t1)[c];
            WL[7] = Wpp(d, 5 + t2)[cl]; WR[7] = Wmp(d, 5 + t2)[c];
            WL[8] = Wpp(d, 8)[cl]; WR[8] = Wmp(d, 8)[c];
            riemann_mhd<T>(WL, WR, P.gamma, P.ch, P.riemann, P.eps, Fr, cnt, nullptr);
          } else {
            riemann_hydro<T>(WL, WR, P.gamma, P.riemann, Fr, cnt);
          }
          Fp(d, 0)[c] = Fr[0];
          Fp(d, 1 + d)[c] = Fr[1]; Fp(d, 1 + t1)[c] = Fr[2]; Fp(d, 1 + t2)[c] = Fr[3];
          Fp(d, 4)[c] = Fr[4];
          if (nf == 9) {
            Fp(d, 5 + d)[c] = Fr[5]; Fp(d, 5 + t1)[c] = Fr[6]; Fp(d, 5 + t2)[c] = Fr[7];
            Fp(d, 8)[c] = Fr[8];
          }
        }
  }

  // O6: conservative update of the interior (bracket order as written), then GLM damping
  const T dtdx = P.dt / P.dx;
  const T damp = (nf == 9) ? (T)std::exp(-(double)P.alpha * (double)P.ch * (double)P.dt / (double)P.dx) : T(1);
  for (int q = 0; q < nf; ++q) {
    const T* u = Uin + G.fld(q, p);
    T* un = Uout + G.fld(q, p);
    const T *fx = Fp(0, q), *fy = Fp(1, q), *fz = Fp(2, q);
    for (int k = 0; k < n; ++k)
      for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) {
          const size_t c = G.cell(i, j, k);
          T r = u[c] - dtdx * ((fx[c + str[0]] - fx[c]) + (fy[c + str[1]] - fy[c]) + (fz[c + str[2]] - fz[c]));
          if (q == 8) r *= damp;
          un[c] = r;
        }
  }
  if (cnt) {
    for (int k = 0; k < n; ++k)
      for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) {
          const size_t c = G.cell(i, j, k);
          if (!(Uout[G.fld(0, p) + c] > 0)) cnt[CNT_NEG_STATE]++;
        }
  }
  if (Fout)  // Fout[d][field][patch][M^3]: flux through the lower d-face of each cell
    for (int d = 0; d < 3; ++d)
      for (int q = 0; q < nf; ++q)
        std::memcpy(Fout + (((size_t)d * nf + q) * G.np + p) * M3, Fp(d, q), M3 * sizeof(T));
  if (FSout)  // FSout[d][side(0:-,1:+)][field][patch][M^3]: face states W^-_d, W^+_d
    for (int d = 0; d < 3; ++d)
      for (int q = 0; q < nf; ++q) {
        std::memcpy(FSout + ((((size_t)d * 2 + 0) * nf + q) * G.np + p) * M3, Wmp(d, q), M3 * sizeof(T));
        std::memcpy(FSout + ((((size_t)d * 2 + 1) * nf + q) * G.np + p) * M3, Wpp(d, q), M3 * sizeof(T));
      }
}

template <class T>
int step_all(const T* Uin, T* Uout, T* Fout, T* FSout, const Geom& G, const StepParams<T>& P,
             long long* counters) {
  long long tot[4] = {0, 0, 0, 0};
#pragma omp parallel
  {
    Scratch<T> S;
    S.init(G.nf, G.M3());
    long long cnt[4] = {0, 0, 0, 0};
#pragma omp for schedule(dynamic, 1)
    for (int p = 0; p < G.np; ++p) step_patch<T>(Uin, Uout, Fout, FSout, G, p, P, S, cnt);
#pragma omp critical
    for (int q = 0; q < 4; ++q) tot[q] += cnt[q];
  }
  if (counters) for (int q = 0; q < 4; ++q) counters[q] = tot[q];
  return 0;
}

// ------------------------------------------------------------------------------------------
// PPM (SURVEY.md 8(f1); PAPER.md:43 "the Piecewise Parabolic Method, PPM [9]", :76 "the PLM/PPM hydro
// solver, have been ported to NVIDIA's CUDA").  The paper gives no formula; reading R-PPM of DESIGN.md
// section 13: Colella & Woodward 1984 in the direct Eulerian, dimensionally split form (as in Enzo), hydro
// only, primitive variables (rho, u, v, w, p) with u along the sweep, WITHOUT the optional dissipation of
// CW84 section 4 (no contact steepening, no flattening, no artificial viscosity), and with the boundary's
// HLL / HLLC flux (O5) in place of CW84's two-shock solver.  One sweep along direction d:
//   P1  interface values, CW84 (1.6)-(1.8) on a uniform grid:
//         da_i  = (a_{i+1} - a_{i-1}) / 2
//         dm_i  = min(|da_i|, 2|a_i - a_{i-1}|, 2|a_{i+1} - a_i|) sgn(da_i)  if (a_{i+1}-a_i)(a_i-a_{i-1}) > 0, else 0
//         a_{i+1/2} = a_i + (a_{i+1} - a_i)/2 - (dm_{i+1} - dm_i)/6 ;   aL_i = a_{i-1/2}, aR_i = a_{i+1/2}
//   P2  monotonisation, CW84 (1.10):
//         (aR-a)(a-aL) <= 0                          -> aL = aR = a
//         (aR-aL)(a-(aL+aR)/2) >  (aR-aL)^2/6        -> aL = 3a - 2aR
//         (aR-aL)(a-(aL+aR)/2) < -(aR-aL)^2/6        -> aR = 3a - 2aL
//       then  Da = aR - aL,  a6 = 6(a - (aL+aR)/2)
//   P3  averages over the domain of dependence of a wave of speed lambda, CW84 (1.12), s = |lambda| dt/dx:
//         towards the upper face: Ip(s) = aR - s/2 (Da - (1 - 2s/3) a6)
//         towards the lower face: Im(s) = aL + s/2 (Da + (1 - 2s/3) a6)
//   P4  characteristic tracing, CW84 section 3 (3.5)-(3.7), written with the eigenvectors of the primitive
//       system at the cell centre (c = sqrt(gamma p / rho); waves lambda_- = u-c, lambda_0 = u, lambda_+ = u+c):
//       upper-face state W^+ : reference = Ip(max(lambda_+,0) dt/dx) of every variable; for every wave k with
//         lambda_k > 0 subtract  [l_k . (ref - Ip_k)] r_k ,  Ip_k = Ip(lambda_k dt/dx)
//       lower-face state W^- : reference = Im(max(-lambda_-,0) dt/dx); for every wave k with lambda_k < 0
//         subtract  [l_k . (ref - Im_k)] r_k ,  Im_k = Im(-lambda_k dt/dx)
//       on (rho, u, p):  l_- = (0, -rho/(2c), 1/(2c^2)), r_- = (1, -c/rho, c^2);  l_0 = (1, 0, -1/c^2),
//       r_0 = (1, 0, 0);  l_+ = (0, rho/(2c), 1/(2c^2)), r_+ = (1, c/rho, c^2);  the transverse velocities
//       ride on lambda_0: v^+ = Ip_0(v) if u > 0 else ref, v^- = Im_0(v) if u < 0 else ref.
//       A cell whose traced rho or p is <= 0 (or non-finite) uses its cell-centre W for both states (counted).
//   P5  flux at the lower face of cell i from (W^+_{i-1}, W^-_i) with O5's HLL / HLLC;  U_i -= dt/dx (F_{i+1/2} - F_{i-1/2}).
// A step is three sweeps, x-y-z (order 0) or z-y-x (order 1), the ghost cells refilled before every sweep
// (sequenced by oracle/api.py).  Needs g >= 3 ghost layers along the sweep (reading A11).
// ------------------------------------------------------------------------------------------
template <class T>
void ppm_parabola(T am2, T am1, T a0, T ap1, T ap2, T* aL, T* aR) {
  auto dm = [](T l, T c, T r) {
    const T da = T(0.5) * (r - l);
    if ((r - c) * (c - l) > 0) {
      const T m = std::min(std::min(std::fabs(da), T(2) * std::fabs(c - l)), T(2) * std::fabs(r - c));
      return da > 0 ? m : -m;
    }
    return T(0);
  };
  const T dmm = dm(am2, am1, a0), dm0 = dm(am1, a0, ap1), dmp = dm(a0, ap1, ap2);
  T l = am1 + T(0.5) * (a0 - am1) - (dm0 - dmm) / T(6);   // a_{i-1/2}
  T r = a0 + T(0.5) * (ap1 - a0) - (dmp - dm0) / T(6);    // a_{i+1/2}
  if ((r - a0) * (a0 - l) <= 0) { l = a0; r = a0; }
  else {
    const T d = r - l, m = a0 - T(0.5) * (l + r);
    if (d * m > d * d / T(6)) l = T(3) * a0 - T(2) * r;
    else if (-(d * d) / T(6) > d * m) r = T(3) * a0 - T(2) * l;
  }
  *aL = l; *aR = r;
}

template <class T>
void ppm_sweep_patch(const T* Uin, T* Uout, const Geom& G, int p, int d, T dt, T dx, T gamma, int solver,
                     std::vector<T>& W, std::vector<T>& Wm, std::vector<T>& Wp, std::vector<T>& F, long long* cnt) {
  const int n = G.n, M = G.M;
  const size_t M3 = G.M3();
  const size_t str[3] = {1, (size_t)M, (size_t)M * M};
  const size_t sd = str[d];
  const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  primitives(Uin, G, p, gamma, W.data());      // W[q*M3 + c], q = rho, vx, vy, vz, p
  const int qu = 1 + d, qv = 1 + t1, qw = 1 + t2;
  const int order[5] = {0, qu, qv, qw, 4};     // (rho, u, v, w, p) in sweep order
  const T lam = dt / dx;
  int lo[3] = {0, 0, 0}, hi[3] = {n - 1, n - 1, n - 1};
  lo[d] = -1; hi[d] = n;
  // P1-P4 on the interior grown by one cell along d
  for (int k = lo[2]; k <= hi[2]; ++k)
    for (int j = lo[1]; j <= hi[1]; ++j)
      for (int i = lo[0]; i <= hi[0]; ++i) {
        const size_t c = G.cell(i, j, k);
        T a[5], aL[5], aR[5], Da[5], a6[5];
        for (int m = 0; m < 5; ++m) {
          const T* w = W.data() + (size_t)order[m] * M3;
          a[m] = w[c];
          ppm_parabola<T>(w[c - 2 * sd], w[c - sd], w[c], w[c + sd], w[c + 2 * sd], &aL[m], &aR[m]);
          Da[m] = aR[m] - aL[m];
          a6[m] = T(6) * (a[m] - T(0.5) * (aL[m] + aR[m]));
        }
        auto Ip = [&](int m, T s) { return aR[m] - T(0.5) * s * (Da[m] - (T(1) - T(2) * s / T(3)) * a6[m]); };
        auto Im = [&](int m, T s) { return aL[m] + T(0.5) * s * (Da[m] + (T(1) - T(2) * s / T(3)) * a6[m]); };
        const T rho = a[0], u = a[1], pr = a[4];
        const T cs = std::sqrt(gamma * pr / rho);
        const T lk[3] = {u - cs, u, u + cs};
        T wp[5], wm[5];
        {  // upper-face state
          const T sref = std::max(lk[2], T(0)) * lam;
          T ref[5];
          for (int m = 0; m < 5; ++m) { ref[m] = Ip(m, sref); wp[m] = ref[m]; }
          for (int kx = 0; kx < 3; ++kx) {
            if (!(lk[kx] > 0)) continue;
            const T s = lk[kx] * lam;
            const T dr = ref[0] - Ip(0, s), du = ref[1] - Ip(1, s), dp = ref[4] - Ip(4, s);
            if (kx == 0) { const T b = -rho / (T(2) * cs) * du + dp / (T(2) * cs * cs); wp[0] -= b; wp[1] -= b * (-cs / rho); wp[4] -= b * cs * cs; }
            else if (kx == 2) { const T b = rho / (T(2) * cs) * du + dp / (T(2) * cs * cs); wp[0] -= b; wp[1] -= b * (cs / rho); wp[4] -= b * cs * cs; }
            else { wp[0] -= dr - dp / (cs * cs); wp[2] = Ip(2, s); wp[3] = Ip(3, s); }
          }
        }
        {  // lower-face state
          const T sref = std::max(-lk[0], T(0)) * lam;
          T ref[5];
          for (int m = 0; m < 5; ++m) { ref[m] = Im(m, sref); wm[m] = ref[m]; }
          for (int kx = 0; kx < 3; ++kx) {
            if (!(lk[kx] < 0)) continue;
            const T s = -lk[kx] * lam;
            const T dr = ref[0] - Im(0, s), du = ref[1] - Im(1, s), dp = ref[4] - Im(4, s);
            if (kx == 0) { const T b = -rho / (T(2) * cs) * du + dp / (T(2) * cs * cs); wm[0] -= b; wm[1] -= b * (-cs / rho); wm[4] -= b * cs * cs; }
            else if (kx == 2) { const T b = rho / (T(2) * cs) * du + dp / (T(2) * cs * cs); wm[0] -= b; wm[1] -= b * (cs / rho); wm[4] -= b * cs * cs; }
            else { wm[0] -= dr - dp / (cs * cs); wm[2] = Im(2, s); wm[3] = Im(3, s); }
          }
        }
        const bool ok = (wp[0] > 0) && (wp[4] > 0) && (wm[0] > 0) && (wm[4] > 0) && std::isfinite(wp[0]) &&
                        std::isfinite(wp[4]) && std::isfinite(wm[0]) && std::isfinite(wm[4]);
        if (!ok) {
          if (cnt) cnt[CNT_POSITIVITY]++;
          for (int m = 0; m < 5; ++m) wp[m] = wm[m] = a[m];
        }
        for (int m = 0; m < 5; ++m) { Wp[(size_t)m * M3 + c] = wp[m]; Wm[(size_t)m * M3 + c] = wm[m]; }   // sweep order
      }
  // P5: flux through the lower d-face of every cell 0..n along d
  lo[d] = 0; hi[d] = n;
  for (int k = lo[2]; k <= hi[2]; ++k)
    for (int j = lo[1]; j <= hi[1]; ++j)
      for (int i = lo[0]; i <= hi[0]; ++i) {
        const size_t c = G.cell(i, j, k), cl = c - sd;
        T WL[5], WR[5], Fr[5];
        for (int m = 0; m < 5; ++m) { WL[m] = Wp[(size_t)m * M3 + cl]; WR[m] = Wm[(size_t)m * M3 + c]; }
        riemann_hydro<T>(WL, WR, gamma, solver, Fr, cnt);
        for (int m = 0; m < 5; ++m) F[(size_t)m * M3 + c] = Fr[m];     // (rho, m_n, m_t1, m_t2, E)
      }
  // update (interior), components back in (x, y, z) order
  for (int m = 0; m < 5; ++m) {
    const T* u = Uin + G.fld(order[m], p);
    T* un = Uout + G.fld(order[m], p);
    const T* f = F.data() + (size_t)m * M3;
    for (int k = 0; k < n; ++k)
      for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) {
          const size_t c = G.cell(i, j, k);
          un[c] = u[c] - lam * (f[c + sd] - f[c]);
        }
  }
  if (cnt)
    for (int k = 0; k < n; ++k)
      for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i)
          if (!(Uout[G.fld(0, p) + G.cell(i, j, k)] > 0)) cnt[CNT_NEG_STATE]++;
}

// O7: max over interior cells and directions of |v_d| + c_d
template <class T>
double smax_all(const T* U, const Geom& G, T gamma) {
  double best = 0;
  const int n = G.n;
#pragma omp parallel for reduction(max : best) schedule(static)
  for (int p = 0; p < G.np; ++p)
    for (int k = 0; k < n; ++k)
      for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) {
          const size_t c = G.cell(i, j, k);
          const T rho = U[G.fld(0, p) + c];
          const T v[3] = {U[G.fld(1, p) + c] / rho, U[G.fld(2, p) + c] / rho, U[G.fld(3, p) + c] / rho};
          const T E = U[G.fld(4, p) + c];
          T ke = T(0.5) * rho * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
          for (int d = 0; d < 3; ++d) {
            T cd;
            if (G.nf == 9) {
              const T B[3] = {U[G.fld(5, p) + c], U[G.fld(6, p) + c], U[G.fld(7, p) + c]};
              const T B2 = B[0] * B[0] + B[1] * B[1] + B[2] * B[2];
              const T pr = (gamma - 1) * (E - ke - T(0.5) * B2);
              const T a = (gamma * pr + B2) / rho;
              const T disc = std::max(a * a - T(4) * gamma * pr * B[d] * B[d] / (rho * rho), T(0));
              cd = std::sqrt(T(0.5) * (a + std::sqrt(disc)));
            } else {
              const T pr = (gamma - 1) * (E - ke);
              cd = std::sqrt(gamma * pr / rho);
            }
            const double sgn = (double)(std::fabs(v[d]) + cd);
            if (sgn > best) best = sgn;
          }
        }
  return best;
}

template <class T>
void totals_all(const T* U, const Geom& G, double* out) {
  const int n = G.n;
  for (int q = 0; q < G.nf; ++q) {
    long double s = 0;
    for (int p = 0; p < G.np; ++p)
      for (int k = 0; k < n; ++k)
        for (int j = 0; j < n; ++j)
          for (int i = 0; i < n; ++i) s += (long double)U[G.fld(q, p) + G.cell(i, j, k)];
    out[q] = (double)s;
  }
}

// ------------------------------------------------------------------------------------------
// O0. Ghost fill: (i) sibling copy with periodic wrap, (ii) outflow clamp; cells that neither
// rule can fill are left untouched (mask = 0) for O8.  All three layers, faces+edges+corners.
// ------------------------------------------------------------------------------------------
template <class T>
void fill_ghosts(T* U, unsigned char* mask, const Geom& G) {
  const int n = G.n, g = G.g;
  PatchMap pm(G);
#pragma omp parallel for schedule(dynamic, 1)
  for (int p = 0; p < G.np; ++p) {
    const int* o = G.origin + 3 * p;
    for (int k = -g; k < n + g; ++k)
      for (int j = -g; j < n + g; ++j)
        for (int i = -g; i < n + g; ++i) {
          const size_t c = G.cell(i, j, k);
          const bool interior = (i >= 0 && i < n && j >= 0 && j < n && k >= 0 && k < n);
          if (interior) { if (mask) mask[(size_t)p * G.M3() + c] = 1; continue; }
          int src_p = -1, li[3] = {i, j, k};
          if (G.selfp) {
            src_p = p;
            for (int d = 0; d < 3; ++d) li[d] = ((li[d] % n) + n) % n;
          } else {
            int gi[3] = {o[0] + i, o[1] + j, o[2] + k};
            for (int d = 0; d < 3; ++d) {
              if (gi[d] < 0) {
                if (G.bc[2 * d] == BC_PERIODIC) gi[d] += G.dom[d]; else gi[d] = 0;
              } else if (gi[d] >= G.dom[d]) {
                if (G.bc[2 * d + 1] == BC_PERIODIC) gi[d] -= G.dom[d]; else gi[d] = G.dom[d] - 1;
              }
            }
            src_p = pm.at(gi[0], gi[1], gi[2], n);
            if (src_p >= 0) for (int d = 0; d < 3; ++d) li[d] = gi[d] - G.origin[3 * src_p + d];
          }
          if (src_p < 0) { if (mask) mask[(size_t)p * G.M3() + c] = 0; continue; }
          const size_t cs = G.cell(li[0], li[1], li[2]);
          for (int q = 0; q < G.nf; ++q) U[G.fld(q, p) + c] = U[G.fld(q, src_p) + cs];
          if (mask) mask[(size_t)p * G.M3() + c] = 1;
        }
  }
}

template <class T>
T minmod2(T a, T b) {
  if (a > 0 && b > 0) return std::min(a, b);
  if (a < 0 && b < 0) return std::max(a, b);
  return T(0);
}

// O8. Prolongation into the fine ghost cells that O0 left unfilled (mask == 0).  Coarse state
// = (1-theta) Uold + theta Unew (interpolated first, slopes second); conserved variables, all
// fields; U_f = U_C + sum_d o_d minmod(U_C - U_{C-e_d}, U_{C+e_d} - U_C), o_d = +-1/4.
template <class T>
void prolong_ghosts(T* Uf, unsigned char* mask, const Geom& Gf, const T* Ucold, const T* Ucnew,
                    const Geom& Gc, T theta) {
  const int n = Gf.n, g = Gf.g;
  PatchMap pmc(Gc);
  const size_t cs[3] = {1, (size_t)Gc.M, (size_t)Gc.M * Gc.M};
#pragma omp parallel for schedule(dynamic, 1)
  for (int p = 0; p < Gf.np; ++p) {
    const int* o = Gf.origin + 3 * p;
    for (int k = -g; k < n + g; ++k)
      for (int j = -g; j < n + g; ++j)
        for (int i = -g; i < n + g; ++i) {
          const size_t c = Gf.cell(i, j, k);
          if (mask[(size_t)p * Gf.M3() + c]) continue;
          int gi[3] = {o[0] + i, o[1] + j, o[2] + k};
          int par[3];  // parity of the fine index inside its coarse cell
          for (int d = 0; d < 3; ++d) {
            // a ghost cell beyond a domain face: periodic -> wrapped cell (even domain: parity unchanged);
            // outflow -> O0 rule (ii): it takes the value of the clamped in-domain cell, which no fine
            // patch covers (else O0 had filled it), i.e. the prolongation AT that cell (A12/A14)
            if (gi[d] < 0) { if (Gf.bc[2 * d] == BC_PERIODIC) gi[d] += Gf.dom[d]; else gi[d] = 0; }
            else if (gi[d] >= Gf.dom[d]) { if (Gf.bc[2 * d + 1] == BC_PERIODIC) gi[d] -= Gf.dom[d]; else gi[d] = Gf.dom[d] - 1; }
            par[d] = gi[d] % 2;
          }
          const int C[3] = {gi[0] / 2, gi[1] / 2, gi[2] / 2};
          const int pc = pmc.at(C[0], C[1], C[2], Gc.n);
          const size_t cc = Gc.cell(C[0] - Gc.origin[3 * pc], C[1] - Gc.origin[3 * pc + 1],
                                    C[2] - Gc.origin[3 * pc + 2]);
          for (int q = 0; q < Gf.nf; ++q) {
            const T* a = Ucold + Gc.fld(q, pc);
            const T* b = Ucnew + Gc.fld(q, pc);
            auto st = [&](size_t idx) { return (T(1) - theta) * a[idx] + theta * b[idx]; };
            const T uc = st(cc);
            T val = uc;
            for (int d = 0; d < 3; ++d) {
              const T sl = minmod2(uc - st(cc - cs[d]), st(cc + cs[d]) - uc);
              val += (par[d] ? T(0.25) : T(-0.25)) * sl;
            }
            Uf[Gf.fld(q, p) + c] = val;
          }
          mask[(size_t)p * Gf.M3() + c] = 2;
        }
  }
}

// O9(6). Restriction: covered coarse cell <- arithmetic mean of its 8 fine cells, all fields.
template <class T>
void restrict_to_coarse(const T* Uf, const Geom& Gf, T* Uc, const Geom& Gc) {
  PatchMap pmc(Gc);
  const int n = Gf.n;
  for (int p = 0; p < Gf.np; ++p) {
    const int* o = Gf.origin + 3 * p;
    for (int k = 0; k < n; k += 2)
      for (int j = 0; j < n; j += 2)
        for (int i = 0; i < n; i += 2) {
          const int C[3] = {(o[0] + i) / 2, (o[1] + j) / 2, (o[2] + k) / 2};
          const int pc = pmc.at(C[0], C[1], C[2], Gc.n);
          const size_t cc = Gc.cell(C[0] - Gc.origin[3 * pc], C[1] - Gc.origin[3 * pc + 1],
                                    C[2] - Gc.origin[3 * pc + 2]);
          for (int q = 0; q < Gf.nf; ++q) {
            T s = 0;
            for (int dk = 0; dk < 2; ++dk)
              for (int dj = 0; dj < 2; ++dj)
                for (int di = 0; di < 2; ++di) s += Uf[Gf.fld(q, p) + Gf.cell(i + di, j + dj, k + dk)];
            Uc[Gc.fld(q, pc) + cc] = s * T(0.125);
          }
        }
  }
}

// O9(7). Reflux.  Fc = coarse flux array of the coarse step (layout of step's Fout); Ffsum =
// SUM over the two fine substeps of the fine step's Fout.  For every coarse face on a fine
// patch boundary whose outside coarse cell is not covered by a fine patch:
//   U_c += s_f (dt0/dx0) (F_coarse - (1/4)(1/2) sum_substeps sum_4 fine faces F_fine).
template <class T>
void reflux(T* Uc, const Geom& Gc, const T* Fc, const Geom& Gf, const T* Ffsum, T dt0, T dx0) {
  PatchMap pmc(Gc), pmf(Gf);
  const int n = Gf.n, nc = n / 2;
  const size_t cstr[3] = {1, (size_t)Gc.M, (size_t)Gc.M * Gc.M};
  for (int p = 0; p < Gf.np; ++p) {
    const int* o = Gf.origin + 3 * p;
    for (int d = 0; d < 3; ++d)
      for (int side = 0; side < 2; ++side) {
        const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
        for (int b = 0; b < nc; ++b)
          for (int a = 0; a < nc; ++a) {
            // coarse cell just outside the fine patch across this face
            int Cin[3];
            Cin[d] = o[d] / 2 + (side ? nc : -1);
            Cin[t1] = o[t1] / 2 + a;
            Cin[t2] = o[t2] / 2 + b;
            // a fine face on a non-periodic domain face has no coarse cell outside it: nothing to correct
            // (its flux is a boundary flux of the composite grid, A12/A14)
            if ((Cin[d] < 0 && Gc.bc[2 * d] != BC_PERIODIC) || (Cin[d] >= Gc.dom[d] && Gc.bc[2 * d + 1] != BC_PERIODIC)) continue;
            int C[3];
            for (int e = 0; e < 3; ++e) C[e] = ((Cin[e] % Gc.dom[e]) + Gc.dom[e]) % Gc.dom[e];
            // covered by a sibling fine patch?  then the face is fine-fine: no correction
            if (pmf.at(2 * C[0], 2 * C[1], 2 * C[2], Gf.n) >= 0) continue;
            const int pc = pmc.at(C[0], C[1], C[2], Gc.n);
            int lc[3] = {C[0] - Gc.origin[3 * pc], C[1] - Gc.origin[3 * pc + 1], C[2] - Gc.origin[3 * pc + 2]};
            const size_t cc = Gc.cell(lc[0], lc[1], lc[2]);
            // the shared face is the UPPER d-face of the outside cell when side == 0 (s_f = +1;
            // stored as the lower face of the next cell), the LOWER face when side == 1 (s_f = -1)
            const size_t cface = side ? cc : cc + cstr[d];
            const T sf = side ? T(-1) : T(1);
            for (int q = 0; q < Gf.nf; ++q) {
              const T Fcoarse = Fc[(((size_t)d * Gc.nf + q) * Gc.np + pc) * Gc.M3() + cface];
              T sum = 0;
              for (int bb = 0; bb < 2; ++bb)
                for (int aa = 0; aa < 2; ++aa) {
                  int lf[3];
                  lf[d] = side ? n : 0;  // fine flux through lower face of cell index n == upper face of n-1
                  lf[t1] = 2 * a + aa;
                  lf[t2] = 2 * b + bb;
                  sum += Ffsum[(((size_t)d * Gf.nf + q) * Gf.np + p) * Gf.M3() + Gf.cell(lf[0], lf[1], lf[2])];
                }
              const T Ffine = T(0.25) * T(0.5) * sum;
              Uc[Gc.fld(q, pc) + cc] += sf * (dt0 / dx0) * (Fcoarse - Ffine);
            }
          }
      }
  }
}

// Composite total (O9): sum over uncovered coarse cells * dx0^3 + sum over fine cells * dx1^3
template <class T>
void composite_totals(const T* Uc, const Geom& Gc, const T* Uf, const Geom& Gf, double dx0, double* out) {
  PatchMap pmf(Gf);
  const double v0 = dx0 * dx0 * dx0, v1 = v0 / 8.0;
  for (int q = 0; q < Gc.nf; ++q) {
    long double s = 0;
    for (int p = 0; p < Gc.np; ++p)
      for (int k = 0; k < Gc.n; ++k)
        for (int j = 0; j < Gc.n; ++j)
          for (int i = 0; i < Gc.n; ++i) {
            const int* o = Gc.origin + 3 * p;
            if (pmf.at(2 * (o[0] + i), 2 * (o[1] + j), 2 * (o[2] + k), Gf.n) >= 0) continue;
            s += (long double)Uc[Gc.fld(q, p) + Gc.cell(i, j, k)] * v0;
          }
    for (int p = 0; p < Gf.np; ++p)
      for (int k = 0; k < Gf.n; ++k)
        for (int j = 0; j < Gf.n; ++j)
          for (int i = 0; i < Gf.n; ++i) s += (long double)Uf[Gf.fld(q, p) + Gf.cell(i, j, k)] * v1;
    out[q] = (double)s;
  }
}

Geom make_geom(int np, int n, int g, int nf, const int* origin, const int* dom, const int* bc, int selfp) {
  Geom G;
  G.np = np; G.n = n; G.g = g; G.nf = nf; G.M = n + 2 * g; G.origin = origin;
  for (int d = 0; d < 3; ++d) G.dom[d] = dom ? dom[d] : n;
  for (int d = 0; d < 6; ++d) G.bc[d] = bc ? bc[d] : BC_PERIODIC;
  G.selfp = selfp;
  return G;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// C-ABI of the oracle (prefix oracle_).  dtype: 0 = float32, 1 = float64.
// ------------------------------------------------------------------------------------------
extern "C" {

int oracle_step(int dtype, const void* Uin, void* Uout, void* Fout, void* FSout, int np, int n, int g,
                int nf, double dt, double dx, double gamma, int limiter, int riemann, double ch,
                double alpha, double eps, long long* counters) {
  if (n < 4 || g < 2 || (nf != 5 && nf != 9)) return -1;
  Geom G = make_geom(np, n, g, nf, nullptr, nullptr, nullptr, 0);
  if (dtype == 1) {
    StepParams<double> P{dt, dx, gamma, ch, alpha, eps, limiter, riemann};
    return step_all<double>((const double*)Uin, (double*)Uout, (double*)Fout, (double*)FSout, G, P, counters);
  }
  StepParams<float> P{(float)dt, (float)dx, (float)gamma, (float)ch, (float)alpha, (float)eps, limiter, riemann};
  return step_all<float>((const float*)Uin, (float*)Uout, (float*)Fout, (float*)FSout, G, P, counters);
}

double oracle_smax(int dtype, const void* U, int np, int n, int g, int nf, double gamma) {
  Geom G = make_geom(np, n, g, nf, nullptr, nullptr, nullptr, 0);
  return dtype == 1 ? smax_all<double>((const double*)U, G, gamma) : smax_all<float>((const float*)U, G, (float)gamma);
}

void oracle_totals(int dtype, const void* U, int np, int n, int g, int nf, double* out) {
  Geom G = make_geom(np, n, g, nf, nullptr, nullptr, nullptr, 0);
  if (dtype == 1) totals_all<double>((const double*)U, G, out); else totals_all<float>((const float*)U, G, out);
}

int oracle_fill_ghosts(int dtype, void* U, unsigned char* mask, int np, int n, int g, int nf,
                       const int* origin, const int* dom, const int* bc, int selfp) {
  Geom G = make_geom(np, n, g, nf, origin, dom, bc, selfp);
  if (dtype == 1) fill_ghosts<double>((double*)U, mask, G); else fill_ghosts<float>((float*)U, mask, G);
  return 0;
}

int oracle_prolong_ghosts(int dtype, void* Uf, unsigned char* mask, int npf, int n, int g, int nf,
                          const int* originf, const int* domf, const void* Ucold, const void* Ucnew,
                          int npc, const int* originc, const int* domc, double theta, const int* bc) {
  Geom Gf = make_geom(npf, n, g, nf, originf, domf, bc, 0);
  Geom Gc = make_geom(npc, n, g, nf, originc, domc, bc, 0);
  if (dtype == 1) prolong_ghosts<double>((double*)Uf, mask, Gf, (const double*)Ucold, (const double*)Ucnew, Gc, theta);
  else prolong_ghosts<float>((float*)Uf, mask, Gf, (const float*)Ucold, (const float*)Ucnew, Gc, (float)theta);
  return 0;
}

int oracle_restrict(int dtype, const void* Uf, int npf, int n, int g, int nf, const int* originf,
                    const int* domf, void* Uc, int npc, const int* originc, const int* domc) {
  Geom Gf = make_geom(npf, n, g, nf, originf, domf, nullptr, 0);
  Geom Gc = make_geom(npc, n, g, nf, originc, domc, nullptr, 0);
  if (dtype == 1) restrict_to_coarse<double>((const double*)Uf, Gf, (double*)Uc, Gc);
  else restrict_to_coarse<float>((const float*)Uf, Gf, (float*)Uc, Gc);
  return 0;
}

int oracle_reflux(int dtype, void* Uc, int npc, int n, int g, int nf, const int* originc, const int* domc,
                  const void* Fc, int npf, const int* originf, const int* domf, const void* Ffsum,
                  double dt0, double dx0, const int* bc) {
  Geom Gf = make_geom(npf, n, g, nf, originf, domf, bc, 0);
  Geom Gc = make_geom(npc, n, g, nf, originc, domc, bc, 0);
  if (dtype == 1) reflux<double>((double*)Uc, Gc, (const double*)Fc, Gf, (const double*)Ffsum, dt0, dx0);
  else reflux<float>((float*)Uc, Gc, (const float*)Fc, Gf, (const float*)Ffsum, (float)dt0, (float)dx0);
  return 0;
}

void oracle_composite_totals(int dtype, const void* Uc, int npc, int n, int g, int nf, const int* originc,
                             const int* domc, const void* Uf, int npf, const int* originf,
                             const int* domf, double dx0, double* out) {
  Geom Gf = make_geom(npf, n, g, nf, originf, domf, nullptr, 0);
  Geom Gc = make_geom(npc, n, g, nf, originc, domc, nullptr, 0);
  if (dtype == 1) composite_totals<double>((const double*)Uc, Gc, (const double*)Uf, Gf, dx0, out);
  else composite_totals<float>((const float*)Uc, Gc, (const float*)Uf, Gf, dx0, out);
}

// One PPM sweep (hydro, nf = 5) along direction d of every patch; Uout's ghosts are the caller's.
int oracle_ppm_sweep(int dtype, const void* Uin, void* Uout, int np, int n, int g, int nf, int d, double dt,
                     double dx, double gamma, int riemann, long long* counters) {
  if (nf != 5 || g < 3 || n < 4 || d < 0 || d > 2 || (riemann != RS_HLL && riemann != RS_HLLC)) return -1;
  Geom G = make_geom(np, n, g, nf, nullptr, nullptr, nullptr, 0);
  const size_t M3 = G.M3();
  long long tot[4] = {0, 0, 0, 0};
  auto run = [&](auto tag) {
    using T = decltype(tag);
    const T* in = (const T*)Uin;
    T* out = (T*)Uout;
#pragma omp parallel
    {
      std::vector<T> W(5 * M3), Wm(5 * M3), Wp(5 * M3), F(5 * M3);
      long long cnt[4] = {0, 0, 0, 0};
#pragma omp for schedule(dynamic, 1)
      for (int p = 0; p < np; ++p)
        ppm_sweep_patch<T>(in, out, G, p, d, (T)dt, (T)dx, (T)gamma, riemann, W, Wm, Wp, F, cnt);
#pragma omp critical
      for (int q = 0; q < 4; ++q) tot[q] += cnt[q];
    }
  };
  if (dtype == 1) run(double(0)); else run(float(0));
  if (counters) for (int q = 0; q < 4; ++q) counters[q] = tot[q];
  return 0;
}

// P1 + P2 of one cell from its five-point stencil (pins of the reconstruction)
void oracle_ppm_parabola(const double* a5, double* aL, double* aR) {
  ppm_parabola<double>(a5[0], a5[1], a5[2], a5[3], a5[4], aL, aR);
}

// Single-face Riemann solvers (fp64) for the pins P7/P8.  nf = 5: hydro; nf = 9: MHD.
int oracle_riemann(int nf, const double* WL, const double* WR, double gamma, double ch, int solver,
                   double eps, double* F, long long* counters) {
  long long cnt[4] = {0, 0, 0, 0};
  if (nf == 5) riemann_hydro<double>(WL, WR, gamma, solver, F, cnt);
  else riemann_mhd<double>(WL, WR, gamma, ch, solver, eps, F, cnt, nullptr);
  if (counters) for (int q = 0; q < 4; ++q) counters[q] = cnt[q];
  return 0;
}

// HLLD intermediate states: out = [S(5) | U(6x7) | FL(7) | FR(7) | ptstar | Bn | path] = 64 doubles
int oracle_hlld_states(const double* WL, const double* WR, double gamma, double ch, double eps, double* F,
                       double* out) {
  HlldDebug<double> dbg;
  std::memset(&dbg, 0, sizeof(dbg));
  riemann_mhd<double>(WL, WR, gamma, ch, RS_HLLD, eps, F, nullptr, &dbg);
  int o = 0;
  for (int q = 0; q < 5; ++q) out[o++] = dbg.S[q];
  for (int s = 0; s < 6; ++s) for (int q = 0; q < 7; ++q) out[o++] = dbg.U[s][q];
  for (int q = 0; q < 7; ++q) out[o++] = dbg.FL[q];
  for (int q = 0; q < 7; ++q) out[o++] = dbg.FR[q];
  out[o++] = dbg.ptstar; out[o++] = dbg.Bn; out[o++] = (double)dbg.path;
  return o;
}

double oracle_limited_slope(double a, double b, int lim) { return limited_slope<double>(a, b, lim); }

// thread count of the OpenMP loops over patches (timing of the CPU baseline on 1 core / all cores; no arithmetic)
void oracle_set_num_threads(int nt) {
#ifdef _OPENMP
  if (nt > 0) omp_set_num_threads(nt);
#else
  (void)nt;
#endif
}

int oracle_num_threads(void) {
  int nt = 1;
#ifdef _OPENMP
#pragma omp parallel
  {
#pragma omp single
    nt = omp_get_num_threads();
  }
#endif
  return nt;
}

}  // extern "C"

// Fused per-tile Godunov step for sm_100a, fp64, one cell per thread, with the STRUCTURE of the fp32 x2 kernel
// (godunov_step_x2.cuh): warp-specialised compute / aux loops, three-plane ring of primitives filled by 8-byte
// cp.async, branch-free Riemann solvers (riemann_x2.cuh instantiated for double), and every face state that
// has to survive a phase staged in a private shared-memory column instead of registers.
// O0 halo assembly -> O1 primitives -> O2 slopes -> O3 predictor -> O4 face states -> O5 Riemann flux -> O6
// update -> O7 signal speed, one pass.
//
// Why (profiles/r1c fp64): the first fp64 kernel (godunov_step.cuh: register-resident face states, branchy
// solvers, all threads loading) spills 592 B per thread at the 168 registers two CTAs per SM allow
// (long_scoreboard 1.56 per issue: with 214 KB of shared memory in use there is no L1 left for the spills) and
// spends 13 % of its instructions on 32-bit halves of fp64 register moves around its role branches.
//
// Work decomposition: one CTA owns an HX x TY column of cells of one patch and marches along z.  HX * TY compute
// threads (whole warps) + aux warps holding the ring of the tile grown by one layer (no corners: right / left
// column, bottom / top row) and doing all loading.  Shared memory ("records" = the NF doubles of a cell, padded
// to 10 / 6 doubles so that 128-bit accesses of consecutive lanes are bank-conflict free):
//   ring   three planes of primitives on the tile + radius-2 halo; raw conserved values of plane k+2 arrive by
//          cp.async in the slot plane k-1 vacated and are converted in place by the aux thread that copied them
//   XL/YL  per x / y face: W^+ of the cell left of / below it, then the face's flux
//   UO     (m, E) of the cell awaiting its update      SCR  private staging: W^+_z of the previous plane;
//          W^-_x, W^-_y for phase 2; the own x / y fluxes for phase 3
// Per plane, two barriers, as in the x2 kernel.  Every face flux is computed once per tile by one
// position-independent routine from bit-identical inputs (conservation to round-off).
#pragma once
#include <cstdio>
#include <cuda_runtime.h>

#include "amr_internal.hpp"
#include "riemann_x2.cuh"
#include "signal_speed.cuh"

namespace amr {
namespace d1 {

using x2::RCD;
enum { D1_LIM_NONE = 0, D1_LIM_MINMOD = 1, D1_LIM_MC = 2 };
enum { D1_CNT_POSITIVITY = 0, D1_CNT_NEG_STATE = 3 };

// O2 as HALF slopes, sign-test form on magnitudes (fp64 has no min/max instruction; see godunov_step.cuh)
template <int LIM>
__device__ __forceinline__ double half_slope(double a, double b) {
  if (LIM == D1_LIM_NONE) return 0.0;
  const bool same = (__double2hiint(a) ^ __double2hiint(b)) >= 0;
  const double aa = fabs(a), ab = fabs(b);
  double m = aa < ab ? aa : ab;
  if (LIM == D1_LIM_MC) {
    const double aq = fabs(0.25 * (a + b));
    m = m < aq ? m : aq;
  } else {
    m = 0.5 * m;
  }
  return same ? copysign(m, a) : 0.0;
}

// a record of N doubles <-> registers, 128-bit accesses (N odd: last one 64-bit)
template <int N>
__device__ __forceinline__ void lds_rec(const double* p, double* o) {
#pragma unroll
  for (int i = 0; i < N / 2; ++i) {
    const double2 v = *reinterpret_cast<const double2*>(p + 2 * i);
    o[2 * i] = v.x; o[2 * i + 1] = v.y;
  }
  if constexpr (N & 1) o[N - 1] = p[N - 1];
}
template <int N>
__device__ __forceinline__ void sts_rec(double* p, const double* o) {
#pragma unroll
  for (int i = 0; i < N / 2; ++i) *reinterpret_cast<double2*>(p + 2 * i) = make_double2(o[2 * i], o[2 * i + 1]);
  if constexpr (N & 1) p[N - 1] = o[N - 1];
}

__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int NF, int HX, int TY>
struct GeomD1 {
  static constexpr int NPX = HX + 4;                // columns of a ring row (two halo cells each side)
  static constexpr int RH = TY + 4;                 // ring rows
  static constexpr int REC = NF == 9 ? 10 : 6;      // doubles per record
  static constexpr int SLOT = RH * NPX * REC;       // doubles per ring plane
  static constexpr int NSLOT = 3;
  static constexpr int BLK = REC / 2;               // double2 per staging block (one record)
  static constexpr int NSCR = 3 * BLK;              // double2 of private staging per compute thread
  static constexpr int NI = HX * TY;                // compute threads
  static constexpr int NPRED = NI + 2 * TY + 2 * HX;
  static constexpr int NXL = TY * (HX + 1);
  static constexpr int NYL = (TY + 1) * HX;
  static constexpr int NCHUNK = RH * NPX;
  static constexpr size_t smem_doubles = (size_t)NSLOT * SLOT + (size_t)(NXL + NYL) * REC + (size_t)NI * 4 + (size_t)NSCR * NI * 2;
  static constexpr size_t smem_bytes = smem_doubles * sizeof(double);
};

// rotated component order handed to the 1-D Riemann routine: x -> (x,y,z), y -> (y,z,x), z -> (z,x,y)
template <int NF, int D>
__device__ __forceinline__ void rot_in(const double* w, double* r) {
  constexpr int qn = 1 + D, q1 = 1 + (D + 1) % 3, q2 = 1 + (D + 2) % 3;
  r[0] = w[0]; r[1] = w[qn]; r[2] = w[q1]; r[3] = w[q2]; r[4] = w[4];
  if (NF == 9) { r[5] = w[4 + qn]; r[6] = w[4 + q1]; r[7] = w[4 + q2]; r[8] = w[8]; }
}
template <int NF, int D>
__device__ __forceinline__ void rot_out(const double* r, double* f) {
  constexpr int qn = 1 + D, q1 = 1 + (D + 1) % 3, q2 = 1 + (D + 2) % 3;
  f[0] = r[0]; f[qn] = r[1]; f[q1] = r[2]; f[q2] = r[3]; f[4] = r[4];
  if (NF == 9) { f[4 + qn] = r[5]; f[4 + q1] = r[6]; f[4 + q2] = r[7]; f[8] = r[8]; }
}

// O2 + O3 + O4 for the cell whose ring record is at element offset rc: half slopes hx, hy, hz, predicted state
// ws.  A cell that fails the positivity test (A10) gets ws = W and zero slopes; returns 1 for such a cell.
template <int NF, int LIM>
__device__ __forceinline__ int predict_cell(const double* Wm, const double* Wc, const double* Wp, int rc, int rowstride,
                                            int recstride, const StepParams<double>& P, double* ws,
                                            double* hx, double* hy, double* hz) {
  double w[NF];
  {
    const double* cc = Wc + rc;
    double a[NF], b[NF];
    lds_rec<NF>(cc, w);
    lds_rec<NF>(cc - recstride, a);
    lds_rec<NF>(cc + recstride, b);
#pragma unroll
    for (int q = 0; q < NF; ++q) hx[q] = half_slope<LIM>(w[q] - a[q], b[q] - w[q]);
    lds_rec<NF>(cc - rowstride, a);
    lds_rec<NF>(cc + rowstride, b);
#pragma unroll
    for (int q = 0; q < NF; ++q) hy[q] = half_slope<LIM>(w[q] - a[q], b[q] - w[q]);
    lds_rec<NF>(Wm + rc, a);
    lds_rec<NF>(Wp + rc, b);
#pragma unroll
    for (int q = 0; q < NF; ++q) hz[q] = half_slope<LIM>(w[q] - a[q], b[q] - w[q]);
  }
  // O3 predictor with half slopes: W* = W - (dt/dx) sum_d A_d h_d
  const double s = P.dtdx;
  const double rho = w[0], pr = w[4];
  const double ir = fast_rcp(rho);
#define ADV(q) (w[1] * hx[q] + w[2] * hy[q] + w[3] * hz[q])
  const double divv = hx[1] + hy[2] + hz[3];
  ws[0] = rho - s * (ADV(0) + rho * divv);
  if (NF == 5) {
    ws[1] = w[1] - s * (ADV(1) + hx[4] * ir);
    ws[2] = w[2] - s * (ADV(2) + hy[4] * ir);
    ws[3] = w[3] - s * (ADV(3) + hz[4] * ir);
    ws[4] = pr - s * (ADV(4) + P.gamma * pr * divv);
  } else {
#define BGRAD(q) (w[5] * hx[q] + w[6] * hy[q] + w[7] * hz[q])
    const double divB = hx[5] + hy[6] + hz[7];
    const double vB = w[1] * w[5] + w[2] * w[6] + w[3] * w[7];
    const double BdBx = w[5] * hx[5] + w[6] * hx[6] + w[7] * hx[7];
    const double BdBy = w[5] * hy[5] + w[6] * hy[6] + w[7] * hy[7];
    const double BdBz = w[5] * hz[5] + w[6] * hz[6] + w[7] * hz[7];
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
  const double hr = x2::max3(fabs(hx[0]), fabs(hy[0]), fabs(hz[0]));
  const double hp = x2::max3(fabs(hx[4]), fabs(hy[4]), fabs(hz[4]));
  const bool ok = (ws[0] - hr > 0.0) && (ws[4] - hp > 0.0) && (ws[0] + hr < CUDART_INF) && (ws[4] + hp < CUDART_INF);
  if (X2_UNLIKELY(!ok)) {
#pragma unroll
    for (int q = 0; q < NF; ++q) { ws[q] = w[q]; hx[q] = 0.0; hy[q] = 0.0; hz[q] = 0.0; }
    return 1;
  }
  return 0;
}

template <int NF, int LIM, int RS, int HX, int TY, int NT, int MAXR>
__global__ void __maxnreg__(MAXR) godunov_step_d1_kernel(const __grid_constant__ StepParams<double> P) {
  using G = GeomD1<NF, HX, TY>;
  constexpr int NPX = G::NPX, RH = G::RH, REC = G::REC, SLOT = G::SLOT, NI = G::NI, NPRED = G::NPRED, NCHUNK = G::NCHUNK;
  constexpr int NA = NT - NI;                 // aux threads: ring cells + the plane loader
  constexpr int LC = (NCHUNK + NA - 1) / NA;  // loader cells of one ring plane per aux thread
  constexpr int BLK = G::BLK, BZ = 0, BX = BLK, BY = 2 * BLK, NFULL = (NF - 1) / 2;
  static_assert(NI % 32 == 0 && NT % 32 == 0 && NT >= NPRED, "compute warps = interior cells; aux warps hold the ring");
  static_assert(LC <= 8, "loader masks");

  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* const ring = reinterpret_cast<double*>(smem_raw);  // [3][RH][NPX][REC]
  double* const XL = ring + G::NSLOT * SLOT;                 // [TY][HX+1][REC]
  double* const YL = XL + G::NXL * REC;                      // [TY+1][HX][REC]
  double* const UO = YL + G::NYL * REC;                      // [2][NI][2]: (m_x, m_y | m_z, E)
  double2* const SCR = reinterpret_cast<double2*>(UO + NI * 4);  // [NSCR][NI] double2
  __shared__ int s_nbr[27];
  __shared__ int s_cnt[4];
  __shared__ double s_red[NI / 32];

  const int tid = threadIdx.x;
  const int n = P.n;
  int bb = blockIdx.x;
  const int tpp = P.ntx * P.nty;
  const int p = bb / tpp;
  bb -= p * tpp;
  const int ty = bb / P.ntx, tx = bb - ty * P.ntx;
  const int x0 = tx * HX, y0 = ty * TY;
  const int zc = n;  // the whole z extent of the patch (ntz = 1)

  if (tid < 27) s_nbr[tid] = P.nbr[p * 27 + tid];
  if (tid < 4) s_cnt[tid] = 0;
  __syncthreads();

  const int n2 = n * n;
  const int n3 = n2 * n;  // host guarantees np * (n+2g)^3 < 2^31
  const size_t fs_int = (size_t)P.np * n3;

  RCD RC;
  RC.gamma = P.gamma; RC.igm1 = P.igm1; RC.ch2 = P.ch2; RC.half_ch = 0.5 * P.ch; RC.half_ich = P.half_ich;
  RC.eps = P.eps;
  const int blk = (P.fblk != nullptr) ? P.fblk_of[p] : -1;  // flux-register block of this patch
  // flux blocks: [block][direction][field][3 face planes: index 0, n/2, n along the normal][n^2 in-plane, the
  // lower remaining axis fastest]
  const size_t fsz = (size_t)3 * n2;

  double* Wm = ring;
  double* Wc = ring + SLOT;
  double* Wp = ring + 2 * SLOT;

  if (tid < NI) {
    // =================================== compute warps: interior cells ===================================
    const int pj = tid / HX, pc = tid - pj * HX;
    const int rc = ((pj + 2) * NPX + pc + 2) * REC;              // ring record of this cell
    double* const xpub = XL + (pj * (HX + 1) + pc + 1) * REC;    // W^+_x for the right neighbour, then its x flux
    double* const xsol = xpub - REC;                             // left state of this cell's lower x face, then its flux
    double* const ypub = YL + ((pj + 1) * HX + pc) * REC;        // W^+_y for the cell above, then its y flux
    double* const ysol = ypub - HX * REC;
    const int cell0 = p * n3 + (y0 + pj) * n + (x0 + pc);
    double* const uo = UO + tid * 2;
    // private staging column (double2 j of thread tid at SCR[j*NI + tid]); blocks of BLK double2 = one record:
    //   BZ  W^+_z of the previous plane     BX  W^-_x, after the x solve the x flux     BY  likewise for y
    double2* const sc = SCR + tid;
    auto st_block = [&](int j0, const double* a) {
#pragma unroll
      for (int i = 0; i < NFULL; ++i) sc[(j0 + i) * NI] = make_double2(a[2 * i], a[2 * i + 1]);
      sc[(j0 + NFULL) * NI] = make_double2(a[NF - 1], 0.0);
    };
    auto ld_block = [&](int j0, double* a) {
#pragma unroll
      for (int i = 0; i < NFULL; ++i) { const double2 v = sc[(j0 + i) * NI]; a[2 * i] = v.x; a[2 * i + 1] = v.y; }
      a[NF - 1] = sc[(j0 + NFULL) * NI].x;
    };
    double dU[NF];    // flux sum of the plane whose update is pending: ((Fx+ - Fx-) + (Fy+ - Fy-)) - Fz-
    double smax_loc = 0.0;
    int npos = 0;
#pragma unroll
    for (int q = 0; q < NF; ++q) dU[q] = 0.0;
    {
      double z[NF];
#pragma unroll
      for (int q = 0; q < NF; ++q) z[q] = 0.0;
      st_block(BZ, z);
    }
    __syncthreads();  // the aux warps have staged and converted planes -2, -1, 0

    for (int t = 0; t <= zc + 1; ++t) {
      const int kk = t - 1;                    // plane being predicted
      const bool mid = (t >= 1) && (t <= zc);  // kk is a plane of this patch (x/y fluxes needed)

      // ---- phase 1: slopes, predictor, face states; z face; update of plane kk-1 --------------------
      {
        double WL[NF], WR[NF];
        {
          double ws[NF], hx[NF], hy[NF], hz[NF], o[NF];
          const int nb = predict_cell<NF, LIM>(Wm, Wc, Wp, rc, NPX * REC, REC, P, ws, hx, hy, hz);
          if (mid) {
            npos += nb;
#pragma unroll
            for (int q = 0; q < NF; ++q) o[q] = ws[q] + hx[q];
            sts_rec<NF>(xpub, o);
            // everything the y solve reads or writes travels in its rotated component order (y, z, x), so that
            // phase 2 runs ONE solver instance over both directions (the kernel is bound by instruction fetch:
            // profiles/r1f)
            double r[NF];
#pragma unroll
            for (int q = 0; q < NF; ++q) o[q] = ws[q] + hy[q];
            rot_in<NF, 1>(o, r);
            sts_rec<NF>(ypub, r);
#pragma unroll
            for (int q = 0; q < NF; ++q) o[q] = ws[q] - hx[q];
            st_block(BX, o);
#pragma unroll
            for (int q = 0; q < NF; ++q) o[q] = ws[q] - hy[q];
            rot_in<NF, 1>(o, r);
            st_block(BY, r);
          }
          // z direction: left state of the face below = W^+_z of the previous plane (scratch), then this
          // plane's W^+_z takes its place
          ld_block(BZ, o);
          rot_in<NF, 2>(o, WL);
#pragma unroll
          for (int q = 0; q < NF; ++q) o[q] = ws[q] + hz[q];
          st_block(BZ, o);
#pragma unroll
          for (int q = 0; q < NF; ++q) o[q] = ws[q] - hz[q];
          rot_in<NF, 2>(o, WR);
        }
        if (t >= 1) {  // z face between planes kk-1 and kk
          double fz[NF];
          {
            double Fr[NF];
            x2::riemann2<NF, RS>(WL, WR, RC, Fr, true, s_cnt);
            rot_out<NF, 2>(Fr, fz);
          }
          // flux registers of a coarse-fine link (a7).  Only the face planes a link can read are recorded: index 0,
          // n/2, n along the normal (fine patches sit on aligned (n/2)^3 blocks of the parent level)
          if (X2_UNLIKELY(blk >= 0) && (kk == 0 || kk == (n >> 1) || kk == n)) {
            double* dstF = P.fblk + ((size_t)blk * 3 + 2) * NF * fsz + ((size_t)((kk) == 0 ? 0 : ((kk) == n ? 2 : 1)) * n2 + (size_t)((y0 + pj) * n + (x0 + pc)));
#pragma unroll
            for (int q = 0; q < NF; ++q) atomicAdd(dstF + (size_t)q * fsz, fz[q]);
          }
          if (t >= 2) {  // O6 for plane kk-1, GLM damping, O7 of the new state
            // U_old: rho, B, psi are the ring record of plane kk-1 (conversion leaves them untouched), (m, E)
            // were staged in phase 2 of the previous iteration
            double un[NF];
            const double* om = Wm + rc;
            un[0] = om[0];
            if (NF == 9) {
              un[5] = om[5];
              const double2 b67 = *reinterpret_cast<const double2*>(om + 6);
              un[6] = b67.x; un[7] = b67.y; un[8] = om[8];
            }
            {
              const double2 v0 = *reinterpret_cast<const double2*>(uo), v1 = *reinterpret_cast<const double2*>(uo + NI * 2);
              un[1] = v0.x; un[2] = v0.y; un[3] = v1.x; un[4] = v1.y;
            }
#pragma unroll
            for (int q = 0; q < NF; ++q) un[q] = un[q] - P.dtdx * (dU[q] + fz[q]);
            if (NF == 9) un[8] *= P.damp;
            double* out = P.Uout + (cell0 + (kk - 1) * n2);
#pragma unroll
            for (int q = 0; q < NF; ++q) out[q * fs_int] = un[q];
            if (X2_UNLIKELY(!(un[0] > 0.0))) atomicAdd(&s_cnt[D1_CNT_NEG_STATE], 1);
            const double sp = signal_speed<double, NF>(un, P.gamma, P.gm1);
            smax_loc = sp > smax_loc ? sp : smax_loc;   // a NaN speed is dropped
          }
#pragma unroll
          for (int q = 0; q < NF; ++q) dU[q] = -fz[q];
        }
      }
      if (t == zc + 1) break;
      __syncthreads();

      // ---- phase 2: copy of (m, E) of plane kk for its update in the next iteration; the x and y Riemann
      //      problems at this cell's lower faces --------------------------------------------------------
      if (mid) {
        const double* src = P.Uin + (cell0 + kk * n2);
        cp_async8(uo, src + fs_int);
        cp_async8(uo + 1, src + 2 * fs_int);
        cp_async8(uo + NI * 2, src + 3 * fs_int);
        cp_async8(uo + NI * 2 + 1, src + 4 * fs_int);
      }
      cp_commit();
      if (mid) {
        // d = 0: the x face left of this cell; d = 1: the y face below it.  One solver instance; inputs and
        // outputs in the solver's component order (identity for x, rotated for y).
#pragma unroll 1
        for (int d = P.ntz - 1; d < 2; ++d) {   // ntz == 1: an opaque lower bound keeps the loop from being unrolled
          double* const rec = d ? ysol : xsol;
          const int bj = d ? BY : BX;
          double WL[NF], WR[NF], Fr[NF];
          lds_rec<NF>(rec, WL);
          ld_block(bj, WR);
          x2::riemann2<NF, RS>(WL, WR, RC, Fr, true, s_cnt);
          sts_rec<NF>(rec, Fr);       // for the left / lower neighbour's phase 3
          st_block(bj, Fr);           // private copy for this thread's phase 3 (the neighbour overwrites rec in ITS
                                      // next phase 1, with no barrier in between)
          const int fidx = d ? y0 + pj : x0 + pc;   // face index along the normal
          if (X2_UNLIKELY(blk >= 0) && (fidx == 0 || fidx == (n >> 1))) {  // record the flux for the reflux
            double f[NF];
            if (d) rot_out<NF, 1>(Fr, f); else rot_out<NF, 0>(Fr, f);
            double* dstF = P.fblk + ((size_t)blk * 3 + d) * NF * fsz +
                           (size_t)((fidx) == 0 ? 0 : ((fidx) == n ? 2 : 1)) * n2 + (size_t)(kk * n + (d ? x0 + pc : y0 + pj));
#pragma unroll
            for (int q = 0; q < NF; ++q) atomicAdd(dstF + (size_t)q * fsz, f[q]);
          }
        }
      }
      cp_wait<0>();
      __syncthreads();

      // ---- phase 3: x/y flux differences of plane kk -> registers (own fluxes from the private scratch, the
      //      right neighbour's and the upper cell's from the slots this thread overwrites next) ---------
      if (mid) {
        double xr[NF], fu[NF], fx[NF], fy[NF];
        lds_rec<NF>(xpub, xr);
        lds_rec<NF>(ypub, fu);
        ld_block(BX, fx);
        ld_block(BY, fy);
#pragma unroll
        for (int q = 0; q < NF; ++q) fu[q] = fu[q] - fy[q];   // (rotated order)
        rot_out<NF, 1>(fu, fy);
#pragma unroll
        for (int q = 0; q < NF; ++q) dU[q] = ((xr[q] - fx[q]) + fy[q]) + dU[q];
      }
      double* tmp = Wm; Wm = Wc; Wc = Wp; Wp = tmp;
    }

    // ---- epilogue: max signal speed of the new state (O7), event counters -------------------------
    if (npos) atomicAdd(&s_cnt[D1_CNT_POSITIVITY], npos);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double v = __shfl_xor_sync(0xffffffffu, smax_loc, o);
      smax_loc = v > smax_loc ? v : smax_loc;
    }
    if ((tid & 31) == 0) s_red[tid >> 5] = smax_loc;
  } else {
    // ======================= aux warps: plane loader (O0, O1) and the ring of the tile =======================
    const int at = tid - NI;
    const int M = n + 2 * P.g;
    const int M2 = M * M;
    const size_t fs_halo = (size_t)P.np * M2 * M;

    // ---- plane loader: raw conserved values of plane lz -> ring slot, asynchronously ----------------
    // ring cell c = ry*NPX + cx <-> patch-local (lx, ly) = (x0 + cx - 2, y0 + ry - 2); cells outside the
    // stencil footprint (corners) are never touched.  Per z region the source of a cell is fixed up to the
    // z term, so its offset is resolved once per region: goff = element offset of (source patch, z = 0, sy,
    // sx); hmask: the source is the prolongation halo; zmask: the z index is clamped (outflow).
    unsigned lmask = 0;
#pragma unroll
    for (int l = 0; l < LC; ++l) {
      const int c = at + l * NA;
      if (c < NCHUNK) {
        const int ry = c / NPX, cx = c - ry * NPX;
        const int hx = cx < 2 ? 2 - cx : (cx >= HX + 2 ? cx - (HX + 1) : 0);
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
          const int c = at + l * NA;
          const int ry = c / NPX, cx = c - ry * NPX;
          const int lx = x0 + cx - 2, ly = y0 + ry - 2;
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
    // the lines issue_plane(lz) is going to copy, asked for in the L2 at the end of phase 1 (see godunov_step_x2.cuh): one
    // thread per (ring row, run of the row: left halo cells / interior / right halo cells); a hint, clamped runs skipped
    const int pf_ry = at / 3, pf_run = at - 3 * pf_ry;
    const bool pf_on = pf_ry < RH && !((pf_ry < 2 || pf_ry >= RH - 2) && pf_run != 1);
    auto prefetch_plane = [&](int lz) {
      if (pf_on) {
        const int rz = lz < 0 ? 0 : (lz >= n ? 2 : 1);
        const int lx = pf_run == 0 ? x0 - 2 : (pf_run == 1 ? x0 : x0 + HX), ly = y0 + pf_ry - 2;
        const int gx = lx < 0 ? 0 : (lx >= n ? 2 : 1), gy = ly < 0 ? 0 : (ly >= n ? 2 : 1);
        const int e = s_nbr[rz * 9 + gy * 3 + gx];
        if (e >= 0 && (e >> NBR_MODE_SHIFT) == 0) {
          const double* src = P.Uin + ((e & NBR_PATCH_MASK) * n3 + (lz - (rz - 1) * n) * n2 + (ly - (gy - 1) * n) * n + (lx - (gx - 1) * n));
#pragma unroll
          for (int q = 0; q < NF; ++q) asm volatile("prefetch.global.L2 [%0];" ::"l"(src + q * fs_int));
        } else if (e < 0) {
          const double* src = P.halo + (p * (M2 * M) + (lz + P.g) * M2 + (ly + P.g) * M + (lx + P.g));
#pragma unroll
          for (int q = 0; q < NF; ++q) asm volatile("prefetch.global.L2 [%0];" ::"l"(src + q * fs_halo));
        }
      }
    };
    auto issue_plane = [&](int lz, double* dst) {
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
          const double* src = (fh ? P.halo : P.Uin) + off;
          const size_t fs = fh ? fs_halo : fs_int;
          double* d = dst + (at + l * NA) * REC;
#pragma unroll
          for (int q = 0; q < NF; ++q) cp_async8(d + q, src + q * fs);
        }
      }
    };
    // O1 in place: conserved -> primitive, each thread on the cells it copied
    auto convert_plane = [&](double* dst) {
#pragma unroll
      for (int l = 0; l < LC; ++l) {
        if (lmask & (1u << l)) {
          double* d = dst + (at + l * NA) * REC;
          double u[NF];
          lds_rec<NF>(d, u);
          const double ir = fast_rcp(u[0]);
          const double vx = u[1] * ir, vy = u[2] * ir, vz = u[3] * ir;
          double e_int = u[4] - 0.5 * u[0] * (vx * vx + vy * vy + vz * vz);
          if (NF == 9) e_int -= 0.5 * (u[5] * u[5] + u[6] * u[6] + u[7] * u[7]);
          d[1] = vx;
          *reinterpret_cast<double2*>(d + 2) = make_double2(vy, vz);
          d[4] = P.gm1 * e_int;
        }
      }
    };

    // ---- ring role: one cell of the tile grown by one layer (no corners) --------------------------------
    //   [0, TY)   right column (cell HX): predictor, the tile's last x face
    //   + TY      left column (cell -1): predictor, publishes W^+_x
    //   + HX      bottom row (row -1): predictor, publishes W^+_y
    //   + HX      top row (row TY): predictor, the tile's last y face
    int pj = 0, cx = 2;
    if (at < TY) { pj = at; cx = HX + 2; }
    else if (at < 2 * TY) { pj = at - TY; cx = 1; }
    else if (at < 2 * TY + HX) { pj = -1; cx = at - 2 * TY + 2; }
    else if (at < 2 * TY + 2 * HX) { pj = TY; cx = at - (2 * TY + HX) + 2; }
    const bool pred = at < 2 * TY + 2 * HX;
    const bool right = at < TY, left = pred && cx == 1, top = pred && pj == TY, bottom = pred && pj == -1;
    const int rc = ((pj + 2) * NPX + cx) * REC;
    double* const xslot = XL + ((right || left) ? pj * (HX + 1) + (right ? HX : 0) : 0) * REC;
    double* const yslot = YL + ((top || bottom) ? (top ? TY * HX : 0) + cx - 2 : 0) * REC;
    double wm[NF];  // right column: W^-_x; top row: W^-_y
#pragma unroll
    for (int q = 0; q < NF; ++q) wm[q] = 0.0;

    issue_plane(-2, Wm);
    issue_plane(-1, Wc);
    issue_plane(0, Wp);
    cp_commit();
    cp_wait<0>();
    convert_plane(Wm);
    convert_plane(Wc);
    convert_plane(Wp);
    __syncthreads();

    for (int t = 0; t <= zc; ++t) {
      const int kk = t - 1;
      const bool mid = t >= 1;
      // ---- phase 1: predictor of the ring cells, publish W^+ ---------------------------------------
      if (mid && pred) {
        double ws[NF], hx[NF], hy[NF], hz[NF], o[NF];
        predict_cell<NF, LIM>(Wm, Wc, Wp, rc, NPX * REC, REC, P, ws, hx, hy, hz);
        if (left) {
#pragma unroll
          for (int q = 0; q < NF; ++q) o[q] = ws[q] + hx[q];
          sts_rec<NF>(xslot, o);
        } else if (bottom) {
          double r[NF];
#pragma unroll
          for (int q = 0; q < NF; ++q) o[q] = ws[q] + hy[q];
          rot_in<NF, 1>(o, r);
          sts_rec<NF>(yslot, r);
        } else if (right) {
#pragma unroll
          for (int q = 0; q < NF; ++q) wm[q] = ws[q] - hx[q];
        } else {
#pragma unroll
          for (int q = 0; q < NF; ++q) o[q] = ws[q] - hy[q];
          rot_in<NF, 1>(o, wm);
        }
      }
      prefetch_plane(kk + 2);
      __syncthreads();

      // ---- phase 2: copies of plane kk+2 into the slot plane kk-1 vacated; the tile's last x / y faces;
      //      convert plane kk+2 when it has landed (these warps have the slack to wait for it) ----------
      issue_plane(kk + 2, Wm);
      cp_commit();
      if (mid && (right || top)) {   // one solver instance: the tile's last x faces (right column) / y faces (top row)
        double* const rec = right ? xslot : yslot;
        double WL[NF], Fr[NF];
        lds_rec<NF>(rec, WL);
        x2::riemann2<NF, RS>(WL, wm, RC, Fr, true, s_cnt);
        sts_rec<NF>(rec, Fr);
        if (X2_UNLIKELY(blk >= 0)) {   // the patch's last x / y face (a7)
          if (right && x0 + HX == n) {
            double* dstF = P.fblk + ((size_t)blk * 3 + 0) * NF * fsz + ((size_t)2 * n2 + (size_t)(kk * n + (y0 + pj)));
#pragma unroll
            for (int q = 0; q < NF; ++q) atomicAdd(dstF + (size_t)q * fsz, Fr[q]);
          } else if (top && y0 + TY == n) {
            double fy[NF];
            rot_out<NF, 1>(Fr, fy);
            double* dstF = P.fblk + ((size_t)blk * 3 + 1) * NF * fsz + ((size_t)2 * n2 + (size_t)(kk * n + (x0 + cx - 2)));
#pragma unroll
            for (int q = 0; q < NF; ++q) atomicAdd(dstF + (size_t)q * fsz, fy[q]);
          }
        }
      }
      cp_wait<0>();
      convert_plane(Wm);
      __syncthreads();
      double* tmp = Wm; Wm = Wc; Wc = Wp; Wp = tmp;
    }
  }

  __syncthreads();
  if (tid == 0) {
    double m = s_red[0];
#pragma unroll
    for (int wv = 1; wv < NI / 32; ++wv) m = s_red[wv] > m ? s_red[wv] : m;
    atomicMax(reinterpret_cast<unsigned long long*>(P.smax), (unsigned long long)__double_as_longlong(m));
  }
  if (tid < 4 && s_cnt[tid] != 0) atomicAdd(P.counters + tid, (unsigned long long)s_cnt[tid]);
}

// host-side launcher for one (NF, HX, TY, NT, MAXR) tile configuration
template <int NF, int LIM, int RS, int HX, int TY, int NT, int MAXR>
cudaError_t launch_variant_d1(const StepParams<double>& P, cudaStream_t s) {
  using G = GeomD1<NF, HX, TY>;
  auto kern = godunov_step_d1_kernel<NF, LIM, RS, HX, TY, NT, MAXR>;
  static std::atomic<unsigned long long> configured{0};  // per instantiation, one bit per device
  {
    cudaError_t e = ensure_dynamic_smem((const void*)kern, (int)G::smem_bytes, configured);
    if (e != cudaSuccess) return e;
  }
  const long long grid = (long long)P.np_active * P.ntx * P.nty;
  kern<<<(unsigned)grid, NT, G::smem_bytes, s>>>(P);
  cudaError_t le = cudaGetLastError();
  if (le != cudaSuccess) {
    cudaFuncAttributes fa;
    if (cudaFuncGetAttributes(&fa, kern) == cudaSuccess)
      fprintf(stderr, "amr: d1 step kernel launch failed: %d threads, %d regs/thread, %zu B dynamic + %zu B static smem\n",
              NT, fa.numRegs, (size_t)G::smem_bytes, fa.sharedSizeBytes);
  }
  return le;
}

template <int NF, int HX, int TY, int NT, int MAXR>
cudaError_t launch_dispatch_d1(const StepParams<double>& P, int limiter, int riemann, cudaStream_t s) {
  constexpr int RSX = (NF == 5) ? x2::X2_RS_HLLC : x2::X2_RS_HLLD;
#define AMR_CASE(L, R) \
  if (limiter == L && riemann == R) return launch_variant_d1<NF, L, R, HX, TY, NT, MAXR>(P, s);
  AMR_CASE(D1_LIM_NONE, x2::X2_RS_HLL)
  AMR_CASE(D1_LIM_MINMOD, x2::X2_RS_HLL)
  AMR_CASE(D1_LIM_MC, x2::X2_RS_HLL)
  AMR_CASE(D1_LIM_NONE, RSX)
  AMR_CASE(D1_LIM_MINMOD, RSX)
  AMR_CASE(D1_LIM_MC, RSX)
#undef AMR_CASE
  return cudaErrorInvalidValue;
}

}  // namespace d1
}  // namespace amr

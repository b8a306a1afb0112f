// Fused per-tile Godunov step for sm_100a, fp32, TWO CELLS PER THREAD with packed f32x2 arithmetic:
// halo assembly (O0) -> primitives (O1) -> limited slopes (O2) -> MUSCL-Hancock predictor (O3) -> face
// states (O4) -> Riemann flux (O5) -> conservative update (O6) -> max signal speed of the new state (O7),
// one pass, nothing but U_old read from and U_new written to HBM.  Formulas: DESIGN.md §3 (SURVEY.md
// §8(c)); PAPER.md:43, 57, 58, 76 name the pieces.  The fp64 path and test-size patches (n = 8) use the
// one-cell-per-thread kernel of godunov_step.cuh.
//
// Why pairs (profiles/r1b_step_mhd_f32_ncu.md): the scalar kernel is bound by instruction issue, half of
// its instructions are FADD/FMUL/FFMA, and sm_100a issues FADD2/FMUL2/FFMA2 on an aligned register pair in
// one slot.  A thread owns the x-adjacent cells (2i, 2i+1) of one row and marches along z; every quantity
// is an F2 (pair_math.cuh).  Riemann solvers are branch-free (riemann_x2.cuh).
//
// Work decomposition: one CTA owns a TX x TY column of one patch (TX = 32 when n % 32 == 0, else 16) and
// marches along z.  Warp-specialised: TX/2 * TY interior pair threads (whole COMPUTE warps) and the AUX warps,
// which hold the ring of the tile grown by one layer (no corners): right / left x-ring pairs (cells
// (TX, TX+1) / (-2, -1), of which only the inner cell is real), bottom / top y-ring rows, and which do all
// loading.  The two roles run separate loops with the same barrier sequence.  Shared memory (all "pair
// records": the NF components of a pair as NF float2, padded to a bank-conflict-free stride, 128-bit LDS/STS):
//   ring   three planes of primitives on the tile + radius-2 halo; the raw conserved pairs of plane k+2 arrive
//          by 8-byte cp.async (LDGSTS.64) in the slot plane k-1 vacated and are converted in place by the aux
//          thread that issued the copies
//   XP     per pair of x faces (left of a pair's even cell, between its cells): their left states (W^+_x of the left
//          neighbour's odd cell - handed over by shuffle - and of the own even cell) as ONE pair record, then the two
//          x fluxes        YP   per pair of y faces: W^+_y of the pair below (y solver's component order), then the fluxes
//   UO     (m, E) of the cell awaiting its update (conversion overwrites them in the ring)
//   SCR    private staging of each compute thread (face states between phases, own fluxes), which keeps a
//          thread that carries two MHD cells within 168 registers (two CTAs per SM)
// Per plane, two barriers:
//   1  compute: slopes, predictor, positivity; publish W^+_x (odd cell), W^+_y; stage W^-; the z faces (left
//      state = staged W^+_z of the previous plane) are solved and the previous plane is updated, stored and
//      its signal speed reduced.  aux: predictor of the ring pairs                          | barrier
//   2  compute: the two x faces (left of the even cell, between the cells) and the two y faces below the
//      pair.  aux: copies of plane k+2 (asked for in the L2 at the end of phase 1), the tile's last x / y
//      faces, convert plane k+2                                                             | barrier
//   3  compute: flux differences of this plane -> registers; falls through into 1 of the next plane
// Every face flux is computed once per tile by one position-independent routine from bit-identical
// inputs, so a face shared by two tiles/patches gets the same bits on both sides (conservation to
// round-off).
#pragma once
#include <cstdio>
#include <cuda_runtime.h>

#include "amr_internal.hpp"
#include "riemann_x2.cuh"
#include "signal_speed.cuh"

namespace amr {
namespace x2 {

enum { X2_LIM_NONE = 0, X2_LIM_MINMOD = 1, X2_LIM_MC = 2 };
enum { X2_CNT_POSITIVITY = 0, X2_CNT_NEG_STATE = 3 };

// O2 as HALF slopes (see godunov_step.cuh): branch-free forms that return exactly the sign-test value.
template <int LIM>
__device__ __forceinline__ F2 half_slope2(F2 a, F2 b) {
  if (LIM == X2_LIM_NONE) return F2(0.f);
  if (LIM == X2_LIM_MINMOD) {
    const F2 ha = 0.5f * a, hb = 0.5f * b;
    return max2(min2(ha, hb), min2(max2(ha, hb), 0.f));
  }
  const F2 q = 0.25f * (a + b);
  return max2(min3(a, b, q), min2(max3(a, b, q), 0.f));
}

// ---- vector shared-memory access: N floats, bulk in VW-wide vectors, tail in narrower ones ---------
template <int N, int VW>
__device__ __forceinline__ void lds_n(const float* p, float* o) {
  constexpr int NV = N / VW;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    if constexpr (VW == 4) {
      const float4 v = *reinterpret_cast<const float4*>(p + 4 * i);
      o[4 * i] = v.x; o[4 * i + 1] = v.y; o[4 * i + 2] = v.z; o[4 * i + 3] = v.w;
    } else {
      const float2 v = *reinterpret_cast<const float2*>(p + 2 * i);
      o[2 * i] = v.x; o[2 * i + 1] = v.y;
    }
  }
  constexpr int R0 = NV * VW;
  if constexpr (N - R0 >= 2) {
    const float2 v = *reinterpret_cast<const float2*>(p + R0);
    o[R0] = v.x; o[R0 + 1] = v.y;
  }
  if constexpr ((N - R0) & 1) o[N - 1] = p[N - 1];
}
template <int N, int VW>
__device__ __forceinline__ void sts_n(float* p, const float* o) {
  constexpr int NV = N / VW;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    if constexpr (VW == 4) *reinterpret_cast<float4*>(p + 4 * i) = make_float4(o[4 * i], o[4 * i + 1], o[4 * i + 2], o[4 * i + 3]);
    else *reinterpret_cast<float2*>(p + 2 * i) = make_float2(o[2 * i], o[2 * i + 1]);
  }
  constexpr int R0 = NV * VW;
  if constexpr (N - R0 >= 2) *reinterpret_cast<float2*>(p + R0) = make_float2(o[R0], o[R0 + 1]);
  if constexpr ((N - R0) & 1) p[N - 1] = o[N - 1];
}
// A whole record through opaque vector loads.  When only one half of every pair is used (the x neighbours' records in
// the slope stencil) the compiler turns a plain vector load into nine scalar loads, and scalar accesses at the record
// stride of 20 words are 4-way bank conflicts (ncu: 8.9e6 wavefronts per instruction where 2.2e6 are ideal); five opaque
// vector loads fetch the record in 20 wavefronts instead of 36.  Worth 0.7 % (config 5) to 1.1 % (config 3) of the MHD
// step; the same for the right neighbour's flux record in phase 3 costs 3 % (more live registers there) and is not done.
template <int N>
__device__ __forceinline__ void lds_n_opaque(const float* p, float* o) {
  static_assert(N == 18 || N == 10, "records of 9 or 5 pairs");
  const unsigned a = (unsigned)__cvta_generic_to_shared(p);
#pragma unroll
  for (int i = 0; i < N / 4; ++i)
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                 : "=f"(o[4 * i]), "=f"(o[4 * i + 1]), "=f"(o[4 * i + 2]), "=f"(o[4 * i + 3]) : "r"(a + 16 * i));
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(o[N - 2]), "=f"(o[N - 1]) : "r"(a + 4 * (N - 2)));
}
// a pair record <-> F2[NF]
template <int NF>
__device__ __forceinline__ void lds_pairs(const float* p, F2* w) {
  float t[2 * NF];
  lds_n<2 * NF, 4>(p, t);
#pragma unroll
  for (int q = 0; q < NF; ++q) w[q] = F2(t[2 * q], t[2 * q + 1]);
}
// MHD records go out as one opaque 64-bit store per component pair.  ptxas merges them back into the same 128-bit
// stores; what changes is the order in which the compiler may schedule the code around them, and that is worth
// 4.7 % of the MHD step (config 5: 12.84 -> 12.23 ms, config 3 fp32: 1.76 -> 1.68 ms; pinning the loads or the
// staging blocks as well, or plain compiler fences at the same places, gains nothing).  The hydro kernel is 0.8 %
// slower with it and keeps the plain vector stores.
template <int NF>
__device__ __forceinline__ void sts_pairs(float* p, const F2* w) {
  if constexpr (NF == 9) {
#pragma unroll
    for (int q = 0; q < NF; ++q) {
      const unsigned d = (unsigned)__cvta_generic_to_shared(p + 2 * q);
      asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(d), "f"(w[q].v.x), "f"(w[q].v.y) : "memory");
    }
  } else {
    float t[2 * NF];
#pragma unroll
    for (int q = 0; q < NF; ++q) { t[2 * q] = w[q].v.x; t[2 * q + 1] = w[q].v.y; }
    sts_n<2 * NF, 4>(p, t);
  }
}

__device__ __forceinline__ void cp_async8(float* smem_dst, const float* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(float* smem_dst, const float* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int NF, int TX, int TY>
struct GeomX2 {
  static constexpr int HX = TX / 2;                 // interior pair columns
  static constexpr int NPX = HX + 2;                // pair columns of a ring row (one halo pair each side)
  static constexpr int RH = TY + 4;                 // ring rows
  static constexpr int REC = NF == 9 ? 20 : 12;     // floats per pair record (NF float2 + pad)
  static constexpr int SLOT = RH * NPX * REC;       // floats per ring plane
  static constexpr int NSLOT = 3;                   // planes k-1, k, k+1; plane k+2 lands in the slot k-1 vacates
  static constexpr int BLK = NF == 9 ? 5 : 3;       // float4 per staging block: NF pairs + 2 floats
  static constexpr int NSCR = 3 * BLK;              // float4 of private staging per interior pair thread
  static constexpr int NI = HX * TY;                // interior pair threads
  static constexpr int NPRED = NI + 2 * TY + 2 * HX;
  static constexpr int NXP = TY * (HX + 1);
  static constexpr int NYP = (TY + 1) * HX;
  static constexpr int NCHUNK = RH * NPX;
  static constexpr size_t smem_floats = (size_t)NSLOT * SLOT + (size_t)NXP * REC + (size_t)NYP * REC + (size_t)2 * 2 * NI * 4 + (size_t)NSCR * NI * 4;
  static constexpr size_t smem_bytes = smem_floats * sizeof(float);
};

// rotated component order handed to the 1-D Riemann routine: x -> (x,y,z), y -> (y,z,x), z -> (z,x,y)
template <int NF, int D>
__device__ __forceinline__ void rot_in(const F2* w, F2* r) {
  constexpr int qn = 1 + D, q1 = 1 + (D + 1) % 3, q2 = 1 + (D + 2) % 3;
  r[0] = w[0]; r[1] = w[qn]; r[2] = w[q1]; r[3] = w[q2]; r[4] = w[4];
  if (NF == 9) { r[5] = w[4 + qn]; r[6] = w[4 + q1]; r[7] = w[4 + q2]; r[8] = w[8]; }
}
template <int NF, int D>
__device__ __forceinline__ void rot_out(const F2* r, F2* f) {
  constexpr int qn = 1 + D, q1 = 1 + (D + 1) % 3, q2 = 1 + (D + 2) % 3;
  f[0] = r[0]; f[qn] = r[1]; f[q1] = r[2]; f[q2] = r[3]; f[4] = r[4];
  if (NF == 9) { f[4 + qn] = r[5]; f[4 + q1] = r[6]; f[4 + q2] = r[7]; f[8] = r[8]; }
}

// O2 + O3 + O4 for the pair whose ring record is at element offset rc: half slopes hx, hy, hz, predicted
// state ws.  A cell that fails the positivity test (A10) gets ws = W and zero slopes (first order); the
// number of such real cells (vcell) is returned.
template <int NF, int LIM>
__device__ __forceinline__ int predict_pair(const float* Wm, const float* Wc, const float* Wp, int rc, int rowstride,
                                            int recstride, const StepParams<float>& P, F2 ms, B2 vcell,
                                            F2* ws, F2* hx, F2* hy, F2* hz) {
  F2 w[NF];
  {
    const float* cc = Wc + rc;
    float c[2 * NF], a[2 * NF], b[2 * NF];
    lds_n<2 * NF, 4>(cc, c);
    lds_n_opaque<2 * NF>(cc - recstride, a);   // only the odd halves are used
    lds_n_opaque<2 * NF>(cc + recstride, b);   // only the even halves are used
#pragma unroll
    for (int q = 0; q < NF; ++q) {
      w[q] = F2(c[2 * q], c[2 * q + 1]);
      const float d0 = c[2 * q] - a[2 * q + 1], d1 = c[2 * q + 1] - c[2 * q], d2 = b[2 * q] - c[2 * q + 1];
      hx[q] = half_slope2<LIM>(F2(d0, d1), F2(d1, d2));
    }
    F2 am[NF], bp[NF];
    lds_pairs<NF>(cc - rowstride, am);
    lds_pairs<NF>(cc + rowstride, bp);
#pragma unroll
    for (int q = 0; q < NF; ++q) hy[q] = half_slope2<LIM>(w[q] - am[q], bp[q] - w[q]);
    lds_pairs<NF>(Wm + rc, am);
    lds_pairs<NF>(Wp + rc, bp);
#pragma unroll
    for (int q = 0; q < NF; ++q) hz[q] = half_slope2<LIM>(w[q] - am[q], bp[q] - w[q]);
  }
  // O3 predictor with half slopes: W* = W - (dt/dx) sum_d A_d h_d
  const F2 rho = w[0], pr = w[4];
  const F2 ir = rcp2(rho);
#define ADV(q) fma(w[3], hz[q], fma(w[2], hy[q], w[1] * hx[q]))
  const F2 divv = hx[1] + hy[2] + hz[3];
  ws[0] = fma(ms, fma(rho, divv, ADV(0)), rho);
  if (NF == 5) {
    ws[1] = fma(ms, fma(hx[4], ir, ADV(1)), w[1]);
    ws[2] = fma(ms, fma(hy[4], ir, ADV(2)), w[2]);
    ws[3] = fma(ms, fma(hz[4], ir, ADV(3)), w[3]);
    ws[4] = fma(ms, fma(P.gamma * pr, divv, ADV(4)), pr);
  } else {
#define BGRAD(q) fma(w[7], hz[q], fma(w[6], hy[q], w[5] * hx[q]))
    const F2 divB = hx[5] + hy[6] + hz[7];
    const F2 vB = fma(w[3], w[7], fma(w[2], w[6], w[1] * w[5]));
    const F2 BdBx = fma(w[7], hx[7], fma(w[6], hx[6], w[5] * hx[5]));
    const F2 BdBy = fma(w[7], hy[7], fma(w[6], hy[6], w[5] * hy[5]));
    const F2 BdBz = fma(w[7], hz[7], fma(w[6], hz[6], w[5] * hz[5]));
    ws[1] = fma(ms, fma((hx[4] + BdBx) - fma(w[5], divB, BGRAD(5)), ir, ADV(1)), w[1]);
    ws[2] = fma(ms, fma((hy[4] + BdBy) - fma(w[6], divB, BGRAD(6)), ir, ADV(2)), w[2]);
    ws[3] = fma(ms, fma((hz[4] + BdBz) - fma(w[7], divB, BGRAD(7)), ir, ADV(3)), w[3]);
    ws[5] = fma(ms, (fma(w[5], divv, ADV(5)) - fma(w[1], divB, BGRAD(1))) + hx[8], w[5]);
    ws[6] = fma(ms, (fma(w[6], divv, ADV(6)) - fma(w[2], divB, BGRAD(2))) + hy[8], w[6]);
    ws[7] = fma(ms, (fma(w[7], divv, ADV(7)) - fma(w[3], divB, BGRAD(3))) + hz[8], w[7]);
    ws[4] = fma(ms, fma(P.gm1, fms(vB, divB, BGRAD(8)), fma(P.gamma * pr, divv, ADV(4))), pr);
    ws[8] = fma(ms * P.ch2, divB, w[8]);
#undef BGRAD
  }
#undef ADV
  // O4 positivity: the smallest/largest of the six face values of rho and p
  const F2 hr = max3(abs2(hx[0]), abs2(hy[0]), abs2(hz[0]));
  const F2 hp = max3(abs2(hx[4]), abs2(hy[4]), abs2(hz[4]));
  const F2 inf = F2(CUDART_INF_F);
  const B2 ok = gt(ws[0] - hr, 0.f) & gt(ws[4] - hp, 0.f) & lt(ws[0] + hr, inf) & lt(ws[4] + hp, inf);
  const B2 bad = !ok & vcell;
  if (X2_UNLIKELY(any(bad))) {  // rare
#pragma unroll
    for (int q = 0; q < NF; ++q) {
      ws[q] = sel(bad, w[q], ws[q]);
      hx[q] = sel(bad, 0.f, hx[q]); hy[q] = sel(bad, 0.f, hy[q]); hz[q] = sel(bad, 0.f, hz[q]);
    }
    return (int)bad.x + (int)bad.y;
  }
  return 0;
}

template <int NF, int LIM, int RS, int TX, int TY, int NT, int MAXR>
__global__ void __maxnreg__(MAXR) godunov_step_x2_kernel(const __grid_constant__ StepParams<float> P) {
  using G = GeomX2<NF, TX, TY>;
  constexpr int HX = G::HX, NPX = G::NPX, RH = G::RH, REC = G::REC;
  constexpr int SLOT = G::SLOT, NI = G::NI, NPRED = G::NPRED, NCHUNK = G::NCHUNK;
  constexpr int NA = NT - NI;                 // aux threads: ring pairs + the plane loader
  constexpr int LC = (NCHUNK + NA - 1) / NA;  // loader chunks (pairs of one ring plane) per aux thread
  static_assert(NI % 32 == 0 && NT % 32 == 0 && NT >= NPRED, "compute warps = interior pairs; aux warps hold the ring");
  static_assert(TX % 4 == 0 && LC <= 8, "tile shape");

  extern __shared__ __align__(16) unsigned char smem_raw[];
  float* const ring = reinterpret_cast<float*>(smem_raw);  // [3][RH][NPX][REC]
  float* const XP = ring + G::NSLOT * SLOT;                // [TY][HX+1][REC]
  float* const YP = XP + G::NXP * REC;                     // [TY+1][HX][REC]
  float* const UO = YP + G::NYP * REC;                     // [2][2][NI][4]
  float4* const SCR = reinterpret_cast<float4*>(UO + 2 * 2 * NI * 4);  // [NSCR][NI] float4
  __shared__ int s_nbr[27];
  __shared__ int s_cnt[4];
  __shared__ float s_red[NI / 32];

  const int tid = threadIdx.x;
  const int n = P.n;
  int bb = blockIdx.x;
  const int tpp = P.ntx * P.nty;
  const int p = bb / tpp;
  bb -= p * tpp;
  const int ty = bb / P.ntx, tx = bb - ty * P.ntx;
  const int x0 = tx * TX, y0 = ty * TY;
  const int zc = n;  // the whole z extent of the patch (ntz = 1)

  if (tid < 27) s_nbr[tid] = P.nbr[p * 27 + tid];
  if (tid < 4) s_cnt[tid] = 0;
  __syncthreads();

  const int n2 = n * n;
  const int n3 = n2 * n;  // host guarantees np * (n+2g)^3 < 2^31
  const size_t fs_int = (size_t)P.np * n3;

  RC2 RC;
  RC.gamma = P.gamma; RC.igm1 = P.igm1; RC.ch2 = P.ch2; RC.half_ch = 0.5f * P.ch; RC.half_ich = P.half_ich;
  RC.eps = P.eps;
  const int blk = (P.fblk != nullptr) ? P.fblk_of[p] : -1;  // flux-register block of this patch
  // flux blocks: [block][direction][field][3 face planes: index 0, n/2, n along the normal][n^2 in-plane, the
  // lower remaining axis fastest]
  const size_t fsz = (size_t)3 * n2;
  const F2 ms = F2(-P.dtdx);

  float* Wm = ring;
  float* Wc = ring + SLOT;
  float* Wp = ring + 2 * SLOT;

  if (tid < NI) {
    // =================================== compute warps: interior pairs ===================================
    const int pj = tid / HX, pc = tid - pj * HX;                 // row, pair column: cells (2 pc, 2 pc + 1)
    const int rc = ((pj + 2) * NPX + pc + 1) * REC;              // ring record of this pair
    float* const xpub = XP + (pj * (HX + 1) + pc + 1) * REC;     // the right neighbour's x face pair: its left states, then its fluxes
    float* const xsol = xpub - REC;                              // this pair's x faces (left of the even cell, between the cells)
    float* const ypub = YP + ((pj + 1) * HX + pc) * REC;         // W^+_y, then the upper pair's y fluxes
    float* const ysol = ypub - HX * REC;                         // W^+_y of the pair below, then this pair's y fluxes
    const int cell0 = p * n3 + (y0 + pj) * n + (x0 + 2 * pc);
    float* const uo = UO + tid * 4;

    // Only the pending flux sum lives in registers across the phases; the face states a later phase needs
    // are staged in this thread's private shared-memory scratch (float4 j of thread tid at SCR[j*NI + tid]):
    // (blocks of BLK float4 = NF pairs + 2 floats: 5 for MHD, 3 for hydro)
    //   BZ      W^+_z of the previous plane (left state of the next z face)
    //   BX      W^-_x pair (right states of the pair's two x faces); after the x solve: the x flux pair
    //   BY      W^-_y pair in the y solver's component order (y, z, x); after the y solve: the y flux pair, same order
    float4* const sc = SCR + tid;
    constexpr int BLK = G::BLK, BZ = 0, BX = BLK, BY = 2 * BLK, NFULL = (NF - 1) / 2;
    auto st_block = [&](int j0, const F2* a, float e0, float e1) {  // NF pairs + 2 floats -> BLK float4
#pragma unroll
      for (int i = 0; i < NFULL; ++i) sc[(j0 + i) * NI] = make_float4(a[2 * i].v.x, a[2 * i].v.y, a[2 * i + 1].v.x, a[2 * i + 1].v.y);
      sc[(j0 + NFULL) * NI] = make_float4(a[NF - 1].v.x, a[NF - 1].v.y, e0, e1);
    };
    auto ld_block = [&](int j0, F2* a, float& e0, float& e1) {
#pragma unroll
      for (int i = 0; i < NFULL; ++i) {
        const float4 v = sc[(j0 + i) * NI];
        a[2 * i] = F2(v.x, v.y); a[2 * i + 1] = F2(v.z, v.w);
      }
      const float4 v = sc[(j0 + NFULL) * NI];
      a[NF - 1] = F2(v.x, v.y); e0 = v.z; e1 = v.w;
    };
    static_assert(NF == 9 || NF == 5, "staging blocks are laid out for 9 fields (hydro uses the first 5)");
    F2 dU[NF];    // flux sum of the plane whose update is pending: ((Fx+ - Fx-) + (Fy+ - Fy-)) - Fz-
    float smax_loc = 0.f;
    int npos = 0;
#pragma unroll
    for (int q = 0; q < NF; ++q) dU[q] = F2(0.f);
    __syncthreads();  // the aux warps have staged and converted planes -2, -1, 0

    for (int t = 0; t <= zc + 1; ++t) {
      const int kk = t - 1;                    // plane being predicted
      const bool mid = (t >= 1) && (t <= zc);  // kk is a plane of this patch (x/y fluxes needed)

      // ---- phase 1: slopes, predictor, face states; z faces; update of plane kk-1 ------------------
      {
        F2 WL[9], WR[9];
        {
          F2 ws[9], hx[NF], hy[NF], hz[NF];
          const int nb = predict_pair<NF, LIM>(Wm, Wc, Wp, rc, NPX * REC, REC, P, ms, B2(true), ws, hx, hy, hz);
          if (mid) {
            npos += nb;
            F2 o[9], r[9];
#pragma unroll
            for (int q = NF; q < 9; ++q) { o[q] = F2(0.f); r[q] = F2(0.f); ws[q] = F2(0.f); }
            // x: the left states of this pair's two x faces are (W^+_x of the left neighbour's odd cell, W^+_x of the own
            // even cell).  The neighbour's value arrives by shuffle (a row of pairs lies inside one warp), so every pair
            // publishes ONE complete pair record, as it does for y.  First pair of a row: its left neighbour is the left
            // ring pair (aux warp), which writes the .x halves itself; last pair of a row: the right ring pair's face
            // needs this pair's odd cell, written here.
            {
              F2 wpx[NF];
#pragma unroll
              for (int q = 0; q < NF; ++q) wpx[q] = ws[q] + hx[q];
#pragma unroll
              for (int q = 0; q < NF; ++q) o[q] = F2(__shfl_up_sync(0xffffffffu, wpx[q].v.y, 1), wpx[q].v.x);
              if (pc != 0) sts_pairs<NF>(xsol, o);
              else {
#pragma unroll
                for (int q = 0; q < NF; ++q) xsol[2 * q + 1] = wpx[q].v.x;
              }
              if (pc == HX - 1) {
#pragma unroll
                for (int q = 0; q < NF; ++q) xpub[2 * q] = wpx[q].v.y;
              }
            }
            // y: W^+_y of this pair = left states of the upper pair's y faces, in the y solver's component order
#pragma unroll
            for (int q = 0; q < NF; ++q) o[q] = ws[q] + hy[q];
            rot_in<NF, 1>(o, r);
            sts_pairs<NF>(ypub, r);
#pragma unroll
            for (int q = 0; q < NF; ++q) o[q] = ws[q] - hx[q];
            st_block(BX, o, 0.f, 0.f);
#pragma unroll
            for (int q = 0; q < NF; ++q) o[q] = ws[q] - hy[q];
            rot_in<NF, 1>(o, r);
            st_block(BY, r, 0.f, 0.f);
          }
          // z direction: left state of the face below = W^+_z of the previous plane (scratch), then this
          // plane's W^+_z takes its place
          float e0, e1;
          F2 zl[9];
          ld_block(BZ, zl, e0, e1);
          rot_in<NF, 2>(zl, WL);
#pragma unroll
          for (int q = 0; q < NF; ++q) zl[q] = ws[q] + hz[q];
#pragma unroll
          for (int q = NF; q < 9; ++q) zl[q] = F2(0.f);
          st_block(BZ, zl, 0.f, 0.f);
#pragma unroll
          for (int q = 0; q < NF; ++q) zl[q] = ws[q] - hz[q];
          rot_in<NF, 2>(zl, WR);
        }
        if (t >= 1) {  // z faces between planes kk-1 and kk
          F2 fz[NF];
          {
            F2 Fr[NF];
            riemann2<NF, RS>(WL, WR, RC, Fr, B2(true), s_cnt);
            rot_out<NF, 2>(Fr, fz);
          }
          // flux registers of a coarse-fine link (a7).  Only the face planes a link can read are recorded: index 0,
          // n/2, n along the normal (fine patches sit on aligned (n/2)^3 blocks of the parent level).  The sum over
          // substeps is a result-less atomicAdd (RED): one writer per address and step, so the value is that of
          // a plain +=, without exposing the load latency of a read-modify-write in this latency-bound loop
          if (X2_UNLIKELY(blk >= 0) && (kk == 0 || kk == (n >> 1) || kk == n)) {
            float* dstF = P.fblk + ((size_t)blk * 3 + 2) * NF * fsz + ((size_t)((kk) == 0 ? 0 : ((kk) == n ? 2 : 1)) * n2 + (size_t)((y0 + pj) * n + (x0 + 2 * pc)));
#pragma unroll
            for (int q = 0; q < NF; ++q) { atomicAdd(dstF + (size_t)q * fsz, fz[q].v.x); atomicAdd(dstF + (size_t)q * fsz + 1, fz[q].v.y); }
          }
          if (t >= 2) {  // O6 for plane kk-1, GLM damping, O7 of the new state
            // U_old: rho, B, psi are the ring record of plane kk-1 (conversion leaves them untouched),
            // (m, E) were staged two iterations ago
            F2 un[NF];
            const float* om = Wm + rc;
            un[0].v = *reinterpret_cast<const float2*>(om);
            if (NF == 9) {
              float t8[8];
              lds_n<8, 2>(om + 10, t8);  // B_x | B_y B_z | psi at floats 10..17 (8-byte aligned)
              un[5] = F2(t8[0], t8[1]); un[6] = F2(t8[2], t8[3]); un[7] = F2(t8[4], t8[5]); un[8] = F2(t8[6], t8[7]);
            }
            {
              const float* ou = uo + ((t & 1) ? 2 * NI * 4 : 0);
              const float4 v0 = *reinterpret_cast<const float4*>(ou), v1 = *reinterpret_cast<const float4*>(ou + NI * 4);
              un[1] = F2(v0.x, v0.y); un[2] = F2(v0.z, v0.w); un[3] = F2(v1.x, v1.y); un[4] = F2(v1.z, v1.w);
            }
#pragma unroll
            for (int q = 0; q < NF; ++q) un[q] = fma(ms, dU[q] + fz[q], un[q]);
            if (NF == 9) un[8] = un[8] * P.damp;
            float* out = P.Uout + (cell0 + (kk - 1) * n2);
#pragma unroll
            for (int q = 0; q < NF; ++q) *reinterpret_cast<float2*>(out + q * fs_int) = un[q].v;
            if (X2_UNLIKELY(!(un[0].v.x > 0.f) || !(un[0].v.y > 0.f)))
              atomicAdd(&s_cnt[X2_CNT_NEG_STATE], (int)!(un[0].v.x > 0.f) + (int)!(un[0].v.y > 0.f));
            const F2 sp = signal_speed<F2, NF>(un, F2(P.gamma), F2(P.gm1));
            smax_loc = fmaxf(smax_loc, fmaxf(sp.v.x, sp.v.y));
          }
#pragma unroll
          for (int q = 0; q < NF; ++q) dU[q] = -fz[q];
        }
      }
      if (t == zc + 1) break;
      __syncthreads();

      // ---- phase 2: copy of (m, E) of plane kk+1; the x and y Riemann problems of plane kk -----------
      if (t <= zc - 1) {
        const float* src = P.Uin + (cell0 + (kk + 1) * n2);
        float* d = uo + ((t & 1) ? 2 * NI * 4 : 0);
        cp_async8(d, src + fs_int);
        cp_async8(d + 2, src + 2 * fs_int);
        cp_async8(d + NI * 4, src + 3 * fs_int);
        cp_async8(d + NI * 4 + 2, src + 4 * fs_int);
      }
      cp_commit();
      if (mid) {
        // d = 0: the pair's two x faces; d = 1: its two y faces.  ONE solver instance (the plane loop is bound by
        // instruction fetch: profiles/r2a); operands and results in the solver's component order (identity for x,
        // rotated for y), uniform pair records / staging blocks, so that nothing but two pointers differs per trip.
#pragma unroll 1
        for (int d = P.ntz - 1; d < 2; ++d) {   // ntz == 1: an opaque lower bound keeps the loop from being unrolled
          float* const rec = d ? ysol : xsol;
          const int bj = d ? BY : BX;
          F2 WL[9], WR[9], Fr[9];
          float e0, e1;
          lds_pairs<NF>(rec, WL);
          ld_block(bj, WR, e0, e1);
          riemann2<NF, RS>(WL, WR, RC, Fr, B2(true), s_cnt);
#pragma unroll
          for (int q = NF; q < 9; ++q) Fr[q] = F2(0.f);
          sts_pairs<NF>(rec, Fr);         // for the left / lower neighbour's phase 3
          st_block(bj, Fr, 0.f, 0.f);     // private copy for this thread's phase 3 (the neighbour overwrites rec in ITS
                                          // next phase 1, with no barrier in between)
          // record the fluxes for the reflux: x faces 0 and n/2 are the even face of a pair
          const int fidx = d ? y0 + pj : x0 + 2 * pc;
          if (X2_UNLIKELY(blk >= 0) && (fidx == 0 || fidx == (n >> 1))) {
            F2 f[NF];
            if (d) rot_out<NF, 1>(Fr, f); else rot_out<NF, 0>(Fr, f);
            float* dstF = P.fblk + ((size_t)blk * 3 + d) * NF * fsz + (size_t)(fidx == 0 ? 0 : 1) * n2 +
                          (size_t)(d ? kk * n + (x0 + 2 * pc) : kk * n + (y0 + pj));
#pragma unroll
            for (int q = 0; q < NF; ++q) {
              atomicAdd(dstF + (size_t)q * fsz, f[q].v.x);
              if (d) atomicAdd(dstF + (size_t)q * fsz + 1, f[q].v.y);
            }
          }
        }
      }
      cp_wait<1>();
      __syncthreads();

      // ---- phase 3: x/y flux differences of plane kk -> registers ----------------------------------
      // own fluxes are read back from the private scratch; the right neighbour's lo-face flux and the upper
      // pair's y fluxes come from the slots this very thread overwrites with its W^+ in the next phase 1,
      // so no barrier is needed before that
      if (mid) {
        float e0, e1;
        F2 xr[NF], fu[NF], fx[9], fy[9], dy[NF], dyu[NF];
        ld_block(BX, fx, e0, e1);
        ld_block(BY, fy, e0, e1);
        lds_pairs<NF>(xpub, xr);     // the right neighbour's x fluxes: its lo face is the face right of this pair's odd cell
        lds_pairs<NF>(ypub, fu);     // the upper pair's y fluxes (y solver's component order)
#pragma unroll
        for (int q = 0; q < NF; ++q) dy[q] = fu[q] - fy[q];
        rot_out<NF, 1>(dy, dyu);
#pragma unroll
        for (int q = 0; q < NF; ++q) {
          const F2 dfx = F2(fx[q].v.y - fx[q].v.x, xr[q].v.x - fx[q].v.y);
          dU[q] = (dfx + dyu[q]) + dU[q];
        }
        // xpub is the right neighbour's record: it rewrites it in its next phase 1.  Neighbours in x are lanes of the
        // same warp (a row of pairs never straddles warps), so a warp-level fence orders the read before that write
        __syncwarp();
      }
      float* tmp = Wm; Wm = Wc; Wc = Wp; Wp = tmp;
    }

    // ---- epilogue: max signal speed of the new state (O7), event counters -------------------------
    if (npos) atomicAdd(&s_cnt[X2_CNT_POSITIVITY], npos);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) smax_loc = fmaxf(smax_loc, __shfl_xor_sync(0xffffffffu, smax_loc, o));
    if ((tid & 31) == 0) s_red[tid >> 5] = smax_loc;
  } else {
    // ======================= aux warps: plane loader (O0, O1) and the ring of the tile =======================
    const int at = tid - NI;
    const int M = n + 2 * P.g;
    const int M2 = M * M;
    const size_t fs_halo = (size_t)P.np * M2 * M;

    // ---- plane loader: raw conserved pairs of plane lz -> ring slot, asynchronously -----------------
    // chunk c = ry*NPX + px <-> cells (lx, lx+1), lx = x0 + 2 px - 2, row ly = y0 + ry - 2.  The halo pairs
    // of the outermost rows (corners outside the stencil footprint) are skipped.  Per z region the source
    // of a chunk is fixed up to the z term, so its offset is resolved once per region:
    //   goff  element offset of (source patch, z = 0, sy, sx)   hmask  source is the prolongation halo
    //   zmask the z index is clamped (outflow)                  smask  two 4-byte copies (x clamped: both
    //   from the same cell; halo buffer: odd element offset) instead of one 8-byte copy; dmask: second = +1
    unsigned lmask = 0;
#pragma unroll
    for (int l = 0; l < LC; ++l) {
      const int c = at + l * NA;
      if (c < NCHUNK) {
        const int ry = c / NPX, px = c - ry * NPX;
        const bool corner = (ry == 0 || ry == RH - 1) && (px == 0 || px == NPX - 1);
        if (!corner) lmask |= 1u << l;
      }
    }
    int goff[LC];
    unsigned hmask = 0, zmask = 0, smask = 0, dmask = 0;
    int cur_rz = -1;
    auto setup_region = [&](int rz) {
      hmask = 0; zmask = 0; smask = 0; dmask = 0;
#pragma unroll
      for (int l = 0; l < LC; ++l) {
        goff[l] = 0;
        if (lmask & (1u << l)) {
          const int c = at + l * NA;
          const int ry = c / NPX, px = c - ry * NPX;
          const int lx = x0 + 2 * px - 2, ly = y0 + ry - 2;
          const int gx = lx < 0 ? 0 : (lx >= n ? 2 : 1), gy = ly < 0 ? 0 : (ly >= n ? 2 : 1);
          const int e = s_nbr[rz * 9 + gy * 3 + gx];
          if (e >= 0) {
            const int sp = e & NBR_PATCH_MASK, md = e >> NBR_MODE_SHIFT;
            int sx = lx - (gx - 1) * n;
            if (gx != 1 && (md & 1)) { sx = gx == 0 ? 0 : n - 1; smask |= 1u << l; }
            const int sy = (gy != 1 && (md & 2)) ? (gy == 0 ? 0 : n - 1) : ly - (gy - 1) * n;
            if (rz != 1 && (md & 4)) zmask |= 1u << l;
            goff[l] = sp * n3 + sy * n + sx;
          } else {
            hmask |= 1u << l; smask |= 1u << l; dmask |= 1u << l;
            goff[l] = p * (M2 * M) + (ly + P.g) * M + (lx + P.g);
          }
        }
      }
      cur_rz = rz;
    };
    // The lines issue_plane(lz) is going to copy, requested into the L2 ahead of time.  The copies can only be issued
    // once the ring slot is free (phase 2), and the copy-solve-convert chain of these warps ends phase 2 for the whole
    // CTA: with two thirds of the plane's lines missing the L2 the copies' DRAM latency sat on that chain.  Asked for at
    // the end of phase 1 they are L2 hits (config 5: 12.15 -> 11.61 ms, config 3 fp32: 1.672 -> 1.624 ms; from phase 2
    // of the previous plane: slower, it lengthens the chain it is meant to shorten).  A request fetches its 128-byte
    // line, so one thread per (ring row, run of the row: left halo pair / interior / right halo pair) asks for the run's
    // first pair in every field.  It is a hint: runs that come from a clamped cell (outflow) are simply not asked for.
    const int pf_ry = at / 3, pf_run = at - 3 * pf_ry;
    const bool pf_on = pf_ry < RH && !((pf_ry == 0 || pf_ry == RH - 1) && pf_run != 1);
    auto prefetch_plane = [&](int lz) {
      if (pf_on) {
        const int rz = lz < 0 ? 0 : (lz >= n ? 2 : 1);
        const int lx = pf_run == 0 ? x0 - 2 : (pf_run == 1 ? x0 : x0 + TX), ly = y0 + pf_ry - 2;
        const int gx = lx < 0 ? 0 : (lx >= n ? 2 : 1), gy = ly < 0 ? 0 : (ly >= n ? 2 : 1);
        const int e = s_nbr[rz * 9 + gy * 3 + gx];
        if (e >= 0 && (e >> NBR_MODE_SHIFT) == 0) {
          const int off = (e & NBR_PATCH_MASK) * n3 + (lz - (rz - 1) * n) * n2 + (ly - (gy - 1) * n) * n + (lx - (gx - 1) * n);
          const float* src = P.Uin + off;
#pragma unroll
          for (int q = 0; q < NF; ++q) asm volatile("prefetch.global.L2 [%0];" ::"l"(src + q * fs_int));
        } else if (e < 0) {   // the run comes from the prolongation halo buffer (coarse-fine boundary)
          const float* src = P.halo + (p * (M2 * M) + (lz + P.g) * M2 + (ly + P.g) * M + (lx + P.g));
#pragma unroll
          for (int q = 0; q < NF; ++q) asm volatile("prefetch.global.L2 [%0];" ::"l"(src + q * fs_halo));
        }
      }
    };
    // the common case (one 8-byte copy per component: a whole pair from a patch interior) first and on its own, the split
    // copies of clamped / halo-buffer chunks behind a rare branch
    auto issue_plane = [&](int lz, float* dst) {
      const int rz = lz < 0 ? 0 : (lz >= n ? 2 : 1);
      if (rz != cur_rz) setup_region(rz);
      const int zt_int = (lz - (rz - 1) * n) * n2;
      const int zt_clamp = (rz == 0 ? 0 : n - 1) * n2;
#pragma unroll
      for (int l = 0; l < LC; ++l) {
        if (lmask & ~smask & (1u << l)) {
          const int off = goff[l] + ((zmask & (1u << l)) ? zt_clamp : zt_int);
          const float* src = P.Uin + off;
          float* d = dst + (at + l * NA) * REC;
#pragma unroll
          for (int q = 0; q < NF; ++q) cp_async8(d + 2 * q, src + q * fs_int);
        }
      }
      if (X2_UNLIKELY(smask != 0)) {
        const int zt_halo = (lz + P.g) * M2;
#pragma unroll
        for (int l = 0; l < LC; ++l) {
          if (smask & (1u << l)) {
            const bool fh = hmask & (1u << l);
            const int off = goff[l] + (fh ? zt_halo : ((zmask & (1u << l)) ? zt_clamp : zt_int));
            const float* src = (fh ? P.halo : P.Uin) + off;
            const size_t fs = fh ? fs_halo : fs_int;
            float* d = dst + (at + l * NA) * REC;
            const int dx = (dmask >> l) & 1;
#pragma unroll
            for (int q = 0; q < NF; ++q) { cp_async4(d + 2 * q, src + q * fs); cp_async4(d + 2 * q + 1, src + q * fs + dx); }
          }
        }
      }
    };
    // O1 in place: conserved -> primitive, each thread on the pairs it copied
    auto convert_plane = [&](float* dst) {
#pragma unroll
      for (int l = 0; l < LC; ++l) {
        if (lmask & (1u << l)) {
          float* d = dst + (at + l * NA) * REC;
          F2 u[NF];
          lds_pairs<NF>(d, u);
          const F2 ir = rcp2(u[0]);
          const F2 vx = u[1] * ir, vy = u[2] * ir, vz = u[3] * ir;
          F2 e2 = u[0] * fma(vx, vx, fma(vy, vy, vz * vz));            // rho |v|^2
          if (NF == 9) e2 = e2 + fma(u[5], u[5], fma(u[6], u[6], u[7] * u[7]));
          const F2 pr = P.gm1 * fma(e2, -0.5f, u[4]);
          // (vx | vy vz | p) sit at floats 2..9 of the record: one 64-bit, one 128-bit, one 64-bit store
          *reinterpret_cast<float2*>(d + 2) = vx.v;
          *reinterpret_cast<float4*>(d + 4) = make_float4(vy.v.x, vy.v.y, vz.v.x, vz.v.y);
          *reinterpret_cast<float2*>(d + 8) = pr.v;
        }
      }
    };

    // ---- ring role: one pair of the tile grown by one layer (no corners) ----------------------------
    //   [0, TY)        right x ring (px = HX + 1, cells TX, TX+1): predictor, the tile's last x face (lo)
    //   + TY           left x ring (px = 0, cells -2, -1): predictor, publishes W^+_x of cell -1 (hi)
    //   + HX           bottom y ring (pj = -1): predictor, publishes W^+_y
    //   + HX           top y ring (pj = TY): predictor, the tile's last y faces
    // (in this order the right ring sits in the first aux warp and the top ring in the second for both tile
    // shapes, so that each aux warp solves one set of faces per plane)
    int pj = 0, px = 1;
    bool vlo = true, vhi = true;  // which cells of the pair are real
    if (at < TY) { pj = at; px = HX + 1; vhi = false; }
    else if (at < 2 * TY) { pj = at - TY; px = 0; vlo = false; }
    else if (at < 2 * TY + HX) { pj = -1; px = at - 2 * TY + 1; }
    else if (at < 2 * TY + 2 * HX) { pj = TY; px = at - (2 * TY + HX) + 1; }
    const bool pred = at < 2 * TY + 2 * HX;
    const bool right = at < TY, left = pred && px == 0, top = pred && pj == TY, bottom = pred && pj == -1;
    const int rc = ((pj + 2) * NPX + px) * REC;
    float* const xslot = XP + ((right || left) ? pj * (HX + 1) + (right ? HX : 0) : 0) * REC;
    float* const yslot = YP + ((top || bottom) ? (top ? TY * HX : 0) + px - 1 : 0) * REC;
    F2 wm[NF];  // right ring: W^-_x (lo half real); top ring: W^-_y
#pragma unroll
    for (int q = 0; q < NF; ++q) wm[q] = F2(0.f);

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
      // ---- phase 1: predictor of the ring pairs, publish W^+ ----------------------------------------
      if (mid && pred) {
        F2 ws[NF], hx[NF], hy[NF], hz[NF];
        predict_pair<NF, LIM>(Wm, Wc, Wp, rc, NPX * REC, REC, P, ms, B2(vlo, vhi), ws, hx, hy, hz);
        if (left) {
          // W^+_x of cell -1 = the .x halves of the first pair's left-state record (that pair writes the .y halves)
#pragma unroll
          for (int q = 0; q < NF; ++q) xslot[2 * q] = ws[q].v.y + hx[q].v.y;
        } else if (bottom) {
          F2 o[NF], r[NF];
#pragma unroll
          for (int q = 0; q < NF; ++q) o[q] = ws[q] + hy[q];
          rot_in<NF, 1>(o, r);            // y solver's component order
          sts_pairs<NF>(yslot, r);
        } else if (right) {
#pragma unroll
          for (int q = 0; q < NF; ++q) wm[q] = ws[q] - hx[q];
        } else {
          F2 o[NF];
#pragma unroll
          for (int q = 0; q < NF; ++q) o[q] = ws[q] - hy[q];
          rot_in<NF, 1>(o, wm);
        }
      }
      prefetch_plane(kk + 2);
      __syncthreads();

      // ---- phase 2: copies of plane kk+2 into the slot plane kk-1 vacated; the tile's last x / y faces;
      //      convert plane kk+2 when it has landed (these warps have the slack to wait for it) ---------
      issue_plane(kk + 2, Wm);
      cp_commit();
      if (mid && (right || top)) {
        // ONE solver instance for the tile's last x faces (right ring: lo half real) and last y faces (top ring):
        // the kernel is bound by instruction fetch (profiles/r1c), these warps have the slack for the few moves
        // that bring the two roles' operands into the same registers
        // (operands arrive in the solver's component order: identity for x, rotated for y)
        F2 WL[NF], Fr[NF];
        lds_pairs<NF>(right ? xslot : yslot, WL);
        if (right) {   // only the lo face (TX - 1/2) is real: its left state is the .x half the last interior pair wrote
#pragma unroll
          for (int q = 0; q < NF; ++q) WL[q] = F2(WL[q].v.x, WL[q].v.x);
        }
        riemann2<NF, RS>(WL, wm, RC, Fr, B2(true, !right), s_cnt);
        sts_pairs<NF>(right ? xslot : yslot, Fr);
        if (X2_UNLIKELY(blk >= 0)) {
          if (right && x0 + TX == n) {  // the patch's last x face (a7)
            F2 f[NF];
            rot_out<NF, 0>(Fr, f);
            float* dstF = P.fblk + ((size_t)blk * 3 + 0) * NF * fsz + ((size_t)2 * n2 + (size_t)(kk * n + (y0 + pj)));
#pragma unroll
            for (int q = 0; q < NF; ++q) atomicAdd(dstF + (size_t)q * fsz, f[q].v.x);
          } else if (!right && y0 + TY == n) {
            F2 f[NF];
            rot_out<NF, 1>(Fr, f);
            float* dstF = P.fblk + ((size_t)blk * 3 + 1) * NF * fsz + ((size_t)2 * n2 + (size_t)(kk * n + (x0 + 2 * (px - 1))));
#pragma unroll
            for (int q = 0; q < NF; ++q) { atomicAdd(dstF + (size_t)q * fsz, f[q].v.x); atomicAdd(dstF + (size_t)q * fsz + 1, f[q].v.y); }
          }
        }
      }
      cp_wait<0>();
      convert_plane(Wm);
      __syncthreads();
      float* tmp = Wm; Wm = Wc; Wc = Wp; Wp = tmp;
    }
  }

  __syncthreads();
  if (tid == 0) {
    float m = s_red[0];
#pragma unroll
    for (int wv = 1; wv < NI / 32; ++wv) m = fmaxf(m, s_red[wv]);
    atomicMax(reinterpret_cast<unsigned int*>(P.smax), __float_as_uint(m));
  }
  if (tid < 4 && s_cnt[tid] != 0) atomicAdd(P.counters + tid, (unsigned long long)s_cnt[tid]);
}

// host-side launcher for one (NF, TX, TY, NT, MAXR) tile configuration
template <int NF, int LIM, int RS, int TX, int TY, int NT, int MAXR>
cudaError_t launch_variant_x2(const StepParams<float>& P, cudaStream_t s) {
  using G = GeomX2<NF, TX, TY>;
  auto kern = godunov_step_x2_kernel<NF, LIM, RS, TX, TY, NT, MAXR>;
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
      fprintf(stderr, "amr: x2 step kernel launch failed: %d threads, %d regs/thread, %zu B dynamic + %zu B static smem\n",
              NT, fa.numRegs, (size_t)G::smem_bytes, fa.sharedSizeBytes);
  }
  return le;
}

template <int NF, int TX, int TY, int NT, int MAXR>
cudaError_t launch_dispatch_x2(const StepParams<float>& P, int limiter, int riemann, cudaStream_t s) {
  constexpr int RSX = (NF == 5) ? X2_RS_HLLC : X2_RS_HLLD;
#define AMR_CASE(L, R) \
  if (limiter == L && riemann == R) return launch_variant_x2<NF, L, R, TX, TY, NT, MAXR>(P, s);
  AMR_CASE(X2_LIM_NONE, X2_RS_HLL)
  AMR_CASE(X2_LIM_MINMOD, X2_RS_HLL)
  AMR_CASE(X2_LIM_MC, X2_RS_HLL)
  AMR_CASE(X2_LIM_NONE, RSX)
  AMR_CASE(X2_LIM_MINMOD, RSX)
  AMR_CASE(X2_LIM_MC, RSX)
#undef AMR_CASE
  return cudaErrorInvalidValue;
}

}  // namespace x2
}  // namespace amr

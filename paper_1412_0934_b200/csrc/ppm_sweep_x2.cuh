// PPM hydro sweep, fp32, TWO PENCILS PER THREAD with packed f32x2 arithmetic (pair_math.cuh): the same reading R-PPM
// and the same formulas as ppm_sweep.cuh, in the branch-free form the packed
// PLM kernel uses - the two pencils of a pair generally take different branches of the limiter, the monotonisation
// and the characteristic tracing, so every decision is a select on a per-half mask; the wave corrections are
// computed for every wave and multiplied by 0 where the wave runs away from the face.
//
// Why (profiles/r2c): the one-cell-per-thread sweep is bound by instruction issue (35 warp-instructions per cell and
// sweep, issue slots 75 % busy), not by HBM; sm_100a issues FADD2 / FMUL2 / FFMA2 on a register pair in one slot.
//
// Work decomposition: one CTA owns 16 neighbouring pencils of one patch = 8 pairs, a pair = two pencils adjacent along
// the fast transverse axis (x for the y and z sweeps: one 8-byte access per field and cell; y for the x sweep).  Thread
// (pair, s) owns the cells s - 1 of its two pencils, s = 0 .. n+1.  2-D block, x along the memory-contiguous axis.
// Patch sizes that are not a multiple of 16 run the scalar kernel.
#pragma once
#include <cuda_runtime.h>

#include "amr_internal.hpp"
#include "godunov_step.cuh"
#include "ppm_params.hpp"
#include "riemann_x2.cuh"

namespace amr {
namespace ppm {

using x2::F2;
using x2::B2;

constexpr int PP = 8;  // pencil pairs per CTA

// P1: limited slope (CW84 1.7-1.8), both halves
__device__ __forceinline__ F2 limited_dm2(F2 l, F2 c, F2 r) {
  const F2 da = 0.5f * (r - l), t1 = c - l, t2 = r - c;
  const F2 m = x2::min3(x2::abs2(da), x2::abs2(2.f * t1), x2::abs2(2.f * t2));
  const B2 mono = x2::gt(t2 * t1, 0.f);
  return x2::sel(mono, F2(copysignf(m.v.x, da.v.x), copysignf(m.v.y, da.v.y)), 0.f);
}

// P1 interface values (1.6) + P2 monotonisation (1.10), both halves
__device__ __forceinline__ void parabola2(F2 am1, F2 a0, F2 ap1, F2 dmm, F2 dm0, F2 dmp, F2& aL, F2& aR) {
  const float sixth = 1.f / 6.f;
  const F2 l = (am1 + 0.5f * (a0 - am1)) - (dm0 - dmm) * sixth;
  const F2 r = (a0 + 0.5f * (ap1 - a0)) - (dmp - dm0) * sixth;
  const B2 flat = !x2::gt((r - a0) * (a0 - l), 0.f);
  const F2 d = r - l, mm = a0 - 0.5f * (l + r);
  const F2 dm_ = d * mm, dd6 = (d * d) * sixth;
  const B2 c2 = x2::gt(dm_, dd6);
  const B2 c3 = x2::gt(-dd6, dm_) & !c2;
  const F2 l3 = 3.f * a0 - 2.f * r, r3 = 3.f * a0 - 2.f * l;
  aL = x2::sel(flat, a0, x2::sel(c2, l3, l));
  aR = x2::sel(flat, a0, x2::sel(c3, r3, r));
}

#ifndef PPM_X2_MAXR
#define PPM_X2_MAXR 72   /* 3 CTAs of 9 warps per SM; 96 (no spills, 2 CTAs) and 64 (4 CTAs, 180 B of spills) are slower: 17.6 / 15.1 vs 13.9 ms */
#endif
template <int RS, int D>
__global__ void __maxnreg__(PPM_X2_MAXR) ppm_sweep_x2_kernel(const __grid_constant__ SweepParams<float> P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = P.n, n2 = n * n, n3 = n2 * n;
  const int LW = n + 6, LS = n + 2, LF = n + 1;
  float2* const W = reinterpret_cast<float2*>(smem_raw);   // [5][PP][n+6] primitives of the pair, cells -3 .. n+2
  float2* const Wp = W + 5 * PP * LW;                      // [5][PP][n+2] traced upper-face states, sweep order
  float2* const Wm = Wp + 5 * PP * LS;                     // [5][PP][n+2] traced lower-face states
  float2* const F = Wm + 5 * PP * LS;                      // [5][PP][n+1] fluxes through the lower faces of cells 0 .. n
  __shared__ int s_cnt[4];
  __shared__ int s_nb[2];

  const int tid = threadIdx.y * blockDim.x + threadIdx.x;
  const int pen = D == 0 ? threadIdx.y : threadIdx.x, s = D == 0 ? threadIdx.x : threadIdx.y;
  const int p = blockIdx.y;
  const int pg0 = blockIdx.x * (2 * PP);   // first pencil of this CTA (pencils of a patch are numbered fast-axis first)
  if (tid < 4) s_cnt[tid] = 0;
  if (tid < 2) {
    const int pw = D == 0 ? 1 : (D == 1 ? 3 : 9);
    s_nb[tid] = P.nbr[p * 27 + 13 + (tid ? pw : -pw)];
  }
  __syncthreads();

  constexpr int qu = 1 + D, qv = 1 + (D + 1) % 3, qw = 1 + (D + 2) % 3;
  const int sd = D == 0 ? 1 : (D == 1 ? n : n2);    // stride along the sweep inside a patch
  const int pd = D == 0 ? n : 1;                    // stride between the two pencils of a pair inside a patch
  const size_t fs = (size_t)P.np * n3;
  const int M = n + 2 * P.g, M2 = M * M;
  const size_t fsh = (size_t)P.np * M2 * M;
  // 16 divides n: the CTA's pencils share the slow transverse coordinate a1; a0 = fast transverse coordinate (even)
  const int a1 = pg0 / n, a0 = pg0 - a1 * n + 2 * pen;
  const int base = D == 0 ? (a1 * n + a0) * n : (D == 1 ? a1 * n2 + a0 : a1 * n + a0);

  // ---- load + O1: cells -3 .. n+2 of the pair -> primitives ---------------------------------------------------------
  for (int sp = s; sp < LW; sp += LS) {
    const int c = sp - 3;
    F2 u[5];
    if (c >= 0 && c < n) {
      const float* src = P.Uin + (size_t)p * n3 + base + c * sd;
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        if (D != 0) u[q].v = *reinterpret_cast<const float2*>(src + q * fs);   // a0 even: 8-byte aligned
        else u[q] = F2(src[q * fs], src[q * fs + pd]);
      }
    } else {
      const int ent = s_nb[c < 0 ? 0 : 1];
      if (ent == NBR_FROM_HALO) {
        int ix, iy, iz;
        if (D == 0) { ix = c; iy = a0; iz = a1; } else if (D == 1) { ix = a0; iy = c; iz = a1; } else { ix = a0; iy = a1; iz = c; }
        const float* src = P.halo + (size_t)p * M2 * M + ((size_t)(iz + P.g) * M + (iy + P.g)) * M + (ix + P.g);
        const int hd = D == 0 ? M : 1;
#pragma unroll
        for (int q = 0; q < 5; ++q) u[q] = F2(src[q * fsh], src[q * fsh + hd]);
      } else {
        const int spatch = ent & NBR_PATCH_MASK, mode = ent >> NBR_MODE_SHIFT;
        const int cc = ((mode >> D) & 1) ? (c < 0 ? 0 : n - 1) : (c < 0 ? c + n : c - n);
        const float* src = P.Uin + (size_t)spatch * n3 + base + cc * sd;
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          if (D != 0) u[q].v = *reinterpret_cast<const float2*>(src + q * fs);
          else u[q] = F2(src[q * fs], src[q * fs + pd]);
        }
      }
    }
    const F2 ir = x2::rcp2(u[0]);
    const F2 vx = u[1] * ir, vy = u[2] * ir, vz = u[3] * ir;
    const F2 pr = P.gm1 * (u[4] - (0.5f * u[0]) * (vx * vx + vy * vy + vz * vz));
    float2* w = W + pen * LW + sp;
    w[0] = u[0].v; w[PP * LW] = vx.v; w[2 * PP * LW] = vy.v; w[3 * PP * LW] = vz.v; w[4 * PP * LW] = pr.v;
    if (s >= 4) break;
  }
  __syncthreads();

  // ---- P1..P4: traced states of the cells -1 .. n of the pair ----------------------------------------------------------
  {
    const int order[5] = {0, qu, qv, qw, 4};
    F2 a[5], aL[5], aR[5], Da[5], a6[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      const float2* w = W + (order[m] * PP + pen) * LW + (s + 2);   // cell s-1 sits at position s+2
      F2 wm2, wm1, w0, wp1, wp2;
      wm2.v = w[-2]; wm1.v = w[-1]; w0.v = w[0]; wp1.v = w[1]; wp2.v = w[2];
      a[m] = w0;
      parabola2(wm1, w0, wp1, limited_dm2(wm2, wm1, w0), limited_dm2(wm1, w0, wp1), limited_dm2(w0, wp1, wp2), aL[m], aR[m]);
      Da[m] = aR[m] - aL[m];
      a6[m] = 6.f * (a[m] - 0.5f * (aL[m] + aR[m]));
    }
    const float twothirds = 2.f / 3.f;
    auto Ip = [&](int m, F2 sg) { return aR[m] - (0.5f * sg) * (Da[m] - (F2(1.f) - twothirds * sg) * a6[m]); };
    auto Im = [&](int m, F2 sg) { return aL[m] + (0.5f * sg) * (Da[m] + (F2(1.f) - twothirds * sg) * a6[m]); };
    const F2 rho = a[0], u = a[1], pr = a[4];
    const F2 irho = x2::rcp2(rho);
    const F2 cs = x2::sqrt2((P.gamma * pr) * irho);
    const F2 ics = x2::rcp2(cs), roc = rho * ics, cor = cs * irho, ic2 = ics * ics, c2 = cs * cs;
    const F2 lkm = u - cs, lkp = u + cs;
    const F2 lam = F2(P.dtdx);
    F2 wp[5], wm[5];
    {  // upper face: reference = average for lambda_+ (its own correction is exactly zero), corrections of lambda_-, lambda_0
      const F2 sref = x2::max2(lkp, 0.f) * lam;
      F2 ref[5];
#pragma unroll
      for (int m = 0; m < 5; ++m) ref[m] = Ip(m, sref);
      const B2 am = x2::gt(lkm, 0.f), a0m = x2::gt(u, 0.f);
      const F2 sgm = lkm * lam, sg0 = u * lam;
      const F2 b = x2::sel(am, 0.5f * ((ref[4] - Ip(4, sgm)) * ic2 - roc * (ref[1] - Ip(1, sgm))), 0.f);
      const F2 c0 = x2::sel(a0m, (ref[0] - Ip(0, sg0)) - (ref[4] - Ip(4, sg0)) * ic2, 0.f);
      wp[0] = (ref[0] - b) - c0;
      wp[1] = ref[1] + b * cor;
      wp[2] = x2::sel(a0m, Ip(2, sg0), ref[2]);
      wp[3] = x2::sel(a0m, Ip(3, sg0), ref[3]);
      wp[4] = ref[4] - b * c2;
    }
    {  // lower face: reference = average for lambda_-, corrections of lambda_0, lambda_+
      const F2 sref = x2::max2(-lkm, 0.f) * lam;
      F2 ref[5];
#pragma unroll
      for (int m = 0; m < 5; ++m) ref[m] = Im(m, sref);
      const B2 a0m = x2::lt(u, 0.f), ap = x2::lt(lkp, 0.f);
      const F2 sg0 = -(u * lam), sgp = -(lkp * lam);
      const F2 c0 = x2::sel(a0m, (ref[0] - Im(0, sg0)) - (ref[4] - Im(4, sg0)) * ic2, 0.f);
      const F2 b = x2::sel(ap, 0.5f * (roc * (ref[1] - Im(1, sgp)) + (ref[4] - Im(4, sgp)) * ic2), 0.f);
      wm[0] = (ref[0] - c0) - b;
      wm[1] = ref[1] - b * cor;
      wm[2] = x2::sel(a0m, Im(2, sg0), ref[2]);
      wm[3] = x2::sel(a0m, Im(3, sg0), ref[3]);
      wm[4] = ref[4] - b * c2;
    }
    const F2 inf = F2(CUDART_INF_F);
    const B2 ok = x2::gt(wp[0], 0.f) & x2::gt(wp[4], 0.f) & x2::gt(wm[0], 0.f) & x2::gt(wm[4], 0.f) & x2::lt(wp[0], inf) &
                  x2::lt(wp[4], inf) & x2::lt(wm[0], inf) & x2::lt(wm[4], inf);
    const B2 bad = !ok;
    if (X2_UNLIKELY(x2::any(bad))) {
      atomicAdd(&s_cnt[CNT_POSITIVITY], (int)bad.x + (int)bad.y);
#pragma unroll
      for (int m = 0; m < 5; ++m) { wp[m] = x2::sel(bad, a[m], wp[m]); wm[m] = x2::sel(bad, a[m], wm[m]); }
    }
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      Wp[(m * PP + pen) * LS + s] = wp[m].v;
      Wm[(m * PP + pen) * LS + s] = wm[m].v;
    }
  }
  __syncthreads();

  // ---- P5: fluxes through the lower faces of the cells 0 .. n (thread s owns the faces of the cells s of its pair) ----
  if (s <= n) {
    x2::RC2 RC;
    RC.gamma = P.gamma; RC.igm1 = P.igm1; RC.ch2 = 0.f; RC.half_ch = 0.f; RC.half_ich = 0.f; RC.eps = 0.f;
    F2 WL[5], WR[5], Fr[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      WL[m].v = Wp[(m * PP + pen) * LS + s];       // cells s-1
      WR[m].v = Wm[(m * PP + pen) * LS + s + 1];   // cells s
    }
    x2::riemann_hydro2<RS, F2, B2, float>(WL, WR, RC, Fr, B2(true), s_cnt);
#pragma unroll
    for (int m = 0; m < 5; ++m) F[(m * PP + pen) * LF + s] = Fr[m].v;
  }
  __syncthreads();

  // ---- conservative update of the cells 0 .. n-1 of the pair ----------------------------------------------------------
  if (s < n) {
    const size_t cell = (size_t)p * n3 + base + s * sd;
    const int fo[5] = {0, qu, qv, qw, 4};
    const F2 mlam = F2(-P.dtdx);
    F2 rho_new = F2(1.f);
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      const float2* f = F + (m * PP + pen) * LF + s;
      F2 f0, f1, uo;
      f0.v = f[0]; f1.v = f[1];
      const float* in = P.Uin + cell + fo[m] * fs;
      float* out = P.Uout + cell + fo[m] * fs;
      if (D != 0) uo.v = *reinterpret_cast<const float2*>(in); else uo = F2(in[0], in[pd]);
      const F2 un = x2::fma(mlam, f1 - f0, uo);
      if (D != 0) *reinterpret_cast<float2*>(out) = un.v; else { out[0] = un.v.x; out[pd] = un.v.y; }
      if (m == 0) rho_new = un;
    }
    const int neg = (int)!(rho_new.v.x > 0.f) + (int)!(rho_new.v.y > 0.f);
    if (X2_UNLIKELY(neg)) atomicAdd(&s_cnt[CNT_NEG_STATE], neg);
  }
  __syncthreads();
  if (tid < 4 && s_cnt[tid] != 0) atomicAdd(P.counters + tid, (unsigned long long)s_cnt[tid]);
}

inline size_t sweep_x2_smem_bytes(int n) { return sizeof(float2) * 5 * PP * (size_t)((n + 6) + 2 * (n + 2) + (n + 1)); }

template <int RS, int D>
cudaError_t launch_sweep_x2_variant(const SweepParams<float>& P, cudaStream_t s) {
  auto kern = ppm_sweep_x2_kernel<RS, D>;
  static std::atomic<unsigned long long> configured{0};
  const size_t smem = sweep_x2_smem_bytes(P.n);
  {  // up to 160 KB of dynamic shared memory (n = 64), and the shared-memory carve-out that lets several CTAs share an SM
    int dev = 0;
    cudaGetDevice(&dev);
    const bool first = !(configured.load(std::memory_order_acquire) & (1ull << (dev & 63)));
    cudaError_t e = ensure_dynamic_smem((const void*)kern, 160 * 1024, configured);
    if (e == cudaSuccess && first) e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
  }
  const dim3 grid((unsigned)(P.n * P.n / (2 * PP)), (unsigned)P.np_active);
  const dim3 block = D == 0 ? dim3((unsigned)(P.n + 2), PP) : dim3(PP, (unsigned)(P.n + 2));
  kern<<<grid, block, smem, s>>>(P);
  return cudaGetLastError();
}

inline cudaError_t launch_sweep_x2(const SweepParams<float>& P, int riemann, int dir, cudaStream_t s) {
#define AMR_PPM_CASE(R, DD) if (riemann == R && dir == DD) return launch_sweep_x2_variant<R, DD>(P, s);
  AMR_PPM_CASE(x2::X2_RS_HLL, 0) AMR_PPM_CASE(x2::X2_RS_HLL, 1) AMR_PPM_CASE(x2::X2_RS_HLL, 2)
  AMR_PPM_CASE(x2::X2_RS_HLLC, 0) AMR_PPM_CASE(x2::X2_RS_HLLC, 1) AMR_PPM_CASE(x2::X2_RS_HLLC, 2)
#undef AMR_PPM_CASE
  return cudaErrorInvalidValue;
}

}  // namespace ppm
}  // namespace amr

// PPM hydro sweep for sm_100a (SURVEY.md 8(f1); PAPER.md:43 "the Piecewise Parabolic Method, PPM [9]", :76 "the
// PLM/PPM hydro solver, have been ported to NVIDIA's CUDA").  Reading R-PPM: Colella &
// Woodward 1984 in the direct Eulerian, dimensionally split form, hydro only, primitive variables, no optional
// dissipation, the boundary's HLL / HLLC flux.  One launch = one sweep along direction D over every patch:
//   halo of 3 cells along D gathered through the 27-entry neighbour table (sibling / periodic / outflow clamp /
//   prolongation halo buffer)  ->  primitives  ->  P1 interface values (CW84 1.6-1.8)  ->  P2 monotonisation (1.10)
//   ->  P3 + P4 characteristic tracing (1.12, 3.5-3.7)  ->  P5 flux, conservative update.
// Nothing but U_old is read from and U_new written to HBM; every intermediate lives in shared memory / registers.
//
// Work decomposition: one CTA owns PB = 8 neighbouring pencils (lines of n cells along D) of one patch.  Thread
// (pencil, s) owns the cell s - 1 of its pencil, s = 0 .. n+1 (the interior grown by one cell: the traced states of
// the cells -1 and n feed the first and the last face).  Consecutive threads run along x (the memory-contiguous
// axis): along the pencil for D = 0, across the 8 pencils otherwise, so that global loads and stores are 128-byte
// (D = 0) or 32-byte (one sector) segments.  The hot loop is a stream: its roofline is HBM (2 x 5 x sizeof(T) bytes
// per cell and sweep).
#pragma once
#include <cuda_runtime.h>

#include "amr_internal.hpp"
#include "godunov_step.cuh"
#include "ppm_params.hpp"

namespace amr {
namespace ppm {

constexpr int PB = 8;  // pencils per CTA

// P1: the limited slope dm of one cell (CW84 1.7-1.8)
template <class T>
__device__ __forceinline__ T limited_dm(T l, T c, T r) {
  const T da = T(0.5) * (r - l);
  const T m = rmin3(rabs(da), T(2) * rabs(c - l), T(2) * rabs(r - c));
  return ((r - c) * (c - l) > T(0)) ? (da > T(0) ? m : -m) : T(0);
}

// P1 (interface values, CW84 1.6) + P2 (monotonisation, 1.10) of one variable from the cell and its two neighbours
// and their limited slopes
template <class T>
__device__ __forceinline__ void parabola(T am1, T a0, T ap1, T dmm, T dm0, T dmp, T& aL, T& aR) {
  const T sixth = T(1) / T(6);
  T l = am1 + T(0.5) * (a0 - am1) - (dm0 - dmm) * sixth;
  T r = a0 + T(0.5) * (ap1 - a0) - (dmp - dm0) * sixth;
  if ((r - a0) * (a0 - l) <= T(0)) {
    l = a0; r = a0;
  } else {
    const T d = r - l, m = a0 - T(0.5) * (l + r);
    if (d * m > d * d * sixth) l = T(3) * a0 - T(2) * r;
    else if (-(d * d) * sixth > d * m) r = T(3) * a0 - T(2) * l;
  }
  aL = l; aR = r;
}

template <class T, int RS, int D>
__global__ void __launch_bounds__(PB * 66) ppm_sweep_kernel(const __grid_constant__ SweepParams<T> P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = P.n, n2 = n * n, n3 = n2 * n;
  const int LW = n + 6, LS = n + 2, LF = n + 1;
  T* const W = reinterpret_cast<T*>(smem_raw);   // [5][PB][n+6] primitives (rho, vx, vy, vz, p), cells -3 .. n+2
  T* const Wp = W + 5 * PB * LW;                 // [5][PB][n+2] traced upper-face states, sweep order (rho,u,v,w,p)
  T* const Wm = Wp + 5 * PB * LS;                // [5][PB][n+2] traced lower-face states
  T* const F = Wm + 5 * PB * LS;                 // [5][PB][n+1] fluxes through the lower faces of cells 0 .. n
  __shared__ int s_cnt[4];
  __shared__ int s_nb[2];

  // 2-D block, x along the memory-contiguous axis: (s, pencil) for D = 0, (pencil, s) otherwise - no integer division
  const int tid = threadIdx.y * blockDim.x + threadIdx.x;
  const int pen = D == 0 ? threadIdx.y : threadIdx.x, s = D == 0 ? threadIdx.x : threadIdx.y;
  const int p = blockIdx.y;
  const int pg0 = blockIdx.x * PB;   // first pencil of this CTA (pencils of a patch are numbered x-fastest)
  if (tid < 4) s_cnt[tid] = 0;
  if (tid < 2) {
    // neighbour regions across the lower / upper D-face: region index rz*9 + ry*3 + rx, 1 = centre
    const int pw = D == 0 ? 1 : (D == 1 ? 3 : 9);
    s_nb[tid] = P.nbr[p * 27 + 13 + (tid ? pw : -pw)];
  }
  __syncthreads();

  constexpr int qu = 1 + D, qv = 1 + (D + 1) % 3, qw = 1 + (D + 2) % 3;
  const int sd = D == 0 ? 1 : (D == 1 ? n : n2);   // stride along the sweep inside a patch
  const size_t fs = (size_t)P.np * n3;
  const int M = n + 2 * P.g, M2 = M * M;
  const size_t fsh = (size_t)P.np * M2 * M;

  // pencil -> offset of its cell 0 inside a patch, and its two transverse coordinates (for the halo buffer)
  // PB divides n: the CTA's pencils share their slow transverse coordinate a1; a0 = fast transverse coordinate
  const int a1 = pg0 / n, a0 = pg0 - a1 * n + pen;
  const int base = D == 0 ? (a1 * n + a0) * n : (D == 1 ? a1 * n2 + a0 : a1 * n + a0);   // D=0: (y,z); D=1: (x,z); D=2: (x,y)

  // ---- load + O1: cells -3 .. n+2 of the PB pencils -> primitives (thread s: positions s and, for s < 4, LS + s) ----
  for (int sp = s; sp < LW; sp += LS) {
    const int c = sp - 3;   // cell index along D
    const T* src;
    size_t fstride;
    if (c >= 0 && c < n) {
      src = P.Uin + (size_t)p * n3 + base + c * sd;
      fstride = fs;
    } else {
      const int ent = s_nb[c < 0 ? 0 : 1];
      if (ent == NBR_FROM_HALO) {
        int ix, iy, iz;
        if (D == 0) { ix = c; iy = a0; iz = a1; } else if (D == 1) { ix = a0; iy = c; iz = a1; } else { ix = a0; iy = a1; iz = c; }
        src = P.halo + (size_t)p * M2 * M + ((size_t)(iz + P.g) * M + (iy + P.g)) * M + (ix + P.g);
        fstride = fsh;
      } else {
        const int spatch = ent & NBR_PATCH_MASK, mode = ent >> NBR_MODE_SHIFT;
        const int cc = ((mode >> D) & 1) ? (c < 0 ? 0 : n - 1) : (c < 0 ? c + n : c - n);
        src = P.Uin + (size_t)spatch * n3 + base + cc * sd;
        fstride = fs;
      }
    }
    const T rho = src[0], mx = src[fstride], my = src[2 * fstride], mz = src[3 * fstride], E = src[4 * fstride];
    const T ir = rrcp(rho);
    const T vx = mx * ir, vy = my * ir, vz = mz * ir;
    const T pr = P.gm1 * (E - T(0.5) * rho * (vx * vx + vy * vy + vz * vz));
    T* w = W + pen * LW + sp;
    w[0] = rho; w[PB * LW] = vx; w[2 * PB * LW] = vy; w[3 * PB * LW] = vz; w[4 * PB * LW] = pr;
    if (s >= 4) break;
  }
  __syncthreads();

  // ---- P1..P4: traced states of the cells -1 .. n ------------------------------------------------------------
  const bool active = true;
  {
    const int order[5] = {0, qu, qv, qw, 4};
    T a[5], aL[5], aR[5], Da[5], a6[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      const T* w = W + (order[m] * PB + pen) * LW + (s + 2);   // cell s-1 sits at position s+2
      a[m] = w[0];
      // the three limited slopes are recomputed here: staging them once per cell in shared memory (one more phase and
      // barrier) was measured slower, 17.8 vs 16.2 ms per 512^3 step
      parabola<T>(w[-1], w[0], w[1], limited_dm<T>(w[-2], w[-1], w[0]), limited_dm<T>(w[-1], w[0], w[1]),
                  limited_dm<T>(w[0], w[1], w[2]), aL[m], aR[m]);
      Da[m] = aR[m] - aL[m];
      a6[m] = T(6) * (a[m] - T(0.5) * (aL[m] + aR[m]));
    }
    const T twothirds = T(2) / T(3);
    auto Ip = [&](int m, T sg) { return aR[m] - T(0.5) * sg * (Da[m] - (T(1) - twothirds * sg) * a6[m]); };
    auto Im = [&](int m, T sg) { return aL[m] + T(0.5) * sg * (Da[m] + (T(1) - twothirds * sg) * a6[m]); };
    const T rho = a[0], u = a[1], pr = a[4];
    const T cs = rsqrt_(P.gamma * pr * rrcp(rho));
    const T ics = rrcp(cs), roc = rho * ics, cor = cs * rrcp(rho), ic2 = ics * ics, c2 = cs * cs;
    const T lk[3] = {u - cs, u, u + cs};
    const T lam = P.dtdx;
    T wp[5], wm[5];
    {
      const T sref = rmax(lk[2], T(0)) * lam;
      T ref[5];
#pragma unroll
      for (int m = 0; m < 5; ++m) { ref[m] = Ip(m, sref); wp[m] = ref[m]; }
      if (lk[0] > T(0)) {
        const T sg = lk[0] * lam;
        const T b = T(0.5) * (-roc * (ref[1] - Ip(1, sg)) + (ref[4] - Ip(4, sg)) * ic2);
        wp[0] -= b; wp[1] += b * cor; wp[4] -= b * c2;
      }
      if (lk[1] > T(0)) {
        const T sg = lk[1] * lam;
        wp[0] -= (ref[0] - Ip(0, sg)) - (ref[4] - Ip(4, sg)) * ic2;
        wp[2] = Ip(2, sg); wp[3] = Ip(3, sg);
      }
      // (the lambda_+ wave: its average IS the reference state, its correction is exactly zero)
    }
    {
      const T sref = rmax(-lk[0], T(0)) * lam;
      T ref[5];
#pragma unroll
      for (int m = 0; m < 5; ++m) { ref[m] = Im(m, sref); wm[m] = ref[m]; }
      // (the lambda_- wave: its average IS the reference state, its correction is exactly zero)
      if (lk[1] < T(0)) {
        const T sg = -lk[1] * lam;
        wm[0] -= (ref[0] - Im(0, sg)) - (ref[4] - Im(4, sg)) * ic2;
        wm[2] = Im(2, sg); wm[3] = Im(3, sg);
      }
      if (lk[2] < T(0)) {
        const T sg = -lk[2] * lam;
        const T b = T(0.5) * (roc * (ref[1] - Im(1, sg)) + (ref[4] - Im(4, sg)) * ic2);
        wm[0] -= b; wm[1] -= b * cor; wm[4] -= b * c2;
      }
    }
    const T inf = rinf<T>();
    const bool ok = (wp[0] > T(0)) && (wp[4] > T(0)) && (wm[0] > T(0)) && (wm[4] > T(0)) && (wp[0] < inf) &&
                    (wp[4] < inf) && (wm[0] < inf) && (wm[4] < inf);
    if (!ok) {
      atomicAdd(&s_cnt[CNT_POSITIVITY], 1);
#pragma unroll
      for (int m = 0; m < 5; ++m) wp[m] = wm[m] = a[m];
    }
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      Wp[(m * PB + pen) * LS + s] = wp[m];
      Wm[(m * PB + pen) * LS + s] = wm[m];
    }
  }
  __syncthreads();

  // ---- P5: flux through the lower face of the cells 0 .. n (thread s owns the face of the cell s) -------------
  if (active && s <= n) {
    RiemannConst<T> RC;
    RC.gamma = P.gamma; RC.igm1 = P.igm1; RC.ch2 = T(0); RC.half_ch = T(0); RC.half_ich = T(0); RC.eps = T(0);
    T WL[5], WR[5], Fr[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      WL[m] = Wp[(m * PB + pen) * LS + s];       // cell s-1
      WR[m] = Wm[(m * PB + pen) * LS + s + 1];   // cell s
    }
    riemann_hydro<T, RS>(WL, WR, RC, Fr, s_cnt);
#pragma unroll
    for (int m = 0; m < 5; ++m) F[(m * PB + pen) * LF + s] = Fr[m];
  }
  __syncthreads();

  // ---- conservative update of the cells 0 .. n-1 ------------------------------------------------------------------
  if (active && s < n) {
    const size_t cell = (size_t)p * n3 + base + s * sd;
    const int fo[5] = {0, qu, qv, qw, 4};
    T rho_new = T(1);
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      const T* f = F + (m * PB + pen) * LF + s;
      const T un = P.Uin[cell + fo[m] * fs] - P.dtdx * (f[1] - f[0]);
      P.Uout[cell + fo[m] * fs] = un;
      if (m == 0) rho_new = un;
    }
    if (!(rho_new > T(0))) atomicAdd(&s_cnt[CNT_NEG_STATE], 1);
  }
  __syncthreads();
  if (tid < 4 && s_cnt[tid] != 0) atomicAdd(P.counters + tid, (unsigned long long)s_cnt[tid]);
}

template <class T>
size_t sweep_smem_bytes(int n) { return sizeof(T) * 5 * PB * (size_t)((n + 6) + 2 * (n + 2) + (n + 1)); }

template <class T, int RS, int D>
cudaError_t launch_sweep_variant(const SweepParams<T>& P, cudaStream_t s) {
  auto kern = ppm_sweep_kernel<T, RS, D>;
  static std::atomic<unsigned long long> configured{0};
  const size_t smem = sweep_smem_bytes<T>(P.n);
  if (smem > 48 * 1024) {
    cudaError_t e = ensure_dynamic_smem((const void*)kern, 160 * 1024, configured);
    if (e != cudaSuccess) return e;
  }
  const dim3 grid((unsigned)(P.n * P.n / PB), (unsigned)P.np_active);
  const dim3 block = D == 0 ? dim3((unsigned)(P.n + 2), PB) : dim3(PB, (unsigned)(P.n + 2));
  kern<<<grid, block, smem, s>>>(P);
  return cudaGetLastError();
}

template <class T>
cudaError_t launch_sweep(const SweepParams<T>& P, int riemann, int dir, cudaStream_t s) {
#define AMR_PPM_CASE(R, DD) if (riemann == R && dir == DD) return launch_sweep_variant<T, R, DD>(P, s);
  AMR_PPM_CASE(RS_HLL, 0) AMR_PPM_CASE(RS_HLL, 1) AMR_PPM_CASE(RS_HLL, 2)
  AMR_PPM_CASE(RS_HLLC, 0) AMR_PPM_CASE(RS_HLLC, 1) AMR_PPM_CASE(RS_HLLC, 2)
#undef AMR_PPM_CASE
  return cudaErrorInvalidValue;
}

}  // namespace ppm
}  // namespace amr

// O7 (reading A9): max over directions of |v_d| + c_d for one cell, from its conserved state.
// Used by the fused epilogue of the step kernels and by the standalone reduction (amr_cfl_dt); written
// with explicitly rounded intrinsics (no FMA contraction) so that all kernels give bitwise the same
// number for the same stored state (pin P15).  T = double: SFU seed + two Newton steps (fast_rcp,
// fast_sqrt below, <= 2 ulp).  T = float and T = x2::F2 (two cells at once): the SFU reciprocal and
// square root (<= 2 ulp each, deterministic), like the rest of the fp32 path; the packed *_rn operations round exactly like the scalar ones, so the F2
// instantiation gives the float one's bits in each half.
#pragma once
#include <cuda_runtime.h>

#include "pair_math.cuh"

namespace amr {

// fp64: MUFU seed (rcp / rsqrt.approx.ftz.f64, ~20 bits) + two Newton steps, <= 2 ulp, no slow-path
// branch (the IEEE sequences cost ~3x the instructions and a divergent special-case check each; operands
// here are normal-range positive numbers or differences of wave speeds).  rsqrt_(0) returns 0.
__device__ __forceinline__ double fast_rcp(double a) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));
  double e = fma(-a, r, 1.0);
  r = fma(r, e, r);
  e = fma(-a, r, 1.0);
  return fma(r, e, r);
}
// g ~ sqrt(a), 2 h ~ 1/sqrt(a) (coupled Newton iteration)
__device__ __forceinline__ void sqrt_pair(double a, double& g, double& h) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
  g = a * y;
  h = 0.5 * y;
  double r = fma(-g, h, 0.5);
  g = fma(g, r, g);
  h = fma(h, r, h);
  r = fma(-g, h, 0.5);
  g = fma(g, r, g);
  h = fma(h, r, h);
}
__device__ __forceinline__ double fast_sqrt(double a) {
  double g, h;
  sqrt_pair(a > 1e-300 ? a : 1e-300, g, h);
  return a > 1e-300 ? g : 0.0;
}

__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float div_rn(float a, float b) { return __fmul_rn(a, x2::rcpf(b)); }
__device__ __forceinline__ double div_rn(double a, double b) { return __dmul_rn(a, fast_rcp(b)); }
__device__ __forceinline__ float sqrt_rn(float a) { return x2::sqrtf_(a); }
__device__ __forceinline__ double sqrt_rn(double a) { return fast_sqrt(a); }
__device__ __forceinline__ float max_(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ double max_(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float abs_(float a) { return fabsf(a); }
__device__ __forceinline__ double abs_(double a) { return fabs(a); }
__device__ __forceinline__ x2::F2 mul_rn(x2::F2 a, x2::F2 b) { return a * b; }
__device__ __forceinline__ x2::F2 add_rn(x2::F2 a, x2::F2 b) { return a + b; }
__device__ __forceinline__ x2::F2 div_rn(x2::F2 a, x2::F2 b) { return a * x2::rcp2(b); }
__device__ __forceinline__ x2::F2 sqrt_rn(x2::F2 a) { return x2::sqrt2(a); }
__device__ __forceinline__ x2::F2 max_(x2::F2 a, x2::F2 b) { return x2::max2(a, b); }
__device__ __forceinline__ x2::F2 abs_(x2::F2 a) { return x2::abs2(a); }

template <class T, int NF>
__device__ __forceinline__ T signal_speed(const T* u, T gamma, T gm1) {
  const T rho = u[0];
  const T vx = div_rn(u[1], rho), vy = div_rn(u[2], rho), vz = div_rn(u[3], rho);
  const T v2 = add_rn(add_rn(mul_rn(vx, vx), mul_rn(vy, vy)), mul_rn(vz, vz));
  const T ke = mul_rn(mul_rn(T(0.5), rho), v2);
  const T vmax = max_(max_(abs_(vx), abs_(vy)), abs_(vz));
  if (NF == 5) {
    const T pr = mul_rn(gm1, add_rn(u[4], -ke));
    const T c = sqrt_rn(div_rn(mul_rn(gamma, pr), rho));
    return add_rn(vmax, c);  // c is the same in all directions
  } else {
    const T bx2 = mul_rn(u[5], u[5]), by2 = mul_rn(u[6], u[6]), bz2 = mul_rn(u[7], u[7]);
    const T B2 = add_rn(add_rn(bx2, by2), bz2);
    const T pr = mul_rn(gm1, add_rn(add_rn(u[4], -ke), -mul_rn(T(0.5), B2)));
    const T gp = mul_rn(gamma, pr);
    const T a = div_rn(add_rn(gp, B2), rho);
    const T a2 = mul_rn(a, a);
    const T k = div_rn(mul_rn(T(4), gp), mul_rn(rho, rho));  // 4 gamma p / rho^2
    const T cx = sqrt_rn(mul_rn(T(0.5), add_rn(a, sqrt_rn(max_(add_rn(a2, -mul_rn(k, bx2)), T(0))))));
    const T cy = sqrt_rn(mul_rn(T(0.5), add_rn(a, sqrt_rn(max_(add_rn(a2, -mul_rn(k, by2)), T(0))))));
    const T cz = sqrt_rn(mul_rn(T(0.5), add_rn(a, sqrt_rn(max_(add_rn(a2, -mul_rn(k, bz2)), T(0))))));
    return max_(max_(add_rn(abs_(vx), cx), add_rn(abs_(vy), cy)), add_rn(abs_(vz), cz));
  }
}

}  // namespace amr

// The operation set of pair_math.cuh for ONE fp64 value per thread, so that the branch-free Riemann solvers of
// riemann_x2.cuh (templates on the value type) and the structure of the x2 step kernel serve the fp64 path too
// (godunov_step_d1.cuh).  fp64 has no packed instructions: these are plain scalar operations; min / max are
// compare-selects (fmin/fmax cost 8 instructions in fp64), reciprocal and square root the SFU-seeded Newton
// iterations of signal_speed.cuh (<= 2 ulp, no slow-path branch).  Masks are plain bool.
#pragma once
#include "pair_math.cuh"
#include "signal_speed.cuh"

namespace amr {
namespace x2 {

__device__ __forceinline__ double fma(double a, double b, double c) { return ::fma(a, b, c); }
__device__ __forceinline__ double fms(double a, double b, double c) { return ::fma(a, b, -c); }
__device__ __forceinline__ double fnma(double a, double b, double c) { return ::fma(-a, b, c); }
__device__ __forceinline__ double abs2(double a) { return fabs(a); }
__device__ __forceinline__ double min2(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double max2(double a, double b) { return a > b ? a : b; }
__device__ __forceinline__ double min3(double a, double b, double c) { return min2(min2(a, b), c); }
__device__ __forceinline__ double max3(double a, double b, double c) { return max2(max2(a, b), c); }
__device__ __forceinline__ double rcp2(double a) { return fast_rcp(a); }
__device__ __forceinline__ double sqrt2(double a) { return fast_sqrt(a); }
__device__ __forceinline__ bool gt(double a, double b) { return a > b; }
__device__ __forceinline__ bool ge(double a, double b) { return a >= b; }
__device__ __forceinline__ bool lt(double a, double b) { return a < b; }
__device__ __forceinline__ bool any(bool a) { return a; }
__device__ __forceinline__ double sel(bool m, double a, double b) { return m ? a : b; }
__device__ __forceinline__ int count_true(bool a) { return (int)a; }
__device__ __forceinline__ int count_true(B2 a) { return (int)a.x + (int)a.y; }

}  // namespace x2
}  // namespace amr

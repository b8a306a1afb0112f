// Packed fp32 pairs for sm_100a: one F2 holds the same quantity of two x-adjacent cells (lo = even cell,
// hi = odd cell) in an aligned register pair, so that add / mul / fma issue as FADD2 / FMUL2 / FFMA2 (one
// issue slot for two lanes; measured on B200: 0.5 packed instructions per clock per scheduler = the same
// flops as scalar FFMA at half the issue slots, profiles/r1b_step_mhd_f32_ncu.md).  min / max / compare /
// select / MUFU have no packed form and are done per half.  Every operation is the IEEE round-to-nearest
// one (the *_rn intrinsics are never contracted), so a formula gives the same bits in either half and on
// either side of a tile boundary; fused multiply-adds are written out explicitly with fma().
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>

#define X2_UNLIKELY(x) __builtin_expect((x), 0)

namespace amr {
namespace x2 {

struct F2 {
  float2 v;
  __device__ __forceinline__ F2() {}
  __device__ __forceinline__ F2(float s) { v.x = s; v.y = s; }  // broadcast (a scalar operand in SASS)
  __device__ __forceinline__ F2(float lo, float hi) { v.x = lo; v.y = hi; }
};
struct B2 {
  bool x, y;
  __device__ __forceinline__ B2() {}
  __device__ __forceinline__ B2(bool a) : x(a), y(a) {}
  __device__ __forceinline__ B2(bool a, bool b) : x(a), y(b) {}
};

__device__ __forceinline__ F2 operator-(F2 a) { return F2(-a.v.x, -a.v.y); }
__device__ __forceinline__ F2 operator+(F2 a, F2 b) { F2 r; r.v = __fadd2_rn(a.v, b.v); return r; }
__device__ __forceinline__ F2 operator-(F2 a, F2 b) { F2 r; r.v = __fadd2_rn(a.v, make_float2(-b.v.x, -b.v.y)); return r; }
__device__ __forceinline__ F2 operator*(F2 a, F2 b) { F2 r; r.v = __fmul2_rn(a.v, b.v); return r; }
__device__ __forceinline__ F2 fma(F2 a, F2 b, F2 c) { F2 r; r.v = __ffma2_rn(a.v, b.v, c.v); return r; }
// a*b - c and c - a*b
__device__ __forceinline__ F2 fms(F2 a, F2 b, F2 c) { return fma(a, b, -c); }
__device__ __forceinline__ F2 fnma(F2 a, F2 b, F2 c) { return fma(-a, b, c); }

__device__ __forceinline__ F2 abs2(F2 a) { return F2(fabsf(a.v.x), fabsf(a.v.y)); }
__device__ __forceinline__ F2 min2(F2 a, F2 b) { return F2(fminf(a.v.x, b.v.x), fminf(a.v.y, b.v.y)); }
__device__ __forceinline__ F2 max2(F2 a, F2 b) { return F2(fmaxf(a.v.x, b.v.x), fmaxf(a.v.y, b.v.y)); }
__device__ __forceinline__ float min3f(float a, float b, float c) {
  float r;
  asm("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));  // FMNMX3
  return r;
}
__device__ __forceinline__ float max3f(float a, float b, float c) {
  float r;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
  return r;
}
__device__ __forceinline__ F2 min3(F2 a, F2 b, F2 c) { return F2(min3f(a.v.x, b.v.x, c.v.x), min3f(a.v.y, b.v.y, c.v.y)); }
__device__ __forceinline__ F2 max3(F2 a, F2 b, F2 c) { return F2(max3f(a.v.x, b.v.x, c.v.x), max3f(a.v.y, b.v.y, c.v.y)); }

// SFU approximations (<= 2 ulp), as in the scalar fp32 kernel (DESIGN.md §3 "arithmetic freedom")
__device__ __forceinline__ float rcpf(float a) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
  return r;
}
__device__ __forceinline__ float sqrtf_(float a) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
  return r;
}
__device__ __forceinline__ float rsqrtf_(float a) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
  return r;
}
__device__ __forceinline__ F2 rcp2(F2 a) { return F2(rcpf(a.v.x), rcpf(a.v.y)); }
__device__ __forceinline__ F2 sqrt2(F2 a) { return F2(sqrtf_(a.v.x), sqrtf_(a.v.y)); }
__device__ __forceinline__ F2 rsqrt2(F2 a) { return F2(rsqrtf_(a.v.x), rsqrtf_(a.v.y)); }

__device__ __forceinline__ B2 gt(F2 a, F2 b) { return B2(a.v.x > b.v.x, a.v.y > b.v.y); }
__device__ __forceinline__ B2 ge(F2 a, F2 b) { return B2(a.v.x >= b.v.x, a.v.y >= b.v.y); }
__device__ __forceinline__ B2 lt(F2 a, F2 b) { return B2(a.v.x < b.v.x, a.v.y < b.v.y); }
__device__ __forceinline__ B2 operator&(B2 a, B2 b) { return B2(a.x && b.x, a.y && b.y); }
__device__ __forceinline__ B2 operator|(B2 a, B2 b) { return B2(a.x || b.x, a.y || b.y); }
__device__ __forceinline__ B2 operator!(B2 a) { return B2(!a.x, !a.y); }
__device__ __forceinline__ bool any(B2 a) { return a.x || a.y; }
__device__ __forceinline__ F2 sel(B2 m, F2 a, F2 b) { return F2(m.x ? a.v.x : b.v.x, m.y ? a.v.y : b.v.y); }

}  // namespace x2
}  // namespace amr

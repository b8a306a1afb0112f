// Tile shapes of the fused step kernels per (physics, dtype): TX x TY interior cells per CTA column,
// NT threads (whole warps), MAXR = register cap per thread (__maxnreg__), which with NT and the
// shared-memory footprint fixes the CTAs per SM.  Chosen from ptxas -v (registers / spills), the
// shared-memory budget and measured step times.
//   fp32: two cells per thread (godunov_step_x2.cuh): TX/2*TY interior pair threads (whole warps) plus the
//         aux warps (ring pairs + loader), NT >= TX/2*TY + 2*TY + TX; W = tile for n % 32 == 0, S = tile for
//         the other multiples of 16; test-size patches (n = 8) run the scalar 8x8 tile
//   fp64: one cell per thread with the x2 kernel's structure (godunov_step_d1.cuh): HX*TY compute threads (whole
//         warps) plus the aux warps, NT >= HX*TY + 2*TY + 2*HX; n = 8 (and other non-multiples of 16) run the first
//         fp64 kernel (godunov_step.cuh) on 8x8 tiles
#pragma once
namespace amr {
// hydro fp32: 3 CTAs per SM = 18 warps, 5 on one scheduler -> at most 102 registers per thread
struct TileCfg_hydro_f32 { static constexpr int WTX = 32, WTY = 8, STX = 16, STY = 16, NT = 192, MAXR = 96; };
struct TileCfg_mhd_f32 { static constexpr int WTX = 32, WTY = 8, STX = 16, STY = 16, NT = 192, WNT = 192, MAXR = 168, WMAXR = 168; };
struct TileCfg_hydro_f64 { static constexpr int HX = 16, TY = 8, NT = 192, MAXR = 168; };
struct TileCfg_mhd_f64 { static constexpr int HX = 16, TY = 8, NT = 192, MAXR = 168; };
}  // namespace amr

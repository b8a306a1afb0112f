// Tile shapes of the fused step kernels per (physics, dtype): TX x TY interior cells per CTA column,
// NT threads (whole warps), MAXR = register cap per thread (__maxnreg__), which with NT and the
// shared-memory footprint fixes the CTAs per SM.  Chosen from ptxas -v (registers / spills), the
// shared-memory budget and measured step times.
//   fp32: two cells per thread (godunov_step_x2.cuh): TX/2*TY interior pair threads (whole warps) plus the
//         aux warps (ring pairs + loader), NT >= TX/2*TY + 2*TY + TX; W = tile for n % 32 == 0, S = tile for
//         the other multiples of 16; test-size patches (n = 8) run the scalar 8x8 tile
//   fp64: one cell per thread (godunov_step.cuh), NT >= TX*TY + 2*TX + 2*TY
// The AMR_TUNE_* macros exist for tuning sweeps only (one -D per value); the defaults are the product.
#pragma once
#ifndef AMR_TUNE_F32_WTX
#define AMR_TUNE_F32_WTX 32
#define AMR_TUNE_F32_WTY 8
#define AMR_TUNE_F32_NT 192
#define AMR_TUNE_F32_MAXR 168
#endif
#ifndef AMR_TUNE_F64_TX
#define AMR_TUNE_F64_TX 16
#define AMR_TUNE_F64_TY 8
#define AMR_TUNE_F64_NT 192
#define AMR_TUNE_F64_MAXR 168
#endif
namespace amr {
#ifndef AMR_TUNE_HYDRO_F32_MAXR
#define AMR_TUNE_HYDRO_F32_MAXR 96   /* 3 CTAs per SM: 18 warps, 5 on one scheduler -> at most 102 registers */
#endif
struct TileCfg_hydro_f32 { static constexpr int WTX = 32, WTY = 8, STX = 16, STY = 16, NT = 192, MAXR = AMR_TUNE_HYDRO_F32_MAXR; };
struct TileCfg_mhd_f32 {
  static constexpr int WTX = AMR_TUNE_F32_WTX, WTY = AMR_TUNE_F32_WTY, STX = 16, STY = 16, NT = 192, WNT = AMR_TUNE_F32_NT,
                       MAXR = 168, WMAXR = AMR_TUNE_F32_MAXR;
};
struct TileCfg_hydro_f64 { static constexpr int TX = 16, TY = 16, NT = 320, MAXR = 168; };
struct TileCfg_mhd_f64 { static constexpr int TX = AMR_TUNE_F64_TX, TY = AMR_TUNE_F64_TY, NT = AMR_TUNE_F64_NT, MAXR = AMR_TUNE_F64_MAXR; };
}  // namespace amr

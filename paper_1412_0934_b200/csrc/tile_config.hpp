// Tile shapes of the fused step kernel per (physics, dtype): TX x TY interior cells per CTA column,
// NT threads (>= TX*TY + 2*TX + 2*TY, whole warps), MAXR = register cap per thread (__maxnreg__), which
// with NT and the shared-memory footprint fixes the CTAs per SM.
// Chosen from ptxas -v (registers / spills) and the shared-memory budget.
#pragma once
namespace amr {
struct TileCfg_hydro_f32 { static constexpr int TX = 16, TY = 16, NT = 320, MAXR = 96; };
struct TileCfg_hydro_f64 { static constexpr int TX = 16, TY = 16, NT = 320, MAXR = 168; };
struct TileCfg_mhd_f32 { static constexpr int TX = 16, TY = 8, NT = 192, MAXR = 128; };
struct TileCfg_mhd_f64 { static constexpr int TX = 16, TY = 8, NT = 192, MAXR = 255; };
}  // namespace amr

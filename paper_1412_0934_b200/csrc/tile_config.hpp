// Tile shapes of the fused step kernel per (physics, dtype): TX x TY interior cells per CTA column,
// NT threads (>= TX*TY + 2*TX + 2*TY, whole warps), MINB = CTAs per SM asked of the register allocator.
// Chosen from ptxas -v (registers / spills) and the shared-memory budget.
#pragma once
namespace amr {
struct TileCfg_hydro_f32 { static constexpr int TX = 16, TY = 16, NT = 320, MINB = 2; };
struct TileCfg_hydro_f64 { static constexpr int TX = 16, TY = 16, NT = 320, MINB = 1; };
struct TileCfg_mhd_f32 { static constexpr int TX = 16, TY = 16, NT = 320, MINB = 2; };
struct TileCfg_mhd_f64 { static constexpr int TX = 16, TY = 8, NT = 192, MINB = 1; };
}  // namespace amr

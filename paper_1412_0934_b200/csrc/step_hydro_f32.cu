// Instantiations of the fused Godunov step kernel: hydro, float (see godunov_step.cuh).
#include "godunov_step.cuh"
#include "tile_config.hpp"

namespace amr {

void tile_shape_hydro_f32(int n, int* tx, int* ty) {
  if (n % TileCfg_hydro_f32::TX == 0 && n % TileCfg_hydro_f32::TY == 0) { *tx = TileCfg_hydro_f32::TX; *ty = TileCfg_hydro_f32::TY; }
  else { *tx = 8; *ty = 8; }
}

cudaError_t launch_step_hydro_f32(const StepParams<float>& P, int limiter, int riemann, cudaStream_t s) {
  using C = TileCfg_hydro_f32;
  if (P.n % C::TX == 0 && P.n % C::TY == 0)
    return launch_dispatch<float, 5, C::TX, C::TY, C::NT, C::MAXR>(P, limiter, riemann, s);
  return launch_dispatch<float, 5, 8, 8, 96, 255>(P, limiter, riemann, s);
}

}  // namespace amr

// Instantiations of the fused Godunov step kernel: hydro, double (see godunov_step.cuh).
#include "godunov_step.cuh"
#include "tile_config.hpp"

namespace amr {

void tile_shape_hydro_f64(int n, int* tx, int* ty) {
  if (n % TileCfg_hydro_f64::TX == 0 && n % TileCfg_hydro_f64::TY == 0) { *tx = TileCfg_hydro_f64::TX; *ty = TileCfg_hydro_f64::TY; }
  else { *tx = 8; *ty = 8; }
}

cudaError_t launch_step_hydro_f64(const StepParams<double>& P, int limiter, int riemann, cudaStream_t s) {
  using C = TileCfg_hydro_f64;
  if (P.n % C::TX == 0 && P.n % C::TY == 0)
    return launch_dispatch<double, 5, C::TX, C::TY, C::NT, C::MAXR>(P, limiter, riemann, s);
  return launch_dispatch<double, 5, 8, 8, 96, 255>(P, limiter, riemann, s);
}

}  // namespace amr

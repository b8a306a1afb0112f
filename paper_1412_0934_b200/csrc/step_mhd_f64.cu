// Instantiations of the fused Godunov step kernels: mhd, double.  Patches whose size is a multiple of 16 run
// the x2-structured fp64 kernel (godunov_step_d1.cuh: staged face states, branch-free solvers, aux loader
// warps); other sizes (multiples of 8) the first fp64 kernel (godunov_step.cuh) on 8x8 tiles.
#include "godunov_step.cuh"
#include "godunov_step_d1.cuh"
#include "tile_config.hpp"

namespace amr {

void tile_shape_mhd_f64(int n, int* tx, int* ty) {
  using C = TileCfg_mhd_f64;
  if (n % C::HX == 0 && n % C::TY == 0) { *tx = C::HX; *ty = C::TY; }
  else { *tx = 8; *ty = 8; }
}

cudaError_t launch_step_mhd_f64(const StepParams<double>& P, int limiter, int riemann, cudaStream_t s) {
  using C = TileCfg_mhd_f64;
  if (P.n % C::HX == 0 && P.n % C::TY == 0)
    return d1::launch_dispatch_d1<9, C::HX, C::TY, C::NT, C::MAXR>(P, limiter, riemann, s);
  return launch_dispatch<double, 9, 8, 8, 96, 255>(P, limiter, riemann, s);
}

}  // namespace amr

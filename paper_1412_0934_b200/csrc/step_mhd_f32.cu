// Instantiations of the fused Godunov step kernels: mhd, float.  Patches whose size is a multiple of 16
// run the two-cells-per-thread kernel (godunov_step_x2.cuh); test-size patches (n = 8) the scalar one.
#include "godunov_step.cuh"
#include "godunov_step_x2.cuh"
#include "tile_config.hpp"

namespace amr {

void tile_shape_mhd_f32(int n, int* tx, int* ty) {
  using C = TileCfg_mhd_f32;
  if (n % C::WTX == 0 && n % C::WTY == 0) { *tx = C::WTX; *ty = C::WTY; }
  else if (n % C::STX == 0 && n % C::STY == 0) { *tx = C::STX; *ty = C::STY; }
  else { *tx = 8; *ty = 8; }
}

cudaError_t launch_step_mhd_f32(const StepParams<float>& P, int limiter, int riemann, cudaStream_t s) {
  using C = TileCfg_mhd_f32;
  if (P.n % C::WTX == 0 && P.n % C::WTY == 0)
    return x2::launch_dispatch_x2<9, C::WTX, C::WTY, C::WNT, C::WMAXR>(P, limiter, riemann, s);
  if (P.n % C::STX == 0 && P.n % C::STY == 0)
    return x2::launch_dispatch_x2<9, C::STX, C::STY, C::NT, C::MAXR>(P, limiter, riemann, s);
  return launch_dispatch<float, 9, 8, 8, 96, 255>(P, limiter, riemann, s);
}

}  // namespace amr

// Instantiations of the PPM hydro sweep (ppm_sweep.cuh): float and double, HLL / HLLC, x / y / z.
#include "ppm_sweep.cuh"

namespace amr {

cudaError_t launch_ppm_sweep_f32(const ppm::SweepParams<float>& P, int riemann, int dir, cudaStream_t s) {
  return ppm::launch_sweep<float>(P, riemann, dir, s);
}
cudaError_t launch_ppm_sweep_f64(const ppm::SweepParams<double>& P, int riemann, int dir, cudaStream_t s) {
  return ppm::launch_sweep<double>(P, riemann, dir, s);
}

}  // namespace amr

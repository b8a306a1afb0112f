// Instantiations of the PPM hydro sweep: float (packed pairs, ppm_sweep_x2.cuh; scalar for n % 16 != 0) and double
// (ppm_sweep.cuh), HLL / HLLC, x / y / z.
#include "ppm_sweep.cuh"
#include "ppm_sweep_x2.cuh"

namespace amr {

cudaError_t launch_ppm_sweep_f32(const ppm::SweepParams<float>& P, int riemann, int dir, cudaStream_t s) {
  // patch sizes that are a multiple of 16: two pencils per thread with packed f32x2 arithmetic
  if (P.n % 16 == 0) return ppm::launch_sweep_x2(P, riemann, dir, s);
  return ppm::launch_sweep<float>(P, riemann, dir, s);
}
cudaError_t launch_ppm_sweep_f64(const ppm::SweepParams<double>& P, int riemann, int dir, cudaStream_t s) {
  return ppm::launch_sweep<double>(P, riemann, dir, s);
}

}  // namespace amr

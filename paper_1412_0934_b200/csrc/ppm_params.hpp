// Parameter block and launchers of the PPM hydro sweep (ppm_sweep.cuh), for the host code of batch.cu.
#pragma once
#include <cuda_runtime.h>

namespace amr {
namespace ppm {
template <class T>
struct SweepParams {
  const T* Uin;    // device, [5][np][n^3]
  T* Uout;         // device, [5][np][n^3]
  const T* halo;   // device, [5][np][(n+2g)^3] or nullptr
  const int* nbr;  // device, [np][27]
  unsigned long long* counters;
  int np, np_active, n, g;   // np: patches in the arena (strides); the grid covers the first np_active
  T dtdx, gamma, gm1, igm1;
};
}  // namespace ppm
cudaError_t launch_ppm_sweep_f32(const ppm::SweepParams<float>& P, int riemann, int dir, cudaStream_t s);
cudaError_t launch_ppm_sweep_f64(const ppm::SweepParams<double>& P, int riemann, int dir, cudaStream_t s);
}  // namespace amr

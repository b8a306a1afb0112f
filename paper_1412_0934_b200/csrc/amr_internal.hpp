// Internal declarations shared by the host code (batch.cu) and the kernel translation units.
// Nothing here crosses the C-ABI (include/amr_godunov.h).  No code is shared with oracle/.
#pragma once
#include <atomic>
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace amr {

constexpr int NBR_PATCH_MASK = 0x0FFFFFFF;  // nbr entry >= 0: low 28 bits = source patch,
constexpr int NBR_MODE_SHIFT = 28;          // bits 28..30 = clamp flags (x,y,z) for outflow
constexpr int NBR_FROM_HALO = -2;           // nbr entry: region comes from the prolongation halo buffer

// sets the thread-local message amr_last_error() returns ("where: what") and returns code (batch.cu)
int set_error(int code, const char* where, const char* what);

// Everything the step kernel needs, passed by value.
template <class T>
struct StepParams {
  const T* Uin;        // device, [NF][np][n^3]
  T* Uout;             // device, [NF][np][n^3]
  const T* halo;       // device, [NF][np][(n+2g)^3] or nullptr (level 0)
  const int* nbr;      // device, [np][27]
  T* fblk;             // device flux blocks [nblk][3][NF][3 face planes 0, n/2, n][n^2] or nullptr
  const int* fblk_of;  // device, [np] block index or -1 (nullptr if fblk is)
  unsigned long long* counters;  // device [4]
  void* smax;          // device, one T-sized slot (bit pattern ordered as unsigned), pre-zeroed
  int np, n, g;        // np = patches in the arena (strides); the grid covers the first np_active of them
  int np_active;
  int ntx, nty, ntz, zc;  // tiles per patch along x,y,z; planes per z-chunk
  T dtdx;              // dt/dx
  T hdtdx;             // dt/(2 dx)
  T gamma, gm1, igm1;
  T ch, ch2, half_ich; // GLM speed, its square, 1/(2 ch)
  T damp;              // exp(-alpha ch dt/dx)
  T eps;               // HLLD degeneracy threshold (A7)
};

// launchers implemented in step_*.cu (one translation unit per (dtype, physics))
cudaError_t launch_step_hydro_f32(const StepParams<float>& P, int limiter, int riemann, cudaStream_t s);
cudaError_t launch_step_hydro_f64(const StepParams<double>& P, int limiter, int riemann, cudaStream_t s);
cudaError_t launch_step_mhd_f32(const StepParams<float>& P, int limiter, int riemann, cudaStream_t s);
cudaError_t launch_step_mhd_f64(const StepParams<double>& P, int limiter, int riemann, cudaStream_t s);
// fills ntx/nty/ntz/zc for the tile shape the launcher of this variant uses
void tile_shape_hydro_f32(int n, int* tx, int* ty);
void tile_shape_hydro_f64(int n, int* tx, int* ty);
void tile_shape_mhd_f32(int n, int* tx, int* ty);
void tile_shape_mhd_f64(int n, int* tx, int* ty);

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute of a kernel: remembered per kernel
// instantiation as a bit mask over devices (atomic; setting it twice is harmless, so no lock is needed)
inline cudaError_t ensure_dynamic_smem(const void* kern, int bytes, std::atomic<unsigned long long>& done) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const unsigned long long bit = 1ull << (dev & 63);
  if (done.load(std::memory_order_acquire) & bit) return cudaSuccess;
  e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e == cudaSuccess) done.fetch_or(bit, std::memory_order_release);
  return e;
}

// aux kernels (aux_kernels.cu); dtype: 0 = f32, 1 = f64
cudaError_t launch_smax(int dtype, const void* U, int nf, int np, int np_active, int n, double gamma, void* smax_slot,
                        cudaStream_t s);
constexpr int TOTALS_BLOCKS = 256;
cudaError_t launch_totals(int dtype, const void* U, int nf, int np, int np_active, int n, double* partials /*[nf][TOTALS_BLOCKS]*/,
                          cudaStream_t s);
// interiors [nf][np][n^3] (device) -> ghosted [nf][npc][(n+2g)^3] (device) for patches [p0, p0+npc)
cudaError_t launch_gather_ghosted(int dtype, const void* U, const void* halo, const int* nbr, int nf, int np,
                                  int n, int g, int p0, int npc, void* out, cudaStream_t s);
// ghosted or interior host-layout staging (device) -> interiors
cudaError_t launch_scatter_interior(int dtype, const void* staged, int with_ghosts, int nf, int np, int n, int g,
                                    int p0, int npc, void* U, cudaStream_t s);
cudaError_t launch_fill_nan(int dtype, void* ptr, size_t count, cudaStream_t s);
cudaError_t launch_fma_chain(int dtype, void* sink, int grid, int iters, cudaStream_t s);

// two-level kernels (aux_kernels.cu); table formats are documented at the kernels
// O8 without tables: parents resolved in the kernel through the coarse patch map (cmap, [cdims z][y][x], -1 = none),
// the fine patches' origins and neighbour table (all device); bc: the six AMR_BC_* of the level pair (host)
cudaError_t launch_prolong_halo(int dtype, void* halo, size_t fs_halo, int nf, int n, int g, int npf, const int* domf,
                                const int* domc, const int* cdims, const int* bc, const int* forigin, const int* nbr,
                                const int* cmap, const void* Ucold, const void* Ucnew, size_t fs_c, double theta,
                                cudaStream_t s);
// O9(6) without a table: the parent block of fine patch p is found through forigin (device, [npf][3]) and cmap
cudaError_t launch_restrict(int dtype, const void* Uf, size_t fs_f, int nf, int n, int npf, const int* domc, const int* cdims,
                            const int* bc, const int* forigin, const int* cmap, void* Uc, size_t fs_c, cudaStream_t s);
// O9(7) without a host table.  cblk (device): int4 (coarse patch, its origin x, y, z) per coarse flux block, block
// index = position (shared = 0) or = patch (shared = 1: the coarse level records per patch); fmap (device): fine patch
// map [fdims z][y][x], -1 = not refined.  launch_reflux_find (link time) fills `list` (device, int2 per uncovered
// coarse cell with a covered face neighbour: flat cell index, block position << 6 | mask of (direction, side)) and
// *count (device; may exceed capacity: the caller checks); launch_reflux / launch_zero_faces give every entry a thread.
cudaError_t launch_reflux_find(int nf, int n, int shared, const int* domc, const int* fdims, const int* bc, const void* cblk,
                               int ncblk, const int* fmap, void* list, int* count, int capacity, cudaStream_t s);
cudaError_t launch_reflux(int dtype, void* Uc, size_t fs_c, int nf, int n, int shared, const int* domc, const int* fdims,
                          const int* bc, const void* cblk, const void* list, int nlist, const int* fmap, const int* forigin,
                          void* Fc, const void* Ff, double dtdx, cudaStream_t s);
// zeroes the coarse flux slots a reflux of this link reads (all fields)
cudaError_t launch_zero_faces(int dtype, void* Fc, int nf, int n, int shared, const int* domc, const int* fdims, const int* bc,
                              const void* cblk, const void* list, int nlist, cudaStream_t s);

// regridding (aux_kernels.cu): block flags of one field [np*8]; whole-patch copies; whole-patch prolongation
cudaError_t launch_flag_blocks(int dtype, const void* Ufield, int np, int n, double threshold, unsigned char* flags,
                               cudaStream_t s);
cudaError_t launch_copy_patches(int dtype, void* Unew, size_t fs_new, const void* Uold, size_t fs_old, const void* pairs,
                                int npairs, int nf, int n, cudaStream_t s);
cudaError_t launch_copy_patches_in(int dtype, void* U, size_t fs, const void* packed, size_t fs_packed, const void* pairs,
                                   int npairs, int nf, int n, cudaStream_t s);
// born: int4 (new patch index, fine origin x, y, z) per new-born patch (device); cmap, domc, cdims, bc as launch_prolong_halo
cudaError_t launch_prolong_patches(int dtype, void* Unew, size_t fs_new, int nf, int n, const int* domc, const int* cdims,
                                   const int* bc, const void* born, const int* cmap, int nparents, const void* Uc,
                                   size_t fs_c, cudaStream_t s);

}  // namespace amr

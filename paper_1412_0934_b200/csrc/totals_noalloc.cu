// amr_conserved_totals_noalloc: the conserved-totals reduction (the check behind north_star's "exact conservation of
// mass, momentum and energy"; same partition and summation order as totals_kernel in aux_kernels.cu) for callers that
// cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The existing path (amr_conserved_totals) keeps its per-block partial sums in the batch's arena, copies them to the host
// and finishes the sum there.  This variant takes plain device pointers, keeps the partial sums and the "blocks done"
// counters in ONE file-scope device array of fixed size, finishes the sum in the last block of each field and writes the
// result to a caller-provided DEVICE array: no allocation, no host copy, no synchronisation - it only enqueues.
//
//  * The array lives in every GPU that loads the library until the process exits: NOALLOC_SCRATCH_BYTES = 33 024 bytes
//    (16 fields x 256 partial sums x 8 B + 16 counters, rounded up to 256 B).  More than 16 fields are rejected.
//  * In host code the array's name is a host-side stand-in, not a device address.  The device address is taken once per
//    device, with that device current, by cudaGetSymbolAddress (scratch_for_current_device below) and passed to the
//    kernel as an ordinary pointer.
//  * Every call on a device shares the array, and it keeps the last call's contents: the counters must start at zero, so
//    each call clears them on its stream before the launch (the partial sums are overwritten before they are read).
//    Two calls that overlap on the GPU (different streams, no ordering between them) race on it; calls on one stream, or
//    ordered by events, do not.
#include <atomic>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "amr_godunov.h"
#include "amr_internal.hpp"

namespace {

constexpr int NOALLOC_MAX_FIELDS = AMR_NOALLOC_MAX_FIELDS;
constexpr int NOALLOC_BLOCKS = amr::TOTALS_BLOCKS;   // blocks per field: the partition of the existing path
constexpr size_t NOALLOC_PARTIAL_BYTES = (size_t)NOALLOC_MAX_FIELDS * NOALLOC_BLOCKS * sizeof(double);
constexpr size_t NOALLOC_SCRATCH_BYTES = ((NOALLOC_PARTIAL_BYTES + NOALLOC_MAX_FIELDS * sizeof(unsigned)) + 255) / 256 * 256;
constexpr int MAX_DEVICES = 64;

static __device__ __align__(256) unsigned char g_totals_scratch[NOALLOC_SCRATCH_BYTES];

// [field][block] partial sums, then one counter per field
__device__ __forceinline__ double* partials_of(unsigned char* scratch) { return reinterpret_cast<double*>(scratch); }
__device__ __forceinline__ unsigned* done_of(unsigned char* scratch) {
  return reinterpret_cast<unsigned*>(scratch + NOALLOC_PARTIAL_BYTES);
}

// grid (NOALLOC_BLOCKS, nf), 256 threads.  Per block exactly totals_kernel's sum (grid-stride, fixed tree); the block
// that finishes a field last adds the field's NOALLOC_BLOCKS partial sums in a fixed order (thread t takes block t: 256
// threads, 256 blocks; the same tree) and writes totals[field].
template <class T>
__global__ void __launch_bounds__(256) totals_noalloc_kernel(const T* __restrict__ U, size_t ncell, size_t fstride,
                                                             unsigned char* __restrict__ scratch,
                                                             double* __restrict__ totals) {
  static_assert(NOALLOC_BLOCKS == 256, "the final sum gives one partial to each of the 256 threads");
  const int q = blockIdx.y;
  const T* u = U + (size_t)q * fstride;
  double s = 0.0;
  for (size_t c = (size_t)blockIdx.x * 256 + threadIdx.x; c < ncell; c += (size_t)gridDim.x * 256) s += (double)u[c];
  __shared__ double red[256];
  __shared__ bool last;
  red[threadIdx.x] = s;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  double* part = partials_of(scratch) + (size_t)q * NOALLOC_BLOCKS;
  if (threadIdx.x == 0) {
    part[blockIdx.x] = red[0];
    __threadfence();                                     // the partial sum is visible before the count is
    last = atomicAdd(done_of(scratch) + q, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  red[threadIdx.x] = __ldcg(part + threadIdx.x);         // written by other SMs: read through L2
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    totals[q] = red[0];
    done_of(scratch)[q] = 0;                             // left clean for the next call (which clears it again anyway)
  }
}

// Device address of the scratch array on the CURRENT device; taken once per device (set-up), cached afterwards.
std::atomic<unsigned char*> g_scratch_ptr[MAX_DEVICES];

int scratch_for_current_device(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return amr::set_error(AMR_ECUDA, "amr_conserved_totals_noalloc", cudaGetErrorString(e));
  if (dev < 0 || dev >= MAX_DEVICES) return amr::set_error(AMR_EINVAL, "amr_conserved_totals_noalloc", "device ordinal >= 64");
  unsigned char* p = g_scratch_ptr[dev].load(std::memory_order_acquire);
  if (!p) {
    e = cudaGetSymbolAddress((void**)&p, g_totals_scratch);   // the symbol's address on the device that is current now
    if (e != cudaSuccess || !p)
      return amr::set_error(AMR_ECUDA, "amr_conserved_totals_noalloc: cudaGetSymbolAddress", cudaGetErrorString(e));
    g_scratch_ptr[dev].store(p, std::memory_order_release);    // two threads racing here store the same value
  }
  *out = p;
  return AMR_OK;
}

// the pointer must be device (or managed) memory that the current device owns
int check_on_device(const void* ptr, int dev, const char* what) {
  cudaPointerAttributes a;
  cudaError_t e = cudaPointerGetAttributes(&a, ptr);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return amr::set_error(AMR_EINVAL, what, "not a CUDA pointer");
  }
  if (a.type != cudaMemoryTypeDevice && a.type != cudaMemoryTypeManaged)
    return amr::set_error(AMR_EINVAL, what, "must be device memory (this entry point copies nothing to the host)");
  if (a.type == cudaMemoryTypeDevice && a.device != dev)
    return amr::set_error(AMR_EINVAL, what, "lives on another device than the current one");
  return AMR_OK;
}

}  // namespace

extern "C" int amr_conserved_totals_noalloc(const void* dev_U, int dtype, int nfields, int64_t ncells, int64_t field_stride,
                                            double* dev_totals, void* cuda_stream) {
  const char* where = "amr_conserved_totals_noalloc";
  if (!dev_U || !dev_totals) return amr::set_error(AMR_EINVAL, where, "null pointer");
  if (dtype != AMR_F32 && dtype != AMR_F64) return amr::set_error(AMR_EINVAL, where, "dtype must be AMR_F32 or AMR_F64");
  if (nfields < 1) return amr::set_error(AMR_EINVAL, where, "nfields must be >= 1");
  if (nfields > NOALLOC_MAX_FIELDS) {
    char msg[160];
    snprintf(msg, sizeof msg, "nfields = %d exceeds AMR_NOALLOC_MAX_FIELDS = %d (the static scratch array holds %d x %d partial sums)",
             nfields, NOALLOC_MAX_FIELDS, NOALLOC_MAX_FIELDS, NOALLOC_BLOCKS);
    return amr::set_error(AMR_EINVAL, where, msg);
  }
  if (ncells < 1 || field_stride < ncells) return amr::set_error(AMR_EINVAL, where, "need 1 <= ncells <= field_stride");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return amr::set_error(AMR_ECUDA, where, "no current CUDA device");
  int rc = check_on_device(dev_U, dev, "amr_conserved_totals_noalloc: dev_U");
  if (rc != AMR_OK) return rc;
  rc = check_on_device(dev_totals, dev, "amr_conserved_totals_noalloc: dev_totals");
  if (rc != AMR_OK) return rc;
  unsigned char* scratch = nullptr;
  rc = scratch_for_current_device(&scratch);
  if (rc != AMR_OK) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  // the counters must start at zero whatever the previous call (perhaps an aborted one) left behind
  cudaError_t e = cudaMemsetAsync(scratch + NOALLOC_PARTIAL_BYTES, 0, NOALLOC_MAX_FIELDS * sizeof(unsigned), s);
  if (e != cudaSuccess) return amr::set_error(AMR_ECUDA, where, cudaGetErrorString(e));
  const dim3 grid(NOALLOC_BLOCKS, (unsigned)nfields);
  if (dtype == AMR_F32)
    totals_noalloc_kernel<float><<<grid, 256, 0, s>>>((const float*)dev_U, (size_t)ncells, (size_t)field_stride, scratch, dev_totals);
  else
    totals_noalloc_kernel<double><<<grid, 256, 0, s>>>((const double*)dev_U, (size_t)ncells, (size_t)field_stride, scratch, dev_totals);
  e = cudaGetLastError();
  if (e != cudaSuccess) return amr::set_error(AMR_ECUDA, where, cudaGetErrorString(e));
  return AMR_OK;
}

// Patch builder: the procedure the paper designed for the GPU (Figure 1):
//   1. order the leaf cells of a level along a space-filling curve        -> Morton keys + LSD radix sort
//   2. group them in compact (hole-free) cubic patches of maximum size    -> per-cell level + head compaction
//   3. gather the patches' data into large contiguous chunks              -> gather into the batch arena layout
// Readings: Morton curve, x least significant; a patch is an octree-aligned cube of side 2^k,
// k <= kmax, all of whose 8^k cells are leaf cells; each cell belongs to the largest such cube.
// An aligned cube is a run of 8^k consecutive keys, so with sorted unique keys "compact" is two look-ups:
// keys[j] == base and keys[j + 8^k - 1] == base + 8^k - 1.  All kernels here are HBM-bound streams.
// Shares no code with oracle/patch_builder.py.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <new>

#include "../../include/amr_godunov.h"
#include "amr_internal.hpp"

namespace {

constexpr int SORT_THREADS = 256;                 // 8 warps
constexpr int SORT_GROUPS = 16;                   // 32-item groups per warp
constexpr int SORT_ITEMS = SORT_THREADS * SORT_GROUPS;   // items per block (4096)
constexpr int CMP_ITEMS = 1024;                   // items per block of the compaction kernels
constexpr size_t ALIGN = 256;
inline size_t up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

// spread the low 10 bits of v: bit b -> bit 3b
__device__ __forceinline__ unsigned spread3(unsigned v) {
  v &= 0x3ffu;
  v = (v | (v << 16)) & 0x030000ffu;
  v = (v | (v << 8)) & 0x0300f00fu;
  v = (v | (v << 4)) & 0x030c30c3u;
  v = (v | (v << 2)) & 0x09249249u;
  return v;
}
__device__ __forceinline__ unsigned compact3(unsigned v) {  // inverse of spread3
  v &= 0x09249249u;
  v = (v | (v >> 2)) & 0x030c30c3u;
  v = (v | (v >> 4)) & 0x0300f00fu;
  v = (v | (v >> 8)) & 0x030000ffu;
  v = (v | (v >> 16)) & 0x3ffu;
  return v;
}

// step 1a: key = x | y << 1 | z << 2 bit-interleaved; value = input index
__global__ void key_kernel(const int* __restrict__ xyz, unsigned n, unsigned* __restrict__ keys, unsigned* __restrict__ vals) {
  const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  keys[i] = spread3((unsigned)xyz[i]) | (spread3((unsigned)xyz[n + i]) << 1) | (spread3((unsigned)xyz[2 * (size_t)n + i]) << 2);
  vals[i] = i;
}

// lanes of the warp whose 8-bit digit equals this lane's (invalid lanes match each other): nine ballots; on
// sm_100a this is several times faster than __match_any_sync, which goes through the MIO queue (profiles/r1d)
__device__ __forceinline__ unsigned same_digit_mask(unsigned d, bool ok) {
  const unsigned okm = __ballot_sync(0xffffffffu, ok);
  unsigned m = ok ? okm : ~okm;
#pragma unroll
  for (int b = 0; b < 8; ++b) {
    const unsigned bal = __ballot_sync(0xffffffffu, (d >> b) & 1u);
    m &= ((d >> b) & 1u) ? bal : ~bal;
  }
  return m;
}

// step 1b, one 8-bit LSD pass.  A block owns SORT_ITEMS consecutive items; warp w owns the w-th run of
// 32 * SORT_GROUPS of them and walks it group by group, so (warp, group, lane) order is input order and the
// pass is stable.  Per group: lanes with equal digits find each other (same_digit_mask); the rank of a lane
// among them is the popcount of the lower lanes of its mask.
__device__ __forceinline__ void warp_digit_counts(const unsigned* __restrict__ keys, unsigned n, unsigned base, int shift,
                                                   unsigned* wh /* [256] of this warp, zeroed */) {
  const int lane = threadIdx.x & 31;
  for (int g = 0; g < SORT_GROUPS; ++g) {
    const unsigned i = base + g * 32 + lane;
    const bool ok = i < n;
    const unsigned d = ok ? (keys[i] >> shift) & 255u : 0u;
    const unsigned m = same_digit_mask(d, ok);
    if (ok && lane == __ffs(m) - 1) wh[d] += __popc(m);
    __syncwarp();
  }
}

__global__ void __launch_bounds__(SORT_THREADS) hist_kernel(const unsigned* __restrict__ keys, unsigned n, int shift,
                                                            unsigned nb, unsigned* __restrict__ hist /* [256][nb] */) {
  __shared__ unsigned wh[SORT_THREADS / 32][256];
  const int w = threadIdx.x >> 5;
  for (int d = threadIdx.x; d < (SORT_THREADS / 32) * 256; d += SORT_THREADS) (&wh[0][0])[d] = 0;
  __syncthreads();
  warp_digit_counts(keys, n, blockIdx.x * SORT_ITEMS + w * 32 * SORT_GROUPS, shift, wh[w]);
  __syncthreads();
  unsigned s = 0;
#pragma unroll
  for (int v = 0; v < SORT_THREADS / 32; ++v) s += wh[v][threadIdx.x];
  hist[(size_t)threadIdx.x * nb + blockIdx.x] = s;
}

// exclusive scan of m values in place, one block: thread-contiguous chunks + a block scan of the chunk sums
__global__ void __launch_bounds__(1024) scan_kernel(unsigned* __restrict__ a, unsigned m) {
  __shared__ unsigned part[1024];
  const unsigned chunk = (m + 1023) / 1024;
  const unsigned lo = threadIdx.x * chunk, hi = min(m, lo + chunk);
  unsigned s = 0;
  for (unsigned i = lo; i < hi; ++i) s += a[i];
  part[threadIdx.x] = s;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {  // Hillis-Steele inclusive scan
    const unsigned v = threadIdx.x >= o ? part[threadIdx.x - o] : 0;
    __syncthreads();
    part[threadIdx.x] += v;
    __syncthreads();
  }
  unsigned run = part[threadIdx.x] - s;
  for (unsigned i = lo; i < hi; ++i) { const unsigned v = a[i]; a[i] = run; run += v; }
}

// the sort's histogram scan in two levels: block d scans row d of hist [256][nb] in place (exclusive) and
// leaves the row total; the scatter kernel adds the exclusive scan of the 256 totals itself
__global__ void __launch_bounds__(256) scan_rows_kernel(unsigned* __restrict__ hist, unsigned nb, unsigned* __restrict__ totals) {
  __shared__ unsigned part[256];
  unsigned* row = hist + (size_t)blockIdx.x * nb;
  const unsigned chunk = (nb + 255) / 256;
  const unsigned lo = min(nb, threadIdx.x * chunk), hi = min(nb, lo + chunk);
  unsigned s = 0;
  for (unsigned i = lo; i < hi; ++i) s += row[i];
  part[threadIdx.x] = s;
  __syncthreads();
  for (int o = 1; o < 256; o <<= 1) {
    const unsigned v = threadIdx.x >= o ? part[threadIdx.x - o] : 0;
    __syncthreads();
    part[threadIdx.x] += v;
    __syncthreads();
  }
  unsigned run = part[threadIdx.x] - s;
  for (unsigned i = lo; i < hi; ++i) { const unsigned v = row[i]; row[i] = run; run += v; }
  if (threadIdx.x == 255) totals[blockIdx.x] = part[255];
}

__global__ void __launch_bounds__(SORT_THREADS) scatter_kernel(const unsigned* __restrict__ keys, const unsigned* __restrict__ vals,
                                                               unsigned n, int shift, unsigned nb,
                                                               const unsigned* __restrict__ offs /* row-scanned [256][nb] */,
                                                               const unsigned* __restrict__ totals /* [256] row totals */,
                                                               unsigned* __restrict__ keys_out, unsigned* __restrict__ vals_out) {
  __shared__ unsigned wh[SORT_THREADS / 32][256];
  __shared__ unsigned dbase[256];
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int d = threadIdx.x; d < (SORT_THREADS / 32) * 256; d += SORT_THREADS) (&wh[0][0])[d] = 0;
  __syncthreads();
  const unsigned base = blockIdx.x * SORT_ITEMS + w * 32 * SORT_GROUPS;
  warp_digit_counts(keys, n, base, shift, wh[w]);
  __syncthreads();
  {  // exclusive scan of the digit totals (thread d = digit d)
    const unsigned tot = totals[threadIdx.x];
    dbase[threadIdx.x] = tot;
    __syncthreads();
    for (int o = 1; o < 256; o <<= 1) {
      const unsigned v = threadIdx.x >= o ? dbase[threadIdx.x - o] : 0;
      __syncthreads();
      dbase[threadIdx.x] += v;
      __syncthreads();
    }
    // counts -> first output position of (warp, digit): digit base + blocks before this one + earlier warps
    unsigned run = (dbase[threadIdx.x] - tot) + offs[(size_t)threadIdx.x * nb + blockIdx.x];
#pragma unroll
    for (int v = 0; v < SORT_THREADS / 32; ++v) { const unsigned c = wh[v][threadIdx.x]; wh[v][threadIdx.x] = run; run += c; }
  }
  __syncthreads();
  for (int g = 0; g < SORT_GROUPS; ++g) {
    const unsigned i = base + g * 32 + lane;
    const bool ok = i < n;
    const unsigned k = ok ? keys[i] : 0u;
    const unsigned d = (k >> shift) & 255u;
    const unsigned m = same_digit_mask(d, ok);
    unsigned pos = 0;
    if (ok) pos = wh[w][d] + __popc(m & ((1u << lane) - 1));
    __syncwarp();
    if (ok && lane == __ffs(m) - 1) wh[w][d] += __popc(m);
    __syncwarp();
    if (ok) { keys_out[pos] = k; vals_out[pos] = vals[i]; }
  }
}

// step 2a: level of the largest compact aligned cube around each cell; head = first cell of that cube
__global__ void level_kernel(const unsigned* __restrict__ keys, unsigned n, int kmax, unsigned char* __restrict__ lev,
                             unsigned* __restrict__ dup) {
  const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const unsigned key = keys[i];
  if (i > 0 && keys[i - 1] == key) atomicAdd(dup, 1u);   // input contract: cells are unique
  int found = 0;
  for (int k = kmax; k >= 1; --k) {
    const unsigned size = 1u << (3 * k);
    const unsigned b = key & ~(size - 1u);
    const unsigned off = key - b;
    if (off > i) continue;
    const unsigned j = i - off;
    if (j + (size - 1u) >= n) continue;
    if (keys[j] == b && keys[j + size - 1u] == b + size - 1u) { found = k; break; }
  }
  const unsigned hmask = (1u << (3 * found)) - 1u;
  lev[i] = (unsigned char)(found | ((key & hmask) == 0u ? 0x80 : 0));   // bit 7: head of its patch
}

// step 2b / 3a: ordered compaction in three kernels (count per block, scan of the counts, write).
// MODE 0: over cells, flag = head bit of lev[i]; writes first[p] = i, plev[p] = level.
// MODE 1: over patches, flag = (plev[p] == k); writes slot_first[s] = first[p].
template <int MODE>
__device__ __forceinline__ bool cmp_flag(const unsigned char* lev, unsigned i, int k) {
  return MODE == 0 ? (lev[i] & 0x80) != 0 : lev[i] == k;
}
template <int MODE>
__global__ void __launch_bounds__(256) count_kernel(const unsigned char* __restrict__ lev, unsigned n, int k,
                                                    unsigned* __restrict__ counts) {
  __shared__ unsigned s_c;
  if (threadIdx.x == 0) s_c = 0;
  __syncthreads();
  unsigned c = 0;
  for (unsigned i = blockIdx.x * CMP_ITEMS + threadIdx.x; i < min(n, (blockIdx.x + 1u) * CMP_ITEMS); i += 256) c += cmp_flag<MODE>(lev, i, k);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
  if ((threadIdx.x & 31) == 0) atomicAdd(&s_c, c);
  __syncthreads();
  if (threadIdx.x == 0) counts[blockIdx.x] = s_c;
}
template <int MODE>
__global__ void __launch_bounds__(256) write_kernel(const unsigned char* __restrict__ lev, const unsigned* __restrict__ src_first,
                                                    unsigned n, int k, const unsigned* __restrict__ offs,
                                                    const unsigned* __restrict__ base /* device scalar or null */,
                                                    unsigned* __restrict__ out_first, unsigned char* __restrict__ out_lev) {
  __shared__ unsigned s_w[8];
  __shared__ unsigned s_run;
  if (threadIdx.x == 0) s_run = offs[blockIdx.x] + (base ? *base : 0u);
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (unsigned i0 = blockIdx.x * CMP_ITEMS; i0 < min(n, (blockIdx.x + 1u) * CMP_ITEMS); i0 += 256) {
    const unsigned i = i0 + threadIdx.x;
    const bool f = i < n && cmp_flag<MODE>(lev, i, k);
    const unsigned m = __ballot_sync(0xffffffffu, f);
    if (lane == 0) s_w[w] = __popc(m);
    __syncthreads();
    unsigned before = s_run;
    for (int v = 0; v < w; ++v) before += s_w[v];
    if (f) {
      const unsigned p = before + __popc(m & ((1u << lane) - 1));
      if (MODE == 0) { out_first[p] = i; out_lev[p] = lev[i] & 0x7f; }
      else out_first[p] = src_first[i];
    }
    __syncthreads();
    if (threadIdx.x == 0) { unsigned t = 0; for (int v = 0; v < 8; ++v) t += s_w[v]; s_run += t; }
    __syncthreads();
  }
}

// step 3b: out[f][s][lz][ly][lx] = in[f][ perm[first_s + morton(lx, ly, lz)] ]; one thread per output cell
template <class T>
__global__ void gather_kernel(const T* __restrict__ in, size_t ncell, int nf, const unsigned* __restrict__ perm,
                              const unsigned* __restrict__ slot_first, unsigned nslot, int k, T* __restrict__ out) {
  const unsigned n3 = 1u << (3 * k);
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (size_t)nslot * n3) return;
  const unsigned s = (unsigned)(t >> (3 * k)), c = (unsigned)(t & (n3 - 1u));
  const unsigned msk = (1u << k) - 1u;
  const unsigned lx = c & msk, ly = (c >> k) & msk, lz = c >> (2 * k);
  const unsigned moff = spread3(lx) | (spread3(ly) << 1) | (spread3(lz) << 2);
  const unsigned src = perm[slot_first[s] + moff];
  for (int f = 0; f < nf; ++f) out[((size_t)f * nslot + s) * n3 + c] = in[(size_t)f * ncell + src];
}

// lbase[k] = number of patches of the levels below k (the per-level totals sit behind each level's counts)
__global__ void bases_kernel(const unsigned* __restrict__ counts, unsigned stride, unsigned ncb, int nlev, unsigned* __restrict__ lbase) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    unsigned run = 0;
    for (int k = 0; k < nlev; ++k) { lbase[k] = run; run += counts[(size_t)k * stride + ncb]; }
    lbase[nlev] = run;
  }
}

__global__ void origin_kernel(const unsigned* __restrict__ keys, const unsigned* __restrict__ first, unsigned np, int* __restrict__ origin) {
  const unsigned p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= np) return;
  const unsigned key = keys[first[p]];
  origin[3 * p] = (int)compact3(key);
  origin[3 * p + 1] = (int)compact3(key >> 1);
  origin[3 * p + 2] = (int)compact3(key >> 2);
}

}  // namespace

// ---- host side: C-ABI of the patch builder (include/amr_godunov.h) ---------------------------------------
struct amr_patch_builder {
  int64_t cap = 0;            // cells the workspace was sized for
  cudaStream_t stream = nullptr;
  unsigned *keys[2] = {nullptr, nullptr}, *vals[2] = {nullptr, nullptr};
  unsigned* hist = nullptr;   // [256][nb]
  unsigned char* lev = nullptr;    // [cap] level | head bit
  unsigned* counts = nullptr;      // compaction block counts
  unsigned* pfirst = nullptr;      // [cap] first cell (curve position) of each patch
  unsigned char* plev = nullptr;   // [cap]
  unsigned* slot_first = nullptr;  // [cap] first cell of every patch, grouped by level (curve order inside a level)
  unsigned* lbase = nullptr;       // [8] device copy of lbase_host
  unsigned lbase_host[8] = {0, 0, 0, 0, 0, 0, 0, 0};   // patches of level k: slots [lbase[k], lbase[k+1])
  int* porigin = nullptr;          // [cap][3] origins of all patches
  int* sorigin = nullptr;          // [cap][3] origins of the patches of the level last gathered
  unsigned* dup = nullptr;
  unsigned* totals = nullptr;      // [256] digit totals of a sort pass
  int cur = 0;                // which keys/vals buffer holds the sorted result
  int64_t ncell = 0, npatch = 0;
  int bits = 0, kmax = 0;
  bool built = false;
};

namespace {

struct BLayout { size_t keys[2], vals[2], hist, lev, counts, pfirst, plev, slot_first, porigin, sorigin, dup, totals, lbase, total; };

BLayout builder_layout(int64_t cap) {
  BLayout L;
  const size_t n = (size_t)cap, nb = (n + SORT_ITEMS - 1) / SORT_ITEMS, ncb = (n + CMP_ITEMS - 1) / CMP_ITEMS;
  size_t off = 0;
  for (int b = 0; b < 2; ++b) { L.keys[b] = off; off += up(n * 4); L.vals[b] = off; off += up(n * 4); }
  L.hist = off; off += up(256 * nb * 4);
  L.lev = off; off += up(n);
  L.counts = off; off += up(7 * (ncb + 1) * 4);   // heads + one row per level
  L.pfirst = off; off += up(n * 4);
  L.plev = off; off += up(n);
  L.slot_first = off; off += up(n * 4);
  L.porigin = off; off += up(n * 12);
  L.sorigin = off; off += up(n * 12);
  L.dup = off; off += up(16);
  L.totals = off; off += up(256 * 4);
  L.lbase = off; off += up(8 * 4);
  L.total = off;
  return L;
}

#define B_TRY(expr)                                                                                     \
  do {                                                                                                  \
    cudaError_t e_ = (expr);                                                                            \
    if (e_ != cudaSuccess) return amr::set_error(AMR_ECUDA, #expr, cudaGetErrorString(e_));             \
  } while (0)

// ordered compaction of the flagged items of [0, n): returns the number of flagged items
template <int MODE>
int compact(amr_patch_builder* b, const unsigned char* flags, const unsigned* src_first, unsigned n, int k,
            unsigned* out_first, unsigned char* out_lev, unsigned* total) {
  const unsigned ncb = (n + CMP_ITEMS - 1) / CMP_ITEMS;
  count_kernel<MODE><<<ncb, 256, 0, b->stream>>>(flags, n, k, b->counts);
  B_TRY(cudaMemsetAsync(b->counts + ncb, 0, 4, b->stream));
  scan_kernel<<<1, 1024, 0, b->stream>>>(b->counts, ncb + 1);     // counts[ncb] becomes the total
  write_kernel<MODE><<<ncb, 256, 0, b->stream>>>(flags, src_first, n, k, b->counts, nullptr, out_first, out_lev);
  B_TRY(cudaGetLastError());
  B_TRY(cudaMemcpyAsync(total, b->counts + ncb, 4, cudaMemcpyDeviceToHost, b->stream));
  B_TRY(cudaStreamSynchronize(b->stream));
  return AMR_OK;
}

}  // namespace

extern "C" {

size_t amr_builder_bytes(int64_t ncell_max) {
  if (ncell_max < 1 || ncell_max > (int64_t)1 << 30) return 0;
  return builder_layout(ncell_max).total;
}

int amr_builder_create(int64_t ncell_max, void* dev_ws, size_t bytes, void* cuda_stream, amr_patch_builder** out) {
  if (!out) return amr::set_error(AMR_EINVAL, "amr_builder_create", "null out");
  *out = nullptr;
  if (ncell_max < 1 || ncell_max > (int64_t)1 << 30) return amr::set_error(AMR_EINVAL, "amr_builder_create", "ncell_max out of range [1, 2^30]");
  if (!dev_ws || ((uintptr_t)dev_ws & (ALIGN - 1))) return amr::set_error(AMR_EINVAL, "amr_builder_create", "workspace null or not 256-byte aligned");
  const BLayout L = builder_layout(ncell_max);
  if (bytes < L.total) return amr::set_error(AMR_ENOMEM, "amr_builder_create", "workspace smaller than amr_builder_bytes()");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return amr::set_error(AMR_ECUDA, "amr_builder_create", "no CUDA device (there is no CPU fallback)");
  amr_patch_builder* b = new (std::nothrow) amr_patch_builder;
  if (!b) return amr::set_error(AMR_ENOMEM, "amr_builder_create", "host allocation failed");
  char* w = (char*)dev_ws;
  b->cap = ncell_max;
  b->stream = (cudaStream_t)cuda_stream;
  for (int i = 0; i < 2; ++i) { b->keys[i] = (unsigned*)(w + L.keys[i]); b->vals[i] = (unsigned*)(w + L.vals[i]); }
  b->hist = (unsigned*)(w + L.hist);
  b->lev = (unsigned char*)(w + L.lev);
  b->counts = (unsigned*)(w + L.counts);
  b->pfirst = (unsigned*)(w + L.pfirst);
  b->plev = (unsigned char*)(w + L.plev);
  b->slot_first = (unsigned*)(w + L.slot_first);
  b->porigin = (int*)(w + L.porigin);
  b->sorigin = (int*)(w + L.sorigin);
  b->dup = (unsigned*)(w + L.dup);
  b->totals = (unsigned*)(w + L.totals);
  b->lbase = (unsigned*)(w + L.lbase);
  *out = b;
  return AMR_OK;
}

int amr_builder_destroy(amr_patch_builder* b) {
  delete b;
  return AMR_OK;
}

int amr_builder_build(amr_patch_builder* b, const int32_t* dev_xyz, int64_t ncell, int32_t bits, int32_t kmax,
                      int64_t* npatch_out) {
  if (!b || !dev_xyz || !npatch_out) return amr::set_error(AMR_EINVAL, "amr_builder_build", "null argument");
  if (ncell < 1 || ncell > b->cap) return amr::set_error(AMR_EINVAL, "amr_builder_build", "ncell out of range for this builder");
  if (bits < 1 || bits > 10) return amr::set_error(AMR_EINVAL, "amr_builder_build", "bits per direction must be 1..10");
  if (kmax < 0 || kmax > 5 || kmax > bits) return amr::set_error(AMR_EINVAL, "amr_builder_build", "kmax must be 0..min(5, bits)");
  b->built = false;
  const unsigned n = (unsigned)ncell, nb = (n + SORT_ITEMS - 1) / SORT_ITEMS;
  key_kernel<<<(n + 255) / 256, 256, 0, b->stream>>>(dev_xyz, n, b->keys[0], b->vals[0]);
  int cur = 0;
  for (int shift = 0; shift < 3 * bits; shift += 8) {   // LSD radix sort, 8 bits per pass
    hist_kernel<<<nb, SORT_THREADS, 0, b->stream>>>(b->keys[cur], n, shift, nb, b->hist);
    scan_rows_kernel<<<256, 256, 0, b->stream>>>(b->hist, nb, b->totals);
    scatter_kernel<<<nb, SORT_THREADS, 0, b->stream>>>(b->keys[cur], b->vals[cur], n, shift, nb, b->hist, b->totals, b->keys[1 - cur], b->vals[1 - cur]);
    cur = 1 - cur;
  }
  B_TRY(cudaGetLastError());
  b->cur = cur;
  B_TRY(cudaMemsetAsync(b->dup, 0, 4, b->stream));
  level_kernel<<<(n + 255) / 256, 256, 0, b->stream>>>(b->keys[cur], n, kmax, b->lev, b->dup);
  unsigned np = 0, dup = 0;
  int rc = compact<0>(b, b->lev, nullptr, n, 0, b->pfirst, b->plev, &np);
  if (rc != AMR_OK) return rc;
  B_TRY(cudaMemcpyAsync(&dup, b->dup, 4, cudaMemcpyDeviceToHost, b->stream));
  origin_kernel<<<(np + 255) / 256, 256, 0, b->stream>>>(b->keys[cur], b->pfirst, np, b->porigin);
  {  // group the patch table by level for the gather (ordered compaction per level, no host round trip)
    const unsigned ncbp = (np + CMP_ITEMS - 1) / CMP_ITEMS, stride = ncbp + 1;
    unsigned* cl = b->counts + ((size_t)n + CMP_ITEMS - 1) / CMP_ITEMS + 1;   // rows 1..6 behind the heads' row
    B_TRY(cudaMemsetAsync(cl, 0, (size_t)(kmax + 1) * stride * 4, b->stream));
    for (int k = 0; k <= kmax; ++k) {
      count_kernel<1><<<ncbp, 256, 0, b->stream>>>(b->plev, np, k, cl + (size_t)k * stride);
      scan_kernel<<<1, 1024, 0, b->stream>>>(cl + (size_t)k * stride, stride);
    }
    bases_kernel<<<1, 32, 0, b->stream>>>(cl, stride, ncbp, kmax + 1, b->lbase);
    for (int k = 0; k <= kmax; ++k)
      write_kernel<1><<<ncbp, 256, 0, b->stream>>>(b->plev, b->pfirst, np, k, cl + (size_t)k * stride, b->lbase + k, b->slot_first, nullptr);
    origin_kernel<<<(np + 255) / 256, 256, 0, b->stream>>>(b->keys[cur], b->slot_first, np, b->sorigin);
    B_TRY(cudaMemcpyAsync(b->lbase_host, b->lbase, (size_t)(kmax + 2) * 4, cudaMemcpyDeviceToHost, b->stream));
  }
  B_TRY(cudaGetLastError());
  B_TRY(cudaStreamSynchronize(b->stream));
  if (dup) return amr::set_error(AMR_EINVAL, "amr_builder_build", "duplicate cells in the input");
  b->ncell = ncell; b->npatch = np; b->bits = bits; b->kmax = kmax; b->built = true;
  *npatch_out = np;
  return AMR_OK;
}

int amr_builder_results(amr_patch_builder* b, int64_t* perm, int64_t* first, int32_t* level, int32_t* origin) {
  if (!b) return amr::set_error(AMR_EINVAL, "amr_builder_results", "null builder");
  if (!b->built) return amr::set_error(AMR_ESTATE, "amr_builder_results", "no successful amr_builder_build yet");
  const size_t n = (size_t)b->ncell, np = (size_t)b->npatch;
  unsigned* tmp = new (std::nothrow) unsigned[n > np ? n : np];
  unsigned char* tl = new (std::nothrow) unsigned char[np ? np : 1];
  if (!tmp || !tl) { delete[] tmp; delete[] tl; return amr::set_error(AMR_ENOMEM, "amr_builder_results", "host allocation failed"); }
  cudaError_t e = cudaSuccess;
  if (perm && e == cudaSuccess) {
    e = cudaMemcpyAsync(tmp, b->vals[b->cur], n * 4, cudaMemcpyDeviceToHost, b->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(b->stream);
    for (size_t i = 0; i < n && e == cudaSuccess; ++i) perm[i] = tmp[i];
  }
  if (first && e == cudaSuccess) {
    e = cudaMemcpyAsync(tmp, b->pfirst, np * 4, cudaMemcpyDeviceToHost, b->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(b->stream);
    for (size_t i = 0; i < np && e == cudaSuccess; ++i) first[i] = tmp[i];
  }
  if (level && e == cudaSuccess) {
    e = cudaMemcpyAsync(tl, b->plev, np, cudaMemcpyDeviceToHost, b->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(b->stream);
    for (size_t i = 0; i < np && e == cudaSuccess; ++i) level[i] = tl[i];
  }
  if (origin && e == cudaSuccess) {
    e = cudaMemcpyAsync(origin, b->porigin, np * 12, cudaMemcpyDeviceToHost, b->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(b->stream);
  }
  delete[] tmp; delete[] tl;
  if (e != cudaSuccess) return amr::set_error(AMR_ECUDA, "amr_builder_results", cudaGetErrorString(e));
  return AMR_OK;
}

int amr_builder_gather(amr_patch_builder* b, const void* dev_fields, int32_t nfields, int32_t dtype, int32_t k,
                       void* dev_out, int64_t max_patches, int32_t* host_origin, int64_t* count_out) {
  if (!b || !count_out) return amr::set_error(AMR_EINVAL, "amr_builder_gather", "null argument");
  if (!b->built) return amr::set_error(AMR_ESTATE, "amr_builder_gather", "no successful amr_builder_build yet");
  if (k < 0 || k > b->kmax) return amr::set_error(AMR_EINVAL, "amr_builder_gather", "k outside 0..kmax of the build");
  if (nfields < 1 || (dtype != AMR_F32 && dtype != AMR_F64)) return amr::set_error(AMR_EINVAL, "amr_builder_gather", "bad nfields or dtype");
  const unsigned ns = b->lbase_host[k + 1] - b->lbase_host[k];
  const unsigned* slots = b->slot_first + b->lbase_host[k];
  *count_out = ns;
  if ((!dev_out && !host_origin) || ns == 0) return AMR_OK;  // count query, or nothing to gather
  if (!dev_fields || !dev_out) return amr::set_error(AMR_EINVAL, "amr_builder_gather", "null field pointers");
  if ((int64_t)ns > max_patches) return amr::set_error(AMR_ENOMEM, "amr_builder_gather", "output holds fewer patches than this level has");
  const size_t total = (size_t)ns << (3 * k);
  const unsigned grid = (unsigned)((total + 255) / 256);
  if (dtype == AMR_F32)
    gather_kernel<float><<<grid, 256, 0, b->stream>>>((const float*)dev_fields, (size_t)b->ncell, nfields, b->vals[b->cur], slots, ns, k, (float*)dev_out);
  else
    gather_kernel<double><<<grid, 256, 0, b->stream>>>((const double*)dev_fields, (size_t)b->ncell, nfields, b->vals[b->cur], slots, ns, k, (double*)dev_out);
  B_TRY(cudaGetLastError());
  if (!host_origin) return AMR_OK;                           // enqueued; the caller's stream orders later work
  B_TRY(cudaMemcpyAsync(host_origin, b->sorigin + 3 * (size_t)b->lbase_host[k], (size_t)ns * 12, cudaMemcpyDeviceToHost, b->stream));
  B_TRY(cudaStreamSynchronize(b->stream));
  return AMR_OK;
}

}  // extern "C"

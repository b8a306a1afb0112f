// Small kernels around the fused step: standalone CFL reduction (O7), conserved totals, ghosted
// gather / interior scatter for upload/download (O0 as seen through the API), and the two-level
// operators prolongation (O8), restriction and reflux (O9).  DESIGN.md §3, §6.
#include <math_constants.h>

#include "amr_internal.hpp"
#include "signal_speed.cuh"

namespace amr {

namespace {

template <class T> __device__ __forceinline__ void atomic_max_slot(void* slot, T v);
template <> __device__ __forceinline__ void atomic_max_slot<float>(void* slot, float v) {
  atomicMax(reinterpret_cast<unsigned int*>(slot), __float_as_uint(v));
}
template <> __device__ __forceinline__ void atomic_max_slot<double>(void* slot, double v) {
  atomicMax(reinterpret_cast<unsigned long long*>(slot), (unsigned long long)__double_as_longlong(v));
}

// ---- O7 standalone: grid-stride over interior cells, warp-shuffle max, one atomic per CTA ----------
template <class T, int NF>
__global__ void __launch_bounds__(256) smax_kernel(const T* __restrict__ U, size_t ncell, size_t fstride, T gamma, T gm1,
                                                   void* slot) {
  T m = T(0);
  for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < ncell; c += (size_t)gridDim.x * blockDim.x) {
    T u[NF];
#pragma unroll
    for (int q = 0; q < NF; ++q) u[q] = __ldg(U + (size_t)q * fstride + c);
    m = max_(m, signal_speed<T, NF>(u, gamma, gm1));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max_(m, __shfl_xor_sync(0xffffffffu, m, o));
  __shared__ T red[8];
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    T r = red[0];
    for (int w = 1; w < 8; ++w) r = max_(r, red[w]);
    atomic_max_slot<T>(slot, r);
  }
}

// ---- conserved totals: fixed grid, fixed per-thread order, tree reduce -> deterministic ------------
template <class T>
__global__ void __launch_bounds__(256) totals_kernel(const T* __restrict__ U, size_t ncell, size_t fstride, double* partials) {
  const int q = blockIdx.y;
  const T* u = U + (size_t)q * fstride;
  double s = 0.0;
  for (size_t c = (size_t)blockIdx.x * 256 + threadIdx.x; c < ncell; c += (size_t)gridDim.x * 256) s += (double)u[c];
  __shared__ double red[256];
  red[threadIdx.x] = s;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) partials[(size_t)q * gridDim.x + blockIdx.x] = red[0];
}

// ---- O0 through the API: ghosted copy of patches [p0, p0+npc) --------------------------------------
template <class T>
__global__ void __launch_bounds__(256) gather_ghosted_kernel(const T* __restrict__ U, const T* __restrict__ halo,
                                                             const int* __restrict__ nbr, int nf, int np, int n,
                                                             int g, int p0, int npc, T* __restrict__ out) {
  const int M = n + 2 * g;
  const size_t M3 = (size_t)M * M * M, n3 = (size_t)n * n * n;
  const size_t total = (size_t)npc * M3;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (size_t)gridDim.x * blockDim.x) {
    const int pc = (int)(t / M3);
    const size_t c = t - (size_t)pc * M3;
    const int p = p0 + pc;
    const int gz = (int)(c / ((size_t)M * M)), gy = (int)((c / M) % M), gx = (int)(c % M);
    const int lx = gx - g, ly = gy - g, lz = gz - g;
    const int rx = lx < 0 ? 0 : (lx >= n ? 2 : 1), ry = ly < 0 ? 0 : (ly >= n ? 2 : 1), rz = lz < 0 ? 0 : (lz >= n ? 2 : 1);
    const int e = nbr[p * 27 + rz * 9 + ry * 3 + rx];
    const T* src;
    size_t fs;
    if (e >= 0) {
      const int sp = e & NBR_PATCH_MASK, md = e >> NBR_MODE_SHIFT;
      const int sx = (rx != 1 && (md & 1)) ? (rx == 0 ? 0 : n - 1) : lx - (rx - 1) * n;
      const int sy = (ry != 1 && (md & 2)) ? (ry == 0 ? 0 : n - 1) : ly - (ry - 1) * n;
      const int sz = (rz != 1 && (md & 4)) ? (rz == 0 ? 0 : n - 1) : lz - (rz - 1) * n;
      src = U + (size_t)sp * n3 + ((size_t)sz * n + sy) * n + sx;
      fs = (size_t)np * n3;
    } else {
      src = halo + (size_t)p * M3 + c;
      fs = (size_t)np * M3;
    }
    for (int q = 0; q < nf; ++q) out[((size_t)q * npc + pc) * M3 + c] = src[(size_t)q * fs];
  }
}

template <class T>
__global__ void __launch_bounds__(256) scatter_interior_kernel(const T* __restrict__ staged, int nf, int np, int n,
                                                               int g, int p0, int npc, T* __restrict__ U) {
  const int M = n + 2 * g;
  const size_t M3 = (size_t)M * M * M, n3 = (size_t)n * n * n;
  const size_t total = (size_t)npc * n3;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (size_t)gridDim.x * blockDim.x) {
    const int pc = (int)(t / n3);
    const size_t c = t - (size_t)pc * n3;
    const int k = (int)(c / ((size_t)n * n)), j = (int)((c / n) % n), i = (int)(c % n);
    const size_t cg = ((size_t)(k + g) * M + (j + g)) * M + (i + g);
    for (int q = 0; q < nf; ++q)
      U[((size_t)q * np + p0 + pc) * n3 + c] = staged[((size_t)q * npc + pc) * M3 + cg];
  }
}

template <class T>
__global__ void fill_nan_kernel(T* ptr, size_t count) {
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < count; t += (size_t)gridDim.x * blockDim.x)
    ptr[t] = (T)CUDART_NAN;
}

// ---- O8: prolongation into the fine halo ----------------------------------------------------------
template <class T> __device__ __forceinline__ T minmod2(T a, T b) {
  const T lo = a < b ? a : b, hi = a < b ? b : a;
  return (lo > T(0) ? lo : T(0)) + (hi < T(0) ? hi : T(0));
}

// O8 without tables (round 2: the host-built lists were 120 B per parent cell - 161 MB for a 944-patch level - and
// 30-137 ms of host time per relink).  One thread per (fine patch p, parent position (li, lj, lk) in the patch's halo
// box): the box spans the fine offsets -4 .. n+3, hp = n/2 + 4 parents per side, parent l <-> children 2(l-2), 2(l-2)+1
// (patch origins and n are even, so a parent never straddles a region boundary).  A parent whose region no sibling
// covers (neighbour table entry NBR_FROM_HALO) has its 7-point stencil resolved here through the coarse level's patch
// map (periodic faces wrap; at an outflow face the fine cells take the prolongation AT the clamped in-domain cell,
// parent and child parity of the clamped index; the +-1 stencil clamps like the coarse ghosts),
// the minmod slopes are taken once, and the children inside the g halo layers are written.
struct ProlongGeom {
  int n, g, npf;
  int domf[3], domc[3], cdims[3];
  int per_lo[3], per_hi[3];   // 1 = periodic face
};

// NC: the patch size as a compile-time constant (16, 32, 8: every division below becomes a shift or a multiply) or 0
// for any other size.  The first version of this kernel spent most of its instructions on run-time integer divisions
// and per-child index arithmetic inside the field loop (84e6 warp instructions, 137 us for a 944-patch level);
// everything that does not depend on the field is now computed once per thread (56e6, 107 us).
template <class T, int NC>
__global__ void __launch_bounds__(128) prolong_halo_kernel(T* __restrict__ halo, size_t fs_halo, int nf, ProlongGeom G,
                                                           const int* __restrict__ forigin, const int* __restrict__ nbr,
                                                           const int* __restrict__ cmap, const T* __restrict__ Uold,
                                                           const T* __restrict__ Unew, size_t fs_c, T theta) {
  const int n = NC ? NC : G.n, g = G.g, hp = n / 2 + 4, hp3 = hp * hp * hp;
  const int r = blockIdx.y * blockDim.x + threadIdx.x;   // parent position in the halo box; blockIdx.x = fine patch
  if (r >= hp3) return;
  const int p = blockIdx.x;
  const int l[3] = {r % hp, (r / hp) % hp, r / (hp * hp)};
  int reg = 0, C[3], forced[3], i0[3];
  const int pw[3] = {1, 3, 9};
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    i0[a] = 2 * (l[a] - 2);                              // fine offset of child 0 along a
    const int ra = i0[a] < 0 ? 0 : (i0[a] >= n ? 2 : 1);
    reg += ra * pw[a];
  }
  if (reg == 13 || nbr[p * 27 + reg] != NBR_FROM_HALO) return;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    int gi = forigin[3 * p + a] + i0[a];                 // even
    forced[a] = -1;
    if (gi < 0) {
      if (G.per_lo[a]) gi += G.domf[a]; else { gi = 0; forced[a] = 0; }
    } else if (gi >= G.domf[a]) {
      if (G.per_hi[a]) gi -= G.domf[a]; else { gi = G.domf[a] - 1; forced[a] = 1; }
    }
    C[a] = gi >> 1;
  }
  const int n2 = n * n, n3 = n2 * n;
  auto coarse_flat = [&](int cx, int cy, int cz) -> int {   // host guarantees np * n^3 < 2^31
    int c[3] = {cx, cy, cz};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      if (c[a] < 0) c[a] = G.per_lo[a] ? c[a] + G.domc[a] : 0;
      else if (c[a] >= G.domc[a]) c[a] = G.per_hi[a] ? c[a] - G.domc[a] : G.domc[a] - 1;
    }
    const int pc = cmap[((c[2] / n) * G.cdims[1] + c[1] / n) * G.cdims[0] + c[0] / n];   // nesting was checked at link time
    return pc * n3 + ((c[2] % n) * n + (c[1] % n)) * n + (c[0] % n);
  };
  // the centre through the map; a +-1 neighbour that stays inside the centre's coarse patch is one stride away
  int s[7];
  s[0] = coarse_flat(C[0], C[1], C[2]);
  const int lcx = C[0] % n, lcy = C[1] % n, lcz = C[2] % n;
  s[1] = lcx > 0 ? s[0] - 1 : coarse_flat(C[0] - 1, C[1], C[2]);
  s[2] = lcx < n - 1 ? s[0] + 1 : coarse_flat(C[0] + 1, C[1], C[2]);
  s[3] = lcy > 0 ? s[0] - n : coarse_flat(C[0], C[1] - 1, C[2]);
  s[4] = lcy < n - 1 ? s[0] + n : coarse_flat(C[0], C[1] + 1, C[2]);
  s[5] = lcz > 0 ? s[0] - n2 : coarse_flat(C[0], C[1], C[2] - 1);
  s[6] = lcz < n - 1 ? s[0] + n2 : coarse_flat(C[0], C[1], C[2] + 1);
  // per axis and child bit: inside the g halo layers?  sign of the slope term (the forced parity of a clamped face)
  const int M = n + 2 * g;
  bool ok[3][2];
  T wgt[3][2];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      const int i = i0[a] + b;
      ok[a][b] = i >= -g && i < n + g;
      wgt[a][b] = ((forced[a] >= 0 ? forced[a] : b) ? T(0.25) : T(-0.25));
    }
  const size_t off0 = ((size_t)p * M + (i0[2] + g)) * M * M + (size_t)(i0[1] + g) * M + (i0[0] + g);
  const T w0 = T(1) - theta;
  for (int q = 0; q < nf; ++q) {
    const T* a = Uold + (size_t)q * fs_c;
    const T* b = Unew + (size_t)q * fs_c;
    T st[7];
    if (theta == T(0)) {        // first substep: the old state alone (w0 = 1: the same value, half the loads)
#pragma unroll
      for (int k = 0; k < 7; ++k) st[k] = a[s[k]];
    } else {
#pragma unroll
      for (int k = 0; k < 7; ++k) st[k] = w0 * a[s[k]] + theta * b[s[k]];
    }
    T sl[3];
#pragma unroll
    for (int dd = 0; dd < 3; ++dd) sl[dd] = minmod2<T>(st[0] - st[1 + 2 * dd], st[2 + 2 * dd] - st[0]);
    T* out = halo + (size_t)q * fs_halo + off0;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const int bx = c & 1, by = (c >> 1) & 1, bz = c >> 2;
      if (!(ok[0][bx] && ok[1][by] && ok[2][bz])) continue;
      // U_C -+ 1/4 slope, accumulated in the order x, y, z (the products are exact: the order of the sums is what counts)
      T val = st[0];
      val += wgt[0][bx] * sl[0];
      val += wgt[1][by] * sl[1];
      val += wgt[2][bz] * sl[2];
      out[((size_t)bz * M + by) * M + bx] = val;
    }
  }
}

// ---- regridding ------------------------------------------------------------------
// One block per (patch, aligned (n/2)^3 block): flag = max of one field over the block > threshold.
template <class T>
__global__ void __launch_bounds__(128) flag_blocks_kernel(const T* __restrict__ U, int n, T threshold,
                                                          unsigned char* __restrict__ flags) {
  const int p = blockIdx.x >> 3, blk = blockIdx.x & 7;
  const int h = n >> 1, h3 = h * h * h;
  const int bx = blk & 1, by = (blk >> 1) & 1, bz = blk >> 2;
  const T* u = U + (size_t)p * n * n * n;
  bool hit = false;
  for (int r = threadIdx.x; r < h3; r += blockDim.x) {
    const int i = r % h, j = (r / h) % h, k = r / (h * h);
    hit |= u[((size_t)(bz * h + k) * n + (by * h + j)) * n + (bx * h + i)] > threshold;
  }
  const int any = __syncthreads_or(hit ? 1 : 0);
  if (threadIdx.x == 0) flags[blockIdx.x] = any ? 1 : 0;
}

// kept patches: pairs[e] = (new patch, old patch); grid (npairs, nf)
template <class T>
__global__ void __launch_bounds__(256) copy_patches_kernel(T* __restrict__ Unew, size_t fs_new,
                                                           const T* __restrict__ Uold, size_t fs_old,
                                                           const int2* __restrict__ pairs, int n3) {
  const int2 pr = pairs[blockIdx.x];
  const T* src = Uold + (size_t)blockIdx.y * fs_old + (size_t)pr.y * n3;
  T* dst = Unew + (size_t)blockIdx.y * fs_new + (size_t)pr.x * n3;
  for (int r = threadIdx.x; r < n3; r += blockDim.x) dst[r] = src[r];
}

// new-born patches, no tables (as prolong_halo_kernel): one thread per coarse parent cell; born[b] = (new patch index,
// fine origin x, y, z).  The parent block of a patch ((n/2)^3 coarse cells from origin / 2) lies inside ONE coarse
// patch; only the +-1 stencil can leave it, and it is resolved through the coarse patch map (periodic faces wrap, the
// stencil clamps at an outflow face like the coarse ghosts).  The 8 children get U_C -+ 1/4 minmod slopes,
// accumulated in the order x, y, z (O8).
template <class T>
__global__ void __launch_bounds__(128) prolong_patches_kernel(T* __restrict__ Unew, size_t fs_new, int nf, ProlongGeom G,
                                                              const int4* __restrict__ born,
                                                              const int* __restrict__ cmap, int nparents,
                                                              const T* __restrict__ Uc, size_t fs_c) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= nparents) return;
  const int n = G.n, h = n >> 1, h3 = h * h * h;
  const int b = e / h3, r = e - b * h3;
  const int ci = r % h, cj = (r / h) % h, ck = r / (h * h);
  const int4 bo = born[b];
  const int C[3] = {(bo.y >> 1) + ci, (bo.z >> 1) + cj, (bo.w >> 1) + ck};
  auto coarse_flat = [&](int cx, int cy, int cz) -> long long {
    int c[3] = {cx, cy, cz};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      if (c[a] < 0) c[a] = G.per_lo[a] ? c[a] + G.domc[a] : 0;
      else if (c[a] >= G.domc[a]) c[a] = G.per_hi[a] ? c[a] - G.domc[a] : G.domc[a] - 1;
    }
    const int pc = cmap[((c[2] / n) * G.cdims[1] + c[1] / n) * G.cdims[0] + c[0] / n];   // nesting was checked by the host
    return (long long)pc * n * n * n + ((long long)(c[2] % n) * n + (c[1] % n)) * n + (c[0] % n);
  };
  long long s[7];
  s[0] = coarse_flat(C[0], C[1], C[2]);
  s[1] = coarse_flat(C[0] - 1, C[1], C[2]); s[2] = coarse_flat(C[0] + 1, C[1], C[2]);
  s[3] = coarse_flat(C[0], C[1] - 1, C[2]); s[4] = coarse_flat(C[0], C[1] + 1, C[2]);
  s[5] = coarse_flat(C[0], C[1], C[2] - 1); s[6] = coarse_flat(C[0], C[1], C[2] + 1);
  T* dst0 = Unew + (size_t)bo.x * n * n * n + ((size_t)(2 * ck) * n + 2 * cj) * n + 2 * ci;
  for (int q = 0; q < nf; ++q) {
    const T* a = Uc + (size_t)q * fs_c;
    T st[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) st[k] = a[s[k]];
    T sl[3];
#pragma unroll
    for (int dd = 0; dd < 3; ++dd) sl[dd] = minmod2<T>(st[0] - st[1 + 2 * dd], st[2 + 2 * dd] - st[0]);
    T* dst = dst0 + (size_t)q * fs_new;
#pragma unroll
    for (int c = 0; c < 4; ++c) {       // the two x children of a (y, z) child pair go out as one vector store
      T lo = st[0], hi = st[0];
      lo += T(-0.25) * sl[0]; hi += T(0.25) * sl[0];
      const T sy = ((c & 1) ? T(0.25) : T(-0.25)) * sl[1], sz = ((c & 2) ? T(0.25) : T(-0.25)) * sl[2];
      lo += sy; hi += sy;
      lo += sz; hi += sz;
      T* d2 = dst + ((size_t)((c >> 1) & 1) * n + (c & 1)) * n;
      if constexpr (sizeof(T) == 4) *reinterpret_cast<float2*>(d2) = make_float2(lo, hi);
      else *reinterpret_cast<double2*>(d2) = make_double2(lo, hi);
    }
  }
}

// ---- O9(6): restriction ---------------------------------------------------------------------------
// No table: entry e <-> (fine patch p, coarse-cell offset (ci, cj, ck) inside the patch's parent block); the parent
// block of a fine patch lies in ONE coarse patch, found through the coarse patch map (nesting was checked at link time).
template <class T>
__global__ void __launch_bounds__(256) restrict_kernel(const T* __restrict__ Uf, size_t fs_f, int nf, ProlongGeom G,
                                                       const int* __restrict__ forigin, const int* __restrict__ cmap,
                                                       int nent, T* __restrict__ Uc, size_t fs_c) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= nent) return;
  const int n = G.n, h = n / 2, h3 = h * h * h;
  const int p = e / h3;
  int r = e - p * h3;
  const int ck = r / (h * h);
  r -= ck * h * h;
  const int cj = r / h, ci = r - cj * h;
  const size_t base = (size_t)p * n * n * n + ((size_t)(2 * ck) * n + 2 * cj) * n + 2 * ci;
  const int Cx = (forigin[3 * p] >> 1) + ci, Cy = (forigin[3 * p + 1] >> 1) + cj, Cz = (forigin[3 * p + 2] >> 1) + ck;
  const int pc = cmap[((Cz / n) * G.cdims[1] + Cy / n) * G.cdims[0] + Cx / n];
  const size_t d = (size_t)pc * n * n * n + ((size_t)(Cz % n) * n + (Cy % n)) * n + (Cx % n);
  for (int q = 0; q < nf; ++q) {
    const T* u = Uf + (size_t)q * fs_f + base;
    T s = T(0);
#pragma unroll
    for (int dk = 0; dk < 2; ++dk)
#pragma unroll
      for (int dj = 0; dj < 2; ++dj)
#pragma unroll
        for (int di = 0; di < 2; ++di) s += u[((size_t)dk * n + dj) * n + di];
    Uc[(size_t)q * fs_c + d] = s * T(0.125);
  }
}

// ---- O9(7): reflux --------------------------------------------------------------------------------
// No host table.  At link time reflux_find_kernel scans the cells of every coarse patch that owns a flux block
// (cblk[b] = (patch, origin x, y, z); block index = b, or = patch when the coarse level records per patch because it
// is a fine level itself) and appends to a device list every cell that is not covered by the fine level but has a
// covered face neighbour: entry = (flat cell index in the level, b << 6 | mask), mask bit d*2 + s set when the
// neighbour across (direction d, fine side s) is covered - fine side 0: the neighbour above (the interface is the fine
// patch's low face and this cell's upper face), 1: the neighbour below.  Neighbours are found through the fine patch
// map (periodic faces wrap; beyond a non-periodic face there is nothing: a fine face on the domain boundary carries a
// boundary flux of the composite grid).  The list order is arbitrary (atomic counter) and does
// not matter: reflux_list_kernel gives every entry one thread, which applies
//   U_C += s_f (dt/dx) (F_coarse - 1/4 * 1/2 * sum of the 4 fine face fluxes summed over the two substeps)
// for its set bits in ascending (d, s) - every cell is corrected by one thread in a fixed order.  ZERO: instead clear
// the coarse flux slots those corrections read (a middle level shares its blocks with its role as a fine level and
// must not clear more than its own faces).
// Flux blocks: [block][direction][field][3 face planes: index 0, n/2, n along the normal][n^2 in-plane, the lower
// remaining axis fastest].
struct RefluxGeom {
  int n, nf, shared;
  int domc[3], fdims[3];
  int per_lo[3], per_hi[3];
};

__device__ __forceinline__ int fine_patch_of(const RefluxGeom& G, const int* __restrict__ fmap, const int* c) {
  const int n = G.n;   // the fine patch covering the children of coarse cell c, or -1
  return fmap[(((2 * c[2]) / n) * G.fdims[1] + (2 * c[1]) / n) * G.fdims[0] + (2 * c[0]) / n];
}
// neighbour of C across (d, side) in level coordinates; false beyond a non-periodic face
__device__ __forceinline__ bool reflux_neighbour(const RefluxGeom& G, const int* C, int d, int side, int* Cn) {
  Cn[0] = C[0]; Cn[1] = C[1]; Cn[2] = C[2];
  Cn[d] += side ? -1 : 1;
  if (Cn[d] < 0) { if (!G.per_lo[d]) return false; Cn[d] += G.domc[d]; }
  else if (Cn[d] >= G.domc[d]) { if (!G.per_hi[d]) return false; Cn[d] -= G.domc[d]; }
  return true;
}

__global__ void __launch_bounds__(256) reflux_find_kernel(RefluxGeom G, const int4* __restrict__ cblk,
                                                          const int* __restrict__ fmap, int2* __restrict__ list,
                                                          int* __restrict__ count, int capacity) {
  const int n = G.n, n2 = n * n, n3 = n2 * n;
  const int r = blockIdx.y * blockDim.x + threadIdx.x;   // grid.x = entry of cblk
  if (r >= n3) return;
  const int l[3] = {r % n, (r / n) % n, r / n2};
  // a covered neighbour lies across the boundary of an aligned (n/2)^3 block: only cells on such a boundary go on
  const int h = n >> 1;
  unsigned cand = 0;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if ((l[d] + 1) % h == 0) cand |= 1u << (2 * d);
    if (l[d] % h == 0) cand |= 2u << (2 * d);
  }
  if (!cand) return;
  const int4 cb = cblk[blockIdx.x];
  const int C[3] = {cb.y + l[0], cb.z + l[1], cb.w + l[2]};
  if (fine_patch_of(G, fmap, C) >= 0) return;
  unsigned mask = 0;
#pragma unroll
  for (int d = 0; d < 3; ++d)
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      const unsigned bit = 1u << (2 * d + side);
      int Cn[3];
      if ((cand & bit) && reflux_neighbour(G, C, d, side, Cn) && fine_patch_of(G, fmap, Cn) >= 0) mask |= bit;
    }
  if (!mask) return;
  const int at = atomicAdd(count, 1);
  if (at < capacity) list[at] = make_int2(cb.x * n3 + r, (int)((blockIdx.x << 6) | mask));
}

template <class T, bool ZERO>
__global__ void __launch_bounds__(128) reflux_list_kernel(T* __restrict__ Uc, size_t fs_c, RefluxGeom G,
                                                          const int4* __restrict__ cblk, const int2* __restrict__ list,
                                                          int nlist, const int* __restrict__ fmap,
                                                          const int* __restrict__ forigin, T* __restrict__ Fc,
                                                          const T* __restrict__ Ff, T dtdx) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= nlist) return;
  const int n = G.n, n2 = n * n, n3 = n2 * n;
  const int2 ent = list[e];
  const int b = ent.y >> 6;
  const unsigned mask = (unsigned)ent.y & 63u;
  const int4 cb = cblk[b];
  const int blk = G.shared ? cb.x : b;
  const int r = ent.x - cb.x * n3;
  const int l[3] = {r % n, (r / n) % n, r / n2};
  const int C[3] = {cb.y + l[0], cb.z + l[1], cb.w + l[2]};
  const size_t fsz = (size_t)3 * n2;
  const size_t cell = (size_t)ent.x;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      if (!(mask & (1u << (2 * d + side)))) continue;
      // the face in this cell's patch: its upper face (index l[d] + 1) when the fine patch is above
      int lc[3] = {l[0], l[1], l[2]};
      if (!side) lc[d] += 1;
      const int sc = lc[d] == 0 ? 0 : (lc[d] == n ? 2 : 1);     // 1 <=> n/2: fine patches sit on aligned (n/2)^3 blocks
      const int ic = d == 0 ? lc[2] * n + lc[1] : (d == 1 ? lc[2] * n + lc[0] : lc[1] * n + lc[0]);
      const size_t oc = ((size_t)blk * 3 + d) * G.nf * fsz + (size_t)sc * n2 + ic;
      if (ZERO) {
        for (int q = 0; q < G.nf; ++q) Fc[oc + (size_t)q * fsz] = T(0);
        continue;
      }
      int Cn[3];
      reflux_neighbour(G, C, d, side, Cn);
      const int pf = fine_patch_of(G, fmap, Cn);
      // the four fine faces: the fine patch's low (side 0) or high (side 1) face plane, children of Cn in-plane
      int lf[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) lf[a] = 2 * Cn[a] - forigin[3 * pf + a];
      lf[d] = side ? n : 0;
      const int iff = d == 0 ? lf[2] * n + lf[1] : (d == 1 ? lf[2] * n + lf[0] : lf[1] * n + lf[0]);
      const size_t of = ((size_t)pf * 3 + d) * G.nf * fsz + (size_t)(side ? 2 : 0) * n2 + iff;
      // in-plane strides of the transverse directions t1 = (d+1)%3, t2 = (d+2)%3: d = 0: (z, y), 1: (z, x), 2: (y, x)
      const size_t sa = (d == 1) ? (size_t)n : 1, sb = (d == 1) ? 1 : (size_t)n;
      const T sf = side ? T(-1) : T(1);
      for (int q = 0; q < G.nf; ++q) {
        const T Fcoarse = Fc[oc + (size_t)q * fsz];
        const T* f = Ff + of + (size_t)q * fsz;
        T sum = T(0);
        sum += f[0];
        sum += f[sa];
        sum += f[sb];
        sum += f[sa + sb];
        const T Ffine = T(0.25) * T(0.5) * sum;
        Uc[(size_t)q * fs_c + cell] += sf * dtdx * (Fcoarse - Ffine);
      }
    }
  }
}

inline unsigned grid_for(size_t work, int block, unsigned cap = 148 * 16) {
  size_t g = (work + block - 1) / block;
  if (g < 1) g = 1;
  if (g > cap) g = cap;
  return (unsigned)g;
}

}  // namespace

cudaError_t launch_smax(int dtype, const void* U, int nf, int np, int np_active, int n, double gamma, void* slot, cudaStream_t s) {
  const size_t ncell = (size_t)np_active * n * n * n, fstride = (size_t)np * n * n * n;
  const unsigned grid = grid_for(ncell, 256, 148 * 8);
  if (dtype == 0) {
    const float g = (float)gamma, gm1 = (float)(gamma - 1.0);
    if (nf == 5) smax_kernel<float, 5><<<grid, 256, 0, s>>>((const float*)U, ncell, fstride, g, gm1, slot);
    else smax_kernel<float, 9><<<grid, 256, 0, s>>>((const float*)U, ncell, fstride, g, gm1, slot);
  } else {
    const double g = gamma, gm1 = gamma - 1.0;
    if (nf == 5) smax_kernel<double, 5><<<grid, 256, 0, s>>>((const double*)U, ncell, fstride, g, gm1, slot);
    else smax_kernel<double, 9><<<grid, 256, 0, s>>>((const double*)U, ncell, fstride, g, gm1, slot);
  }
  return cudaGetLastError();
}

cudaError_t launch_totals(int dtype, const void* U, int nf, int np, int np_active, int n, double* partials, cudaStream_t s) {
  const size_t ncell = (size_t)np_active * n * n * n, fstride = (size_t)np * n * n * n;
  dim3 grid(TOTALS_BLOCKS, nf);
  if (dtype == 0) totals_kernel<float><<<grid, 256, 0, s>>>((const float*)U, ncell, fstride, partials);
  else totals_kernel<double><<<grid, 256, 0, s>>>((const double*)U, ncell, fstride, partials);
  return cudaGetLastError();
}

cudaError_t launch_gather_ghosted(int dtype, const void* U, const void* halo, const int* nbr, int nf, int np, int n,
                                  int g, int p0, int npc, void* out, cudaStream_t s) {
  const int M = n + 2 * g;
  const unsigned grid = grid_for((size_t)npc * M * M * M, 256);
  if (dtype == 0)
    gather_ghosted_kernel<float><<<grid, 256, 0, s>>>((const float*)U, (const float*)halo, nbr, nf, np, n, g, p0, npc,
                                                     (float*)out);
  else
    gather_ghosted_kernel<double><<<grid, 256, 0, s>>>((const double*)U, (const double*)halo, nbr, nf, np, n, g, p0,
                                                      npc, (double*)out);
  return cudaGetLastError();
}

cudaError_t launch_scatter_interior(int dtype, const void* staged, int with_ghosts, int nf, int np, int n, int g,
                                    int p0, int npc, void* U, cudaStream_t s) {
  const unsigned grid = grid_for((size_t)npc * n * n * n, 256);
  const int ge = with_ghosts ? g : 0;
  if (dtype == 0)
    scatter_interior_kernel<float><<<grid, 256, 0, s>>>((const float*)staged, nf, np, n, ge, p0, npc, (float*)U);
  else
    scatter_interior_kernel<double><<<grid, 256, 0, s>>>((const double*)staged, nf, np, n, ge, p0, npc, (double*)U);
  return cudaGetLastError();
}

cudaError_t launch_fill_nan(int dtype, void* ptr, size_t count, cudaStream_t s) {
  const unsigned grid = grid_for(count, 256);
  if (dtype == 0) fill_nan_kernel<float><<<grid, 256, 0, s>>>((float*)ptr, count);
  else fill_nan_kernel<double><<<grid, 256, 0, s>>>((double*)ptr, count);
  return cudaGetLastError();
}

cudaError_t launch_prolong_halo(int dtype, void* halo, size_t fs_halo, int nf, int n, int g, int npf, const int* domf,
                                const int* domc, const int* cdims, const int* bc, const int* forigin, const int* nbr,
                                const int* cmap, const void* Ucold, const void* Ucnew, size_t fs_c, double theta,
                                cudaStream_t s) {
  if (npf == 0) return cudaSuccess;
  ProlongGeom G;
  G.n = n; G.g = g; G.npf = npf;
  for (int a = 0; a < 3; ++a) {
    G.domf[a] = domf[a]; G.domc[a] = domc[a]; G.cdims[a] = cdims[a];
    G.per_lo[a] = bc[2 * a] == 0; G.per_hi[a] = bc[2 * a + 1] == 0;   // AMR_BC_PERIODIC == 0
  }
  const int hp = n / 2 + 4;
  const dim3 grid((unsigned)npf, (unsigned)((hp * hp * hp + 127) / 128));
#define AMR_PROLONG(TT, NCV) \
  prolong_halo_kernel<TT, NCV><<<grid, 128, 0, s>>>((TT*)halo, fs_halo, nf, G, forigin, nbr, cmap, (const TT*)Ucold, \
                                                    (const TT*)Ucnew, fs_c, (TT)theta)
  if (dtype == 0) {
    if (n == 16) AMR_PROLONG(float, 16); else if (n == 32) AMR_PROLONG(float, 32); else if (n == 8) AMR_PROLONG(float, 8);
    else AMR_PROLONG(float, 0);
  } else {
    if (n == 16) AMR_PROLONG(double, 16); else if (n == 32) AMR_PROLONG(double, 32); else if (n == 8) AMR_PROLONG(double, 8);
    else AMR_PROLONG(double, 0);
  }
#undef AMR_PROLONG
  return cudaGetLastError();
}

static ProlongGeom coarse_geom(int n, const int* domc, const int* cdims, const int* bc) {
  ProlongGeom G;
  G.n = n; G.g = 0; G.npf = 0;
  for (int a = 0; a < 3; ++a) {
    G.domf[a] = 2 * domc[a]; G.domc[a] = domc[a]; G.cdims[a] = cdims[a];
    G.per_lo[a] = bc[2 * a] == 0; G.per_hi[a] = bc[2 * a + 1] == 0;   // AMR_BC_PERIODIC == 0
  }
  return G;
}

cudaError_t launch_restrict(int dtype, const void* Uf, size_t fs_f, int nf, int n, int npf, const int* domc, const int* cdims,
                            const int* bc, const int* forigin, const int* cmap, void* Uc, size_t fs_c, cudaStream_t s) {
  const int h = n / 2, nent = npf * h * h * h;
  if (nent == 0) return cudaSuccess;
  const ProlongGeom G = coarse_geom(n, domc, cdims, bc);
  const unsigned grid = (unsigned)((nent + 255) / 256);
  if (dtype == 0)
    restrict_kernel<float><<<grid, 256, 0, s>>>((const float*)Uf, fs_f, nf, G, forigin, cmap, nent, (float*)Uc, fs_c);
  else
    restrict_kernel<double><<<grid, 256, 0, s>>>((const double*)Uf, fs_f, nf, G, forigin, cmap, nent, (double*)Uc, fs_c);
  return cudaGetLastError();
}

static RefluxGeom reflux_geom(int nf, int n, int shared, const int* domc, const int* fdims, const int* bc) {
  RefluxGeom G;
  G.n = n; G.nf = nf; G.shared = shared;
  for (int a = 0; a < 3; ++a) {
    G.domc[a] = domc[a]; G.fdims[a] = fdims[a];
    G.per_lo[a] = bc[2 * a] == 0; G.per_hi[a] = bc[2 * a + 1] == 0;
  }
  return G;
}

cudaError_t launch_reflux_find(int nf, int n, int shared, const int* domc, const int* fdims, const int* bc, const void* cblk,
                               int ncblk, const int* fmap, void* list, int* count, int capacity, cudaStream_t s) {
  cudaError_t e = cudaMemsetAsync(count, 0, sizeof(int), s);
  if (e != cudaSuccess || ncblk == 0) return e;
  const RefluxGeom G = reflux_geom(nf, n, shared, domc, fdims, bc);
  const dim3 grid((unsigned)ncblk, (unsigned)((n * n * n + 255) / 256));
  reflux_find_kernel<<<grid, 256, 0, s>>>(G, (const int4*)cblk, fmap, (int2*)list, count, capacity);
  return cudaGetLastError();
}

cudaError_t launch_reflux(int dtype, void* Uc, size_t fs_c, int nf, int n, int shared, const int* domc, const int* fdims,
                          const int* bc, const void* cblk, const void* list, int nlist, const int* fmap, const int* forigin,
                          void* Fc, const void* Ff, double dtdx, cudaStream_t s) {
  if (nlist == 0) return cudaSuccess;
  const RefluxGeom G = reflux_geom(nf, n, shared, domc, fdims, bc);
  const unsigned grid = (unsigned)((nlist + 127) / 128);
  if (dtype == 0)
    reflux_list_kernel<float, false><<<grid, 128, 0, s>>>((float*)Uc, fs_c, G, (const int4*)cblk, (const int2*)list, nlist, fmap,
                                                          forigin, (float*)Fc, (const float*)Ff, (float)dtdx);
  else
    reflux_list_kernel<double, false><<<grid, 128, 0, s>>>((double*)Uc, fs_c, G, (const int4*)cblk, (const int2*)list, nlist, fmap,
                                                           forigin, (double*)Fc, (const double*)Ff, dtdx);
  return cudaGetLastError();
}

cudaError_t launch_zero_faces(int dtype, void* Fc, int nf, int n, int shared, const int* domc, const int* fdims, const int* bc,
                              const void* cblk, const void* list, int nlist, cudaStream_t s) {
  if (nlist == 0) return cudaSuccess;
  const RefluxGeom G = reflux_geom(nf, n, shared, domc, fdims, bc);
  const unsigned grid = (unsigned)((nlist + 127) / 128);
  if (dtype == 0)
    reflux_list_kernel<float, true><<<grid, 128, 0, s>>>(nullptr, 0, G, (const int4*)cblk, (const int2*)list, nlist, nullptr,
                                                         nullptr, (float*)Fc, nullptr, 0.f);
  else
    reflux_list_kernel<double, true><<<grid, 128, 0, s>>>(nullptr, 0, G, (const int4*)cblk, (const int2*)list, nlist, nullptr,
                                                          nullptr, (double*)Fc, nullptr, 0.0);
  return cudaGetLastError();
}

// ---- measurement aid (bench.py alu_roofline.peak; not on the path): plain FMA throughput of the SMs -----------
// Every thread runs 8 independent chains of dependent fused multiply-adds (enough to cover the pipe latency
// at 8 warps per scheduler); 2 flops per FMA per lane.
template <class T>
__global__ void __launch_bounds__(256) fma_chain_kernel(T* sink, int iters, T a, T b) {
  T x[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) x[c] = (T)(threadIdx.x + c) * (T)1e-3;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int c = 0; c < 8; ++c) x[c] = fma(x[c], a, b);
    }
  }
  T s = 0;
#pragma unroll
  for (int c = 0; c < 8; ++c) s += x[c];
  if (s == (T)-123.456) sink[0] = s;     // never true for the launch arguments: keeps the chains alive
}

cudaError_t launch_fma_chain(int dtype, void* sink, int grid, int iters, cudaStream_t s) {
  if (dtype == 0) fma_chain_kernel<float><<<(unsigned)grid, 256, 0, s>>>((float*)sink, iters, 0.999f, 1e-3f);
  else fma_chain_kernel<double><<<(unsigned)grid, 256, 0, s>>>((double*)sink, iters, 0.999, 1e-3);
  return cudaGetLastError();
}

cudaError_t launch_flag_blocks(int dtype, const void* Ufield, int np, int n, double threshold, unsigned char* flags,
                               cudaStream_t s) {
  if (np == 0) return cudaSuccess;
  if (dtype == 0) flag_blocks_kernel<float><<<(unsigned)np * 8, 128, 0, s>>>((const float*)Ufield, n, (float)threshold, flags);
  else flag_blocks_kernel<double><<<(unsigned)np * 8, 128, 0, s>>>((const double*)Ufield, n, threshold, flags);
  return cudaGetLastError();
}

cudaError_t launch_copy_patches(int dtype, void* Unew, size_t fs_new, const void* Uold, size_t fs_old, const void* pairs,
                                int npairs, int nf, int n, cudaStream_t s) {
  if (npairs == 0) return cudaSuccess;
  const dim3 grid((unsigned)npairs, (unsigned)nf);
  const int n3 = n * n * n;
  if (dtype == 0) copy_patches_kernel<float><<<grid, 256, 0, s>>>((float*)Unew, fs_new, (const float*)Uold, fs_old, (const int2*)pairs, n3);
  else copy_patches_kernel<double><<<grid, 256, 0, s>>>((double*)Unew, fs_new, (const double*)Uold, fs_old, (const int2*)pairs, n3);
  return cudaGetLastError();
}

// the same copy with the roles of the pair swapped: pairs[e] = (slot in the packed source, patch in the destination)
template <class T>
__global__ void __launch_bounds__(256) copy_patches_in_kernel(T* __restrict__ U, size_t fs, const T* __restrict__ packed,
                                                              size_t fs_packed, const int2* __restrict__ pairs, int n3) {
  const int2 pr = pairs[blockIdx.x];
  const T* src = packed + (size_t)blockIdx.y * fs_packed + (size_t)pr.x * n3;
  T* dst = U + (size_t)blockIdx.y * fs + (size_t)pr.y * n3;
  for (int r = threadIdx.x; r < n3; r += blockDim.x) dst[r] = src[r];
}

cudaError_t launch_copy_patches_in(int dtype, void* U, size_t fs, const void* packed, size_t fs_packed, const void* pairs,
                                   int npairs, int nf, int n, cudaStream_t s) {
  if (npairs == 0) return cudaSuccess;
  const dim3 grid((unsigned)npairs, (unsigned)nf);
  const int n3 = n * n * n;
  if (dtype == 0) copy_patches_in_kernel<float><<<grid, 256, 0, s>>>((float*)U, fs, (const float*)packed, fs_packed, (const int2*)pairs, n3);
  else copy_patches_in_kernel<double><<<grid, 256, 0, s>>>((double*)U, fs, (const double*)packed, fs_packed, (const int2*)pairs, n3);
  return cudaGetLastError();
}

cudaError_t launch_prolong_patches(int dtype, void* Unew, size_t fs_new, int nf, int n, const int* domc, const int* cdims,
                                   const int* bc, const void* born, const int* cmap, int nparents, const void* Uc,
                                   size_t fs_c, cudaStream_t s) {
  if (nparents == 0) return cudaSuccess;
  ProlongGeom G;
  G.n = n; G.g = 0; G.npf = 0;
  for (int a = 0; a < 3; ++a) {
    G.domf[a] = 2 * domc[a]; G.domc[a] = domc[a]; G.cdims[a] = cdims[a];
    G.per_lo[a] = bc[2 * a] == 0; G.per_hi[a] = bc[2 * a + 1] == 0;   // AMR_BC_PERIODIC == 0
  }
  const unsigned grid = (unsigned)((nparents + 127) / 128);
  if (dtype == 0)
    prolong_patches_kernel<float><<<grid, 128, 0, s>>>((float*)Unew, fs_new, nf, G, (const int4*)born, cmap, nparents,
                                                       (const float*)Uc, fs_c);
  else
    prolong_patches_kernel<double><<<grid, 128, 0, s>>>((double*)Unew, fs_new, nf, G, (const int4*)born, cmap, nparents,
                                                        (const double*)Uc, fs_c);
  return cudaGetLastError();
}

}  // namespace amr

// Host side of libamrgodunov.so: the C-ABI of include/amr_godunov.h.  Batch object, arena carving,
// neighbour / coarse-fine tables (the "hierarchy and ghost-fill metadata kept on the host" of
// BASELINE.json:north_star), launches.  No solver arithmetic lives here.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>
#include <string>
#include <vector>
#include <cstdlib>
#include <atomic>
#include <utility>

#include "../../include/amr_godunov.h"
#include "amr_internal.hpp"
#include "ppm_params.hpp"

namespace {

thread_local std::string g_err;

int fail(int code, const char* fmt, ...) __attribute__((format(printf, 2, 3)));
int fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}

#define CUDA_TRY(expr)                                                                         \
  do {                                                                                         \
    cudaError_t e_ = (expr);                                                                   \
    if (e_ != cudaSuccess) return fail(AMR_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_));    \
  } while (0)

constexpr size_t ALIGN = 256;
inline size_t up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

struct Layout {
  size_t U[2], halo, nbr, fblk_of, counters, smax, partials, total;
};

bool desc_ok(const amr_batch_desc* d, std::string* why) {
  auto bad = [&](const char* m) { if (why) *why = m; return false; };
  if (!d) return bad("null desc");
  if (d->npatch < 1 || d->npatch > amr::NBR_PATCH_MASK) return bad("npatch out of range");
  if (d->n < 8 || d->n > 64 || d->n % 8) return bad("n must be a multiple of 8 in [8,64]");
  if (d->nghost < 2 || d->nghost > 4) return bad("nghost must be 2..4");
  if (d->nfields != 5 && d->nfields != 9) return bad("nfields must be 5 (hydro) or 9 (MHD)");
  if (d->dtype != AMR_F32 && d->dtype != AMR_F64) return bad("dtype must be AMR_F32 or AMR_F64");
  if (!(d->dx > 0) || !std::isfinite(d->dx)) return bad("dx must be finite and > 0");
  if (d->level < 0) return bad("level < 0");
  if (d->nactive < 0 || d->nactive > d->npatch) return bad("nactive must be in [0, npatch]");
  {  // the step kernel keeps per-field element offsets (interiors and ghosted halo buffer) in 32 bits
    const double M = d->n + 2.0 * d->nghost;
    if ((double)d->npatch * M * M * M > 2.0e9) return bad("more than 2e9 (ghosted) cells in one batch");
  }
  if (!d->self_periodic) {
    if (!d->origin) return bad("null origin");
    for (int a = 0; a < 3; ++a)
      if (d->domain_cells[a] < d->n || d->domain_cells[a] % d->n) return bad("domain_cells must be multiples of n");
    for (int a = 0; a < 6; ++a)
      if (d->bc[a] != AMR_BC_PERIODIC && d->bc[a] != AMR_BC_OUTFLOW) return bad("unknown boundary condition");
  }
  return true;
}

Layout make_layout(const amr_batch_desc* d) {
  Layout L;
  const size_t esz = d->dtype == AMR_F64 ? 8 : 4;
  const size_t n3 = (size_t)d->n * d->n * d->n;
  const size_t M = d->n + 2 * d->nghost, M3 = M * M * M;
  size_t off = 0;
  for (int b = 0; b < 2; ++b) { L.U[b] = off; off += up((size_t)d->nfields * d->npatch * n3 * esz); }
  L.halo = off;
  if (d->level > 0) off += up((size_t)d->nfields * d->npatch * M3 * esz);
  L.nbr = off; off += up((size_t)d->npatch * 27 * sizeof(int));
  L.fblk_of = off; off += up((size_t)d->npatch * sizeof(int));
  L.counters = off; off += up(4 * sizeof(unsigned long long));
  L.smax = off; off += up(16);
  L.partials = off; off += up((size_t)d->nfields * amr::TOTALS_BLOCKS * sizeof(double));
  L.total = off;
  return L;
}

// dense map patch-grid coordinate -> patch index (-1: none)
struct PatchMap {
  int dims[3];
  std::vector<int> idx;
  int at(int a, int b, int c) const { return idx[((size_t)c * dims[1] + b) * dims[0] + a]; }
};

}  // namespace

// Every entry point that takes a batch makes the batch's device current for the call and restores the caller's
// device afterwards (a second GPU in the same process must not receive this batch's launches).
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};

struct amr_patch_batch {
  amr_batch_desc d;
  std::vector<int32_t> origin;
  std::vector<int> nbr_host;
  PatchMap map;
  cudaStream_t stream;
  int nactive;       // the first nactive patches are stepped / reduced; the rest are read-only copies of remote patches (sharding)
  int device;        // the device the arena lives on (recorded at create; every call runs with it current)
  char* arena;
  size_t bytes, esz, n3, M3;
  void* U[2];
  int cur;
  void* halo;
  int* nbr_dev;
  int* fblk_of;  // device [np]; owned here, filled by a link
  void* fblk;    // device flux blocks, owned by a link (nullptr: no recording)
  unsigned long long* counters;
  void* smax_slot;
  double* partials;
  bool needs_halo, halo_valid;
  bool smax_valid;
  double smax_gamma;
  unsigned long long serial;  // unique per created batch (keys the link-table cache)
  amr_level_link* link_up;    // the link this batch is the fine side of (to its parent level)
  amr_level_link* link_down;  // the link this batch is the coarse side of (to its child level)
};

struct amr_level_link {
  amr_patch_batch *c, *f;
  char* ws;
  size_t bytes;
  // device tables: fine patch origins [npf][3], coarse and fine patch maps [z][y][x] (prolongation, restriction and
  // reflux resolve cells through them in the kernels), and per coarse flux block (patch, origin x, y, z)
  int *forg, *cmap, *fmap, *cblk;
  int ncblk;
  int* rlist;   // device, built at link time: (cell, block << 6 | mask) per uncovered coarse cell next to a fine face
  int nrlist;
  void *fblk_c, *fblk_f;
  size_t fblk_c_bytes, fblk_f_bytes;
  int nblk_c;
  bool shared_c;  // the coarse batch is itself a fine one: its per-patch blocks (owned by its link_up) are used
};

namespace {

struct LinkHost {
  std::vector<int> fblk_of_c;   // per coarse patch: its flux block or -1
  std::vector<int> cblk;        // per flux block of this link: (coarse patch, origin x, y, z)
  int nblk_c = 0;
  long long ncf_faces = 0;  // coarse-fine faces of fine patches: (n/2)^2 coarse cells each bound the reflux list
  bool identity_c = false;  // coarse blocks are per patch (block index = patch index)
};

struct LinkLayout {
  size_t forg, cmap, fmap, cblk, rlist, rcount, fblk_c, fblk_f, total, fblk_c_bytes, fblk_f_bytes;
  int rcap;
};

int wrapi(int v, int m) { return ((v % m) + m) % m; }

// Host side of a link (index conventions of include/amr_godunov.h).  O8, O9(6) and O9(7)
// resolve their cells in the kernels through the patch maps; what the host owes is (i) the check of proper nesting
// and (ii) the list of coarse patches that touch a coarse-fine face and therefore record fluxes.
int build_link(const amr_patch_batch* c, const amr_patch_batch* f, LinkHost& H) {
  const int n = f->d.n, g = f->d.nghost, nc = n / 2;
  const int* domf = f->d.domain_cells;
  const int* domc = c->d.domain_cells;
  auto coarse_patch = [&](int Cx, int Cy, int Cz) -> int {   // wrapped / clamped by the level's boundary conditions
    int C[3] = {Cx, Cy, Cz};
    for (int a = 0; a < 3; ++a) {
      if (C[a] < 0) C[a] = (c->d.bc[2 * a] == AMR_BC_PERIODIC) ? C[a] + domc[a] : 0;
      else if (C[a] >= domc[a]) C[a] = (c->d.bc[2 * a + 1] == AMR_BC_PERIODIC) ? C[a] - domc[a] : domc[a] - 1;
    }
    return c->map.at(C[0] / n, C[1] / n, C[2] / n);
  };
  // O8: every halo region of a fine patch that no sibling covers (and its +-1 stencil) must lie inside coarse
  // patches.  Checked per region at coarse-PATCH granularity: the region's parent cells, grown by one, span at most
  // two coarse patches per axis.
  if (g > 4) return fail(AMR_EINVAL, "nghost > 4 is not supported by the prolongation kernel");
  for (int p = 0; p < f->d.npatch; ++p) {
    const int* o = &f->origin[3 * p];
    const int lo[3] = {-g, 0, n}, hi[3] = {0, n, n + g};
    for (int reg = 0; reg < 27; ++reg) {
      if (reg == 13 || f->nbr_host[(size_t)p * 27 + reg] != amr::NBR_FROM_HALO) continue;
      const int rr[3] = {reg % 3, (reg / 3) % 3, reg / 9};
      int plo[3], phi[3];
      for (int a = 0; a < 3; ++a) {
        int flo = o[a] + lo[rr[a]], fhi = o[a] + hi[rr[a]] - 1;      // fine index range of the region along a
        // beyond a periodic face: the wrapped range; beyond an outflow face: the clamped cell
        if (flo < 0) { if (f->d.bc[2 * a] == AMR_BC_PERIODIC) { flo += domf[a]; fhi += domf[a]; } else { flo = fhi = 0; } }
        else if (fhi >= domf[a]) { if (f->d.bc[2 * a + 1] == AMR_BC_PERIODIC) { flo -= domf[a]; fhi -= domf[a]; } else { flo = fhi = domf[a] - 1; } }
        plo[a] = flo / 2 - 1;
        phi[a] = fhi / 2 + 1;
      }
      for (int cz = plo[2]; cz <= phi[2]; cz += (cz == phi[2] ? 1 : std::min(n, phi[2] - cz)))
        for (int cy = plo[1]; cy <= phi[1]; cy += (cy == phi[1] ? 1 : std::min(n, phi[1] - cy)))
          for (int cx = plo[0]; cx <= phi[0]; cx += (cx == phi[0] ? 1 : std::min(n, phi[0] - cx)))
            if (coarse_patch(cx, cy, cz) < 0) return fail(AMR_EINVAL, "fine patch %d has a halo cell with no coarse parent", p);
    }
  }
  // O9(6): the parent block of a fine patch ((n/2)^3 coarse cells, aligned) lies in one coarse patch
  for (int p = 0; p < f->d.npatch; ++p) {
    const int* o = &f->origin[3 * p];
    if (o[0] % nc || o[1] % nc || o[2] % nc) return fail(AMR_EINVAL, "fine patch %d is not aligned to an (n/2)^3 block of its parent level", p);
    if (c->map.at(o[0] / 2 / n, o[1] / 2 / n, o[2] / 2 / n) < 0) return fail(AMR_EINVAL, "fine patch %d is not covered by a coarse patch", p);
  }
  // O9(7): the coarse cells outside one face of a fine patch form one aligned (n/2)^2 x 1 slab of ONE coarse block:
  // either that block is refined too (fine-fine face, nothing to do) or its coarse patch records fluxes.  A fine face
  // on a non-periodic domain face has no coarse cell outside it: its flux is a boundary flux of the composite grid.
  H.fblk_of_c.assign(c->d.npatch, -1);
  for (int p = 0; p < f->d.npatch; ++p) {
    const int* o = &f->origin[3 * p];
    for (int d = 0; d < 3; ++d)
      for (int side = 0; side < 2; ++side) {
        int Cin[3] = {o[0] / 2, o[1] / 2, o[2] / 2};
        Cin[d] += side ? nc : -1;
        if ((Cin[d] < 0 && c->d.bc[2 * d] != AMR_BC_PERIODIC) || (Cin[d] >= domc[d] && c->d.bc[2 * d + 1] != AMR_BC_PERIODIC)) continue;
        int C[3];
        for (int e = 0; e < 3; ++e) C[e] = wrapi(Cin[e], domc[e]);
        if (f->map.at(2 * C[0] / n, 2 * C[1] / n, 2 * C[2] / n) >= 0) continue;  // fine-fine face
        const int pc = c->map.at(C[0] / n, C[1] / n, C[2] / n);
        if (pc < 0) return fail(AMR_EINVAL, "no coarse patch next to fine patch %d", p);
        H.ncf_faces++;
        if (H.fblk_of_c[pc] < 0) {
          H.fblk_of_c[pc] = H.identity_c ? pc : H.nblk_c++;
          const int* oc = &c->origin[3 * pc];
          H.cblk.push_back(pc); H.cblk.push_back(oc[0]); H.cblk.push_back(oc[1]); H.cblk.push_back(oc[2]);
        }
      }
  }
  return AMR_OK;
}

// amr_link_bytes has to build the tables to size the workspace; amr_link_levels, called next for the same pair,
// takes them from here instead of building them again (host work: O(halo cells) map look-ups)
struct LinkCache {
  unsigned long long c = 0, f = 0;
  bool identity_c = false;
  LinkHost H;
};
thread_local LinkCache g_link_cache;

LinkLayout make_link_layout(const amr_patch_batch* c, const amr_patch_batch* f, const LinkHost& H) {
  LinkLayout L;
  size_t off = 0;
  L.forg = off; off += up((size_t)f->d.npatch * 3 * sizeof(int) + 8);
  L.cmap = off; off += up(c->map.idx.size() * sizeof(int) + 8);
  L.fmap = off; off += up(f->map.idx.size() * sizeof(int) + 8);
  L.cblk = off; off += up(H.cblk.size() * sizeof(int) + 16);
  // a coarse cell enters the reflux list once, however many of its faces are coarse-fine: the face count bounds it
  L.rcap = (int)std::min<long long>(H.ncf_faces * (long long)(f->d.n / 2) * (f->d.n / 2), 0x7fffffffLL);
  L.rlist = off; off += up((size_t)L.rcap * 2 * sizeof(int) + 16);
  L.rcount = off; off += up(sizeof(int));
  const size_t n = f->d.n, blk = 3 * (size_t)f->d.nfields * 3 * n * n * f->esz;
  L.fblk_c_bytes = H.identity_c ? 0 : (size_t)H.nblk_c * blk;
  L.fblk_f_bytes = (size_t)f->d.npatch * blk;
  L.fblk_c = off; off += up(L.fblk_c_bytes + 8);
  L.fblk_f = off; off += up(L.fblk_f_bytes + 8);
  L.total = off;
  return L;
}

int check_link_args(const amr_patch_batch* c, const amr_patch_batch* f, int ratio) {
  if (!c || !f) return fail(AMR_EINVAL, "null batch");
  if (ratio != 2) return fail(AMR_EINVAL, "only refinement ratio 2 is supported");
  if (f->d.n % 2) return fail(AMR_EINVAL, "linked batches need an even patch size");
  if (c->d.n != f->d.n || c->d.nfields != f->d.nfields || c->d.dtype != f->d.dtype || c->d.nghost != f->d.nghost)
    return fail(AMR_EINVAL, "coarse and fine batches must agree in n, nfields, dtype, nghost");
  if (c->d.self_periodic || f->d.self_periodic) return fail(AMR_EINVAL, "self-periodic batches cannot be linked");
  for (int a = 0; a < 6; ++a)
    if (c->d.bc[a] != f->d.bc[a]) return fail(AMR_EINVAL, "linked batches must have the same boundary conditions");
  if (c->stream != f->stream) return fail(AMR_EINVAL, "linked batches must have been created on the same stream");
  if (c->device != f->device) return fail(AMR_EINVAL, "linked batches must live on the same device");
  if (f->d.level != c->d.level + 1) return fail(AMR_EINVAL, "fine.level must be coarse.level + 1");
  for (int a = 0; a < 3; ++a)
    if (f->d.domain_cells[a] != 2 * c->d.domain_cells[a]) return fail(AMR_EINVAL, "fine domain must be 2x the coarse domain");
  return AMR_OK;
}

template <class T>
amr::StepParams<T> make_params(amr_patch_batch* b, double dt, double gamma, double ch, double alpha) {
  amr::StepParams<T> P;
  std::memset(&P, 0, sizeof P);
  P.Uin = (const T*)b->U[b->cur];
  P.Uout = (T*)b->U[1 - b->cur];
  P.halo = (const T*)b->halo;
  P.nbr = b->nbr_dev;
  P.fblk = (T*)b->fblk;
  P.fblk_of = b->fblk ? b->fblk_of : nullptr;
  P.counters = b->counters;
  P.smax = b->smax_slot;
  P.np = b->d.npatch;
  P.np_active = b->nactive;
  P.n = b->d.n;
  P.g = b->d.nghost;
  const T dtT = (T)dt, dxT = (T)b->d.dx;
  P.dtdx = dtT / dxT;
  P.hdtdx = dtT / (T(2) * dxT);
  P.gamma = (T)gamma;
  P.gm1 = P.gamma - T(1);
  P.igm1 = T(1) / P.gm1;
  P.ch = (T)ch;
  P.ch2 = P.ch * P.ch;
  P.half_ich = ch > 0 ? T(1) / (T(2) * P.ch) : T(0);
  P.damp = (T)std::exp(-alpha * ch * dt / b->d.dx);
  P.eps = (T)(sizeof(T) == 8 ? 1e-12 : 1e-6);
  return P;
}

int do_step(amr_patch_batch* b, bool mhd, double dt, double gamma, int limiter, int riemann, double ch, double alpha) {
  if (!b) return fail(AMR_EINVAL, "null batch");
  DeviceGuard guard(b->device);
  if (mhd != (b->d.nfields == 9))
    return fail(AMR_EINVAL, "%s step on a batch with %d fields", mhd ? "MHD" : "hydro", b->d.nfields);
  if (!(dt > 0) || !std::isfinite(dt)) return fail(AMR_EINVAL, "dt must be finite and > 0");
  if (!std::isfinite(gamma) || !(gamma > 1)) return fail(AMR_EINVAL, "gamma must be finite and > 1");
  if (limiter < AMR_LIM_NONE || limiter > AMR_LIM_MC) return fail(AMR_EINVAL, "unknown limiter %d", limiter);
  if (mhd) {
    if (riemann != AMR_RS_HLL && riemann != AMR_RS_HLLD) return fail(AMR_EINVAL, "MHD step takes HLL or HLLD");
    if (!(ch > 0) || !std::isfinite(ch)) return fail(AMR_EINVAL, "ch must be finite and > 0");
    if (!(alpha >= 0) || !std::isfinite(alpha)) return fail(AMR_EINVAL, "alpha must be finite and >= 0");
  } else if (riemann != AMR_RS_HLL && riemann != AMR_RS_HLLC) {
    return fail(AMR_EINVAL, "hydro step takes HLL or HLLC");
  }
  if (b->needs_halo && !b->halo_valid)
    return fail(AMR_ESTATE, "level-%d batch has coarse-fine halo regions but amr_prolong_ghosts was never called", b->d.level);
  b->smax_valid = false;   // the slot is about to be zeroed; it holds the new state's smax only after a successful launch
  CUDA_TRY(cudaMemsetAsync(b->smax_slot, 0, 16, b->stream));
  cudaError_t e;
  int tx = 0, ty = 0;
  if (b->d.dtype == AMR_F32) {
    amr::StepParams<float> P = make_params<float>(b, dt, gamma, ch, alpha);
    if (mhd) amr::tile_shape_mhd_f32(P.n, &tx, &ty); else amr::tile_shape_hydro_f32(P.n, &tx, &ty);
    P.ntx = P.n / tx; P.nty = P.n / ty; P.ntz = 1; P.zc = P.n;
    e = mhd ? amr::launch_step_mhd_f32(P, limiter, riemann, b->stream)
            : amr::launch_step_hydro_f32(P, limiter, riemann, b->stream);
  } else {
    amr::StepParams<double> P = make_params<double>(b, dt, gamma, ch, alpha);
    if (mhd) amr::tile_shape_mhd_f64(P.n, &tx, &ty); else amr::tile_shape_hydro_f64(P.n, &tx, &ty);
    P.ntx = P.n / tx; P.nty = P.n / ty; P.ntz = 1; P.zc = P.n;
    e = mhd ? amr::launch_step_mhd_f64(P, limiter, riemann, b->stream)
            : amr::launch_step_hydro_f64(P, limiter, riemann, b->stream);
  }
  if (e != cudaSuccess) return fail(AMR_ECUDA, "step kernel launch: %s", cudaGetErrorString(e));
  b->cur = 1 - b->cur;
  b->smax_valid = true;
  b->smax_gamma = gamma;
  return AMR_OK;
}

}  // namespace

namespace amr {
int set_error(int code, const char* where, const char* what) { return fail(code, "%s: %s", where, what); }
}  // namespace amr

extern "C" {

const char* amr_last_error(void) { return g_err.c_str(); }

int amr_measure_fma_peak(int32_t dtype, void* dev_scratch, void* cuda_stream, double ms_target, double* tflops_out) {
  if (!dev_scratch || !tflops_out) return fail(AMR_EINVAL, "null argument");
  if (dtype != AMR_F32 && dtype != AMR_F64) return fail(AMR_EINVAL, "dtype must be AMR_F32 or AMR_F64");
  if (!(ms_target > 0) || ms_target > 1000) return fail(AMR_EINVAL, "ms_target must be in (0, 1000]");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return fail(AMR_ECUDA, "no CUDA device");
  const int grid = sms * 8;                      // 8 CTAs of 256 threads per SM: 16 warps per scheduler
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return fail(AMR_ECUDA, "cudaEventCreate");
  auto run = [&](int iters, float* ms) -> cudaError_t {
    cudaEventRecord(e0, s);
    cudaError_t e = amr::launch_fma_chain(dtype, dev_scratch, grid, iters, s);
    cudaEventRecord(e1, s);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
    return e;
  };
  float ms = 0;
  int iters = 256;
  cudaError_t e = run(iters, &ms);               // warm-up and calibration
  if (e == cudaSuccess) e = run(iters, &ms);
  if (e == cudaSuccess) {
    const double scale = ms_target / (ms > 1e-3 ? ms : 1e-3);
    iters = (int)std::min(1.0e7, std::max(64.0, iters * scale));
    e = run(iters, &ms);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (e != cudaSuccess) return fail(AMR_ECUDA, "fma chain: %s", cudaGetErrorString(e));
  const double flops = 2.0 * 64.0 * (double)iters * 256.0 * (double)grid;
  *tflops_out = flops / (ms * 1e-3) / 1e12;
  return AMR_OK;
}
const char* amr_version(void) { return "amr_godunov 0.1 (sm_100a; fused MUSCL-Hancock/HLLC/HLLD step, interiors-only SoA arena)"; }

size_t amr_patch_batch_bytes(const amr_batch_desc* desc) {
  std::string why;
  if (!desc_ok(desc, &why)) { fail(AMR_EINVAL, "%s", why.c_str()); return 0; }
  return make_layout(desc).total;
}

int amr_patch_batch_create(const amr_batch_desc* desc, void* dev_arena, size_t bytes, void* cuda_stream,
                           amr_patch_batch** out) {
  if (!out) return fail(AMR_EINVAL, "null out");
  *out = nullptr;
  std::string why;
  if (!desc_ok(desc, &why)) return fail(AMR_EINVAL, "%s", why.c_str());
  if (!dev_arena) return fail(AMR_EINVAL, "null device arena");
  if ((uintptr_t)dev_arena % ALIGN) return fail(AMR_EINVAL, "device arena must be %zu-byte aligned", ALIGN);
  const Layout L = make_layout(desc);
  if (bytes < L.total) return fail(AMR_EINVAL, "arena too small: %zu < %zu bytes", bytes, L.total);

  amr_patch_batch* b = new (std::nothrow) amr_patch_batch();
  static std::atomic<unsigned long long> next_serial{1};
  if (b) b->serial = next_serial.fetch_add(1);
  if (!b) return fail(AMR_ENOMEM, "out of host memory");
  b->d = *desc;
  b->d.origin = nullptr;
  const int np = desc->npatch, n = desc->n;
  const int nactive = desc->nactive > 0 ? desc->nactive : np;
  b->nactive = nactive;
  b->origin.assign((size_t)np * 3, 0);
  if (desc->self_periodic) {
    for (int a = 0; a < 3; ++a) b->d.domain_cells[a] = n;
    for (int a = 0; a < 6; ++a) b->d.bc[a] = AMR_BC_PERIODIC;
  } else {
    std::memcpy(b->origin.data(), desc->origin, (size_t)np * 3 * sizeof(int32_t));
  }
  // neighbour table (O0 rules (i) sibling copy with periodic wrap, (ii) outflow clamp)
  b->nbr_host.assign((size_t)np * 27, 0);
  b->needs_halo = false;
  if (desc->self_periodic) {
    for (int p = 0; p < np; ++p)
      for (int r = 0; r < 27; ++r) b->nbr_host[(size_t)p * 27 + r] = p;
    b->map.dims[0] = b->map.dims[1] = b->map.dims[2] = 1;
    b->map.idx.assign(1, 0);
  } else {
    PatchMap& m = b->map;
    for (int a = 0; a < 3; ++a) m.dims[a] = desc->domain_cells[a] / n;
    m.idx.assign((size_t)m.dims[0] * m.dims[1] * m.dims[2], -1);
    for (int p = 0; p < np; ++p) {
      const int32_t* o = &b->origin[3 * p];
      for (int a = 0; a < 3; ++a)
        if (o[a] < 0 || o[a] % n || o[a] + n > desc->domain_cells[a]) {
          delete b;
          return fail(AMR_EINVAL, "origin of patch %d is not a multiple of n inside the domain", p);
        }
      int& slot = m.idx[((size_t)(o[2] / n) * m.dims[1] + o[1] / n) * m.dims[0] + o[0] / n];
      if (slot >= 0) { delete b; return fail(AMR_EINVAL, "patches %d and %d coincide", slot, p); }
      slot = p;
    }
    for (int p = 0; p < np; ++p) {
      const int32_t* o = &b->origin[3 * p];
      const int pc[3] = {o[0] / n, o[1] / n, o[2] / n};
      for (int r = 0; r < 27; ++r) {
        const int rr[3] = {r % 3, (r / 3) % 3, r / 9};
        int q[3], mode = 0;
        for (int a = 0; a < 3; ++a) {
          q[a] = pc[a] + rr[a] - 1;
          if (q[a] < 0) {
            if (desc->bc[2 * a] == AMR_BC_PERIODIC) q[a] += m.dims[a]; else { q[a] = 0; mode |= 1 << a; }
          } else if (q[a] >= m.dims[a]) {
            if (desc->bc[2 * a + 1] == AMR_BC_PERIODIC) q[a] -= m.dims[a]; else { q[a] = m.dims[a] - 1; mode |= 1 << a; }
          }
        }
        const int src = m.at(q[0], q[1], q[2]);
        int e;
        if (src >= 0) e = src | (mode << amr::NBR_MODE_SHIFT);
        else if (p >= nactive) e = p;   // a read-only copy of a remote patch is never stepped: its halo is never gathered
        else if (desc->level > 0) { e = amr::NBR_FROM_HALO; b->needs_halo = true; }
        else { delete b; return fail(AMR_EINVAL, "root-level patch %d has no neighbour in region %d", p, r); }
        b->nbr_host[(size_t)p * 27 + r] = e;
      }
    }
  }
  b->stream = (cudaStream_t)cuda_stream;
  {
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, dev_arena) != cudaSuccess || pa.type != cudaMemoryTypeDevice) {
      cudaGetLastError();
      delete b;
      return fail(AMR_EINVAL, "dev_arena is not a device allocation");
    }
    b->device = pa.device;
  }
  DeviceGuard guard(b->device);
  b->arena = (char*)dev_arena;
  b->bytes = bytes;
  b->esz = desc->dtype == AMR_F64 ? 8 : 4;
  b->n3 = (size_t)n * n * n;
  const size_t M = n + 2 * desc->nghost;
  b->M3 = M * M * M;
  b->U[0] = b->arena + L.U[0];
  b->U[1] = b->arena + L.U[1];
  b->cur = 0;
  b->halo = desc->level > 0 ? b->arena + L.halo : nullptr;
  b->nbr_dev = (int*)(b->arena + L.nbr);
  b->fblk_of = (int*)(b->arena + L.fblk_of);
  b->fblk = nullptr;
  b->counters = (unsigned long long*)(b->arena + L.counters);
  b->smax_slot = b->arena + L.smax;
  b->partials = (double*)(b->arena + L.partials);
  b->halo_valid = false;
  b->smax_valid = false;
  b->smax_gamma = 0;
  b->link_up = b->link_down = nullptr;
  auto bail = [&](cudaError_t e, const char* what) {
    delete b;
    return fail(AMR_ECUDA, "%s: %s", what, cudaGetErrorString(e));
  };
  cudaError_t e = cudaMemcpyAsync(b->nbr_dev, b->nbr_host.data(), (size_t)np * 27 * sizeof(int), cudaMemcpyHostToDevice, b->stream);
  if (e != cudaSuccess) return bail(e, "upload of the neighbour table");
  e = cudaMemsetAsync(b->counters, 0, 4 * sizeof(unsigned long long), b->stream);
  if (e != cudaSuccess) return bail(e, "cudaMemsetAsync");
  e = cudaMemsetAsync(b->fblk_of, 0xff, (size_t)np * sizeof(int), b->stream);
  if (e != cudaSuccess) return bail(e, "cudaMemsetAsync");
  if (b->halo) {
    e = amr::launch_fill_nan(desc->dtype, b->halo, (size_t)desc->nfields * np * b->M3, b->stream);
    if (e != cudaSuccess) return bail(e, "halo initialisation");
  }
  e = cudaStreamSynchronize(b->stream);  // nbr_host stays alive, but report upload errors here
  if (e != cudaSuccess) return bail(e, "cudaStreamSynchronize");
  *out = b;
  return AMR_OK;
}

int amr_patch_batch_destroy(amr_patch_batch* b) {
  if (!b) return AMR_OK;
  DeviceGuard guard(b->device);
  if (b->link_up || b->link_down) return fail(AMR_ESTATE, "batch is still linked; call amr_link_destroy first");
  cudaStreamSynchronize(b->stream);
  delete b;
  return AMR_OK;
}

void* amr_patch_batch_state(amr_patch_batch* b, int which) {
  if (!b || which < 0 || which > 1) { fail(AMR_EINVAL, "bad arguments"); return nullptr; }
  return b->U[which == 0 ? b->cur : 1 - b->cur];
}

int amr_patch_batch_upload(amr_patch_batch* b, const void* host, int with_ghosts) {
  if (!b || !host) return fail(AMR_EINVAL, "null pointer");
  DeviceGuard guard(b->device);
  const int nf = b->d.nfields, np = b->d.npatch;
  const size_t state_bytes = (size_t)nf * np * b->n3 * b->esz;
  if (!with_ghosts) {
    CUDA_TRY(cudaMemcpyAsync(b->U[b->cur], host, state_bytes, cudaMemcpyHostToDevice, b->stream));
  } else {
    const size_t per_patch = (size_t)nf * b->M3 * b->esz;
    int chunk = (int)std::max<size_t>(1, std::min<size_t>((size_t)np, ((size_t)512 << 20) / per_patch));
    void* stage = nullptr;
    CUDA_TRY(cudaMallocAsync(&stage, (size_t)chunk * per_patch, b->stream));   // stream-ordered, returned below
    for (int p0 = 0; p0 < np; p0 += chunk) {
      const int npc = std::min(chunk, np - p0);
      for (int q = 0; q < nf; ++q) {
        cudaError_t e = cudaMemcpyAsync((char*)stage + (size_t)q * npc * b->M3 * b->esz,
                                        (const char*)host + ((size_t)q * np + p0) * b->M3 * b->esz,
                                        (size_t)npc * b->M3 * b->esz, cudaMemcpyHostToDevice, b->stream);
        if (e != cudaSuccess) { cudaFreeAsync(stage, b->stream); return fail(AMR_ECUDA, "upload: %s", cudaGetErrorString(e)); }
      }
      cudaError_t e = amr::launch_scatter_interior(b->d.dtype, stage, 1, nf, np, b->d.n, b->d.nghost, p0, npc,
                                                   b->U[b->cur], b->stream);
      if (e == cudaSuccess) e = cudaStreamSynchronize(b->stream);
      if (e != cudaSuccess) { cudaFreeAsync(stage, b->stream); return fail(AMR_ECUDA, "upload: %s", cudaGetErrorString(e)); }
    }
    cudaFreeAsync(stage, b->stream);
  }
  // both buffers hold the uploaded state, so that "previous state" is defined before the first step
  CUDA_TRY(cudaMemcpyAsync(b->U[1 - b->cur], b->U[b->cur], state_bytes, cudaMemcpyDeviceToDevice, b->stream));
  CUDA_TRY(cudaStreamSynchronize(b->stream));
  b->smax_valid = false;
  return AMR_OK;
}

int amr_patch_batch_download(amr_patch_batch* b, void* host, int with_ghosts) {
  if (!b || !host) return fail(AMR_EINVAL, "null pointer");
  DeviceGuard guard(b->device);
  const int nf = b->d.nfields, np = b->d.npatch;
  if (!with_ghosts) {
    CUDA_TRY(cudaMemcpyAsync(host, b->U[b->cur], (size_t)nf * np * b->n3 * b->esz, cudaMemcpyDeviceToHost, b->stream));
    CUDA_TRY(cudaStreamSynchronize(b->stream));
    return AMR_OK;
  }
  const size_t per_patch = (size_t)nf * b->M3 * b->esz;
  int chunk = (int)std::max<size_t>(1, std::min<size_t>((size_t)np, ((size_t)512 << 20) / per_patch));
  void* stage = nullptr;
  CUDA_TRY(cudaMallocAsync(&stage, (size_t)chunk * per_patch, b->stream));   // stream-ordered, returned below
  for (int p0 = 0; p0 < np; p0 += chunk) {
    const int npc = std::min(chunk, np - p0);
    cudaError_t e = amr::launch_gather_ghosted(b->d.dtype, b->U[b->cur], b->halo, b->nbr_dev, nf, np, b->d.n,
                                               b->d.nghost, p0, npc, stage, b->stream);
    for (int q = 0; q < nf && e == cudaSuccess; ++q)
      e = cudaMemcpyAsync((char*)host + ((size_t)q * np + p0) * b->M3 * b->esz,
                          (const char*)stage + (size_t)q * npc * b->M3 * b->esz, (size_t)npc * b->M3 * b->esz,
                          cudaMemcpyDeviceToHost, b->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(b->stream);
    if (e != cudaSuccess) { cudaFreeAsync(stage, b->stream); return fail(AMR_ECUDA, "download: %s", cudaGetErrorString(e)); }
  }
  cudaFreeAsync(stage, b->stream);
  return AMR_OK;
}

int amr_fill_ghosts(amr_patch_batch* b) {
  if (!b) return fail(AMR_EINVAL, "null batch");
  return AMR_OK;
}

int amr_cfl_dt(amr_patch_batch* b, double gamma, double cfl, int mhd, double* dt_out, double* smax_out) {
  if (!b) return fail(AMR_EINVAL, "null batch");
  DeviceGuard guard(b->device);
  if ((mhd != 0) != (b->d.nfields == 9)) return fail(AMR_EINVAL, "mhd flag does not match nfields = %d", b->d.nfields);
  if (!std::isfinite(gamma) || !(gamma > 1)) return fail(AMR_EINVAL, "gamma must be finite and > 1");
  if (!(cfl > 0) || !std::isfinite(cfl)) return fail(AMR_EINVAL, "cfl must be finite and > 0");
  if (!(b->smax_valid && b->smax_gamma == gamma)) {
    CUDA_TRY(cudaMemsetAsync(b->smax_slot, 0, 16, b->stream));
    cudaError_t e = amr::launch_smax(b->d.dtype, b->U[b->cur], b->d.nfields, b->d.npatch, b->nactive, b->d.n, gamma, b->smax_slot, b->stream);
    if (e != cudaSuccess) return fail(AMR_ECUDA, "smax kernel launch: %s", cudaGetErrorString(e));
    b->smax_valid = true;
    b->smax_gamma = gamma;
  }
  double smax;
  if (b->d.dtype == AMR_F32) {
    float v = 0;
    CUDA_TRY(cudaMemcpyAsync(&v, b->smax_slot, 4, cudaMemcpyDeviceToHost, b->stream));
    CUDA_TRY(cudaStreamSynchronize(b->stream));
    smax = v;
  } else {
    CUDA_TRY(cudaMemcpyAsync(&smax, b->smax_slot, 8, cudaMemcpyDeviceToHost, b->stream));
    CUDA_TRY(cudaStreamSynchronize(b->stream));
  }
  if (smax_out) *smax_out = smax;
  if (dt_out) *dt_out = cfl * b->d.dx / smax;
  return AMR_OK;
}

int amr_hydro_step(amr_patch_batch* b, double dt, double gamma, int limiter, int riemann) {
  return do_step(b, false, dt, gamma, limiter, riemann, 0.0, 0.0);
}

int amr_mhd_step(amr_patch_batch* b, double dt, double gamma, int limiter, int riemann, double ch, double alpha) {
  return do_step(b, true, dt, gamma, limiter, riemann, ch, alpha);
}

int amr_patch_batch_export(amr_patch_batch* b, const int32_t* dev_pairs, int32_t count, void* dev_packed) {
  if (!b || (count > 0 && (!dev_pairs || !dev_packed))) return fail(AMR_EINVAL, "null pointer");
  if (count < 0) return fail(AMR_EINVAL, "count < 0");
  DeviceGuard guard(b->device);
  cudaError_t e = amr::launch_copy_patches(b->d.dtype, dev_packed, (size_t)count * b->n3, b->U[b->cur],
                                           (size_t)b->d.npatch * b->n3, dev_pairs, count, b->d.nfields, b->d.n, b->stream);
  if (e != cudaSuccess) return fail(AMR_ECUDA, "export kernel launch: %s", cudaGetErrorString(e));
  return AMR_OK;
}

int amr_patch_batch_import(amr_patch_batch* b, const int32_t* dev_pairs, int32_t count, const void* dev_packed) {
  if (!b || (count > 0 && (!dev_pairs || !dev_packed))) return fail(AMR_EINVAL, "null pointer");
  if (count < 0) return fail(AMR_EINVAL, "count < 0");
  DeviceGuard guard(b->device);
  cudaError_t e = amr::launch_copy_patches_in(b->d.dtype, b->U[b->cur], (size_t)b->d.npatch * b->n3, dev_packed,
                                              (size_t)count * b->n3, dev_pairs, count, b->d.nfields, b->d.n, b->stream);
  if (e != cudaSuccess) return fail(AMR_ECUDA, "import kernel launch: %s", cudaGetErrorString(e));
  return AMR_OK;
}

int amr_hydro_sweep_ppm(amr_patch_batch* b, double dt, double gamma, int riemann, int dir) {
  if (!b) return fail(AMR_EINVAL, "null batch");
  DeviceGuard guard(b->device);
  if (b->d.nfields != 5) return fail(AMR_EINVAL, "PPM is the hydro scheme: the batch has %d fields", b->d.nfields);
  if (!(dt > 0) || !std::isfinite(dt)) return fail(AMR_EINVAL, "dt must be finite and > 0");
  if (!std::isfinite(gamma) || !(gamma > 1)) return fail(AMR_EINVAL, "gamma must be finite and > 1");
  if (riemann != AMR_RS_HLL && riemann != AMR_RS_HLLC) return fail(AMR_EINVAL, "PPM sweep takes HLL or HLLC");
  if (dir < 0 || dir > 2) return fail(AMR_EINVAL, "dir must be 0 (x), 1 (y) or 2 (z)");
  if (b->d.nghost < 3) return fail(AMR_EINVAL, "PPM needs nghost >= 3 (reading A11)");
  if (b->d.n > 64) return fail(AMR_EINVAL, "PPM sweeps are instantiated for n <= 64");
  if (b->link_up || b->link_down)
    return fail(AMR_ESTATE, "PPM sweeps record no flux registers: the batch must not be linked");
  if (b->needs_halo && !b->halo_valid)
    return fail(AMR_ESTATE, "level-%d batch has coarse-fine halo regions but its halo was never filled", b->d.level);
  cudaError_t e;
  if (b->d.dtype == AMR_F32) {
    amr::ppm::SweepParams<float> P;
    P.Uin = (const float*)b->U[b->cur]; P.Uout = (float*)b->U[1 - b->cur]; P.halo = (const float*)b->halo;
    P.nbr = b->nbr_dev; P.counters = b->counters; P.np = b->d.npatch; P.np_active = b->nactive; P.n = b->d.n; P.g = b->d.nghost;
    P.dtdx = (float)(dt / b->d.dx); P.gamma = (float)gamma; P.gm1 = (float)(gamma - 1); P.igm1 = (float)(1.0 / (gamma - 1));
    e = amr::launch_ppm_sweep_f32(P, riemann, dir, b->stream);
  } else {
    amr::ppm::SweepParams<double> P;
    P.Uin = (const double*)b->U[b->cur]; P.Uout = (double*)b->U[1 - b->cur]; P.halo = (const double*)b->halo;
    P.nbr = b->nbr_dev; P.counters = b->counters; P.np = b->d.npatch; P.np_active = b->nactive; P.n = b->d.n; P.g = b->d.nghost;
    P.dtdx = dt / b->d.dx; P.gamma = gamma; P.gm1 = gamma - 1; P.igm1 = 1.0 / (gamma - 1);
    e = amr::launch_ppm_sweep_f64(P, riemann, dir, b->stream);
  }
  if (e != cudaSuccess) return fail(AMR_ECUDA, "PPM sweep kernel launch: %s", cudaGetErrorString(e));
  b->cur = 1 - b->cur;
  b->smax_valid = false;   // the sweeps fuse no CFL reduction: amr_cfl_dt runs the standalone one
  return AMR_OK;
}

int amr_hydro_step_ppm(amr_patch_batch* b, double dt, double gamma, int riemann, int order) {
  if (order != 0 && order != 1) return fail(AMR_EINVAL, "order must be 0 (x-y-z) or 1 (z-y-x)");
  for (int i = 0; i < 3; ++i) {
    const int rc = amr_hydro_sweep_ppm(b, dt, gamma, riemann, order ? 2 - i : i);
    if (rc != AMR_OK) return rc;
  }
  return AMR_OK;
}

int amr_conserved_totals(amr_patch_batch* b, double* totals) {
  if (!b || !totals) return fail(AMR_EINVAL, "null pointer");
  DeviceGuard guard(b->device);
  const int nf = b->d.nfields;
  cudaError_t e = amr::launch_totals(b->d.dtype, b->U[b->cur], nf, b->d.npatch, b->nactive, b->d.n, b->partials, b->stream);
  if (e != cudaSuccess) return fail(AMR_ECUDA, "totals kernel launch: %s", cudaGetErrorString(e));
  std::vector<double> h((size_t)nf * amr::TOTALS_BLOCKS);
  CUDA_TRY(cudaMemcpyAsync(h.data(), b->partials, h.size() * sizeof(double), cudaMemcpyDeviceToHost, b->stream));
  CUDA_TRY(cudaStreamSynchronize(b->stream));
  for (int q = 0; q < nf; ++q) {
    long double s = 0;
    for (int k = 0; k < amr::TOTALS_BLOCKS; ++k) s += (long double)h[(size_t)q * amr::TOTALS_BLOCKS + k];
    totals[q] = (double)s;
  }
  return AMR_OK;
}

int amr_step_counters(amr_patch_batch* b, long long* counters, int reset) {
  if (!b || !counters) return fail(AMR_EINVAL, "null pointer");
  DeviceGuard guard(b->device);
  CUDA_TRY(cudaMemcpyAsync(counters, b->counters, 4 * sizeof(long long), cudaMemcpyDeviceToHost, b->stream));
  if (reset) CUDA_TRY(cudaMemsetAsync(b->counters, 0, 4 * sizeof(long long), b->stream));
  CUDA_TRY(cudaStreamSynchronize(b->stream));
  return AMR_OK;
}

// ---- two-level -------------------------------------------------------------------------------------

size_t amr_link_bytes(const amr_patch_batch* coarse, const amr_patch_batch* fine, int ratio) {
  if (check_link_args(coarse, fine, ratio) != AMR_OK) return 0;
  LinkHost H;
  H.identity_c = coarse->link_up != nullptr;
  if (build_link(coarse, fine, H) != AMR_OK) return 0;
  const size_t total = make_link_layout(coarse, fine, H).total;
  g_link_cache.c = coarse->serial;
  g_link_cache.f = fine->serial;
  g_link_cache.identity_c = H.identity_c;
  g_link_cache.H = std::move(H);
  return total;
}

int amr_link_levels(amr_patch_batch* coarse, amr_patch_batch* fine, int ratio, void* dev_ws, size_t bytes,
                    amr_level_link** out) {
  if (!out) return fail(AMR_EINVAL, "null out");
  *out = nullptr;
  int rc = check_link_args(coarse, fine, ratio);
  if (rc != AMR_OK) return rc;
  if (coarse->link_down) return fail(AMR_ESTATE, "the coarse batch already has a child level");
  DeviceGuard guard(coarse->device);
  if (fine->link_up) return fail(AMR_ESTATE, "the fine batch already has a parent level");
  if (fine->link_down) return fail(AMR_ESTATE, "link a hierarchy from the root upwards: the fine batch already has a child level");
  if (!dev_ws || (uintptr_t)dev_ws % ALIGN) return fail(AMR_EINVAL, "workspace must be a %zu-byte aligned device pointer", ALIGN);
  LinkHost H;
  // a middle level records every patch's fluxes already (it is the fine side of its parent link): its role as
  // the coarse side of this link reads the same per-patch blocks (the two sets of faces are disjoint under
  // proper nesting, and amr_flux_clear of this link zeroes only its own faces there)
  H.identity_c = coarse->link_up != nullptr;
  if (g_link_cache.c == coarse->serial && g_link_cache.f == fine->serial && g_link_cache.identity_c == H.identity_c) {
    H = std::move(g_link_cache.H);
    rc = AMR_OK;
  } else {
    rc = build_link(coarse, fine, H);
  }
  g_link_cache = LinkCache();
  if (rc != AMR_OK) return rc;
  const LinkLayout L = make_link_layout(coarse, fine, H);
  if (bytes < L.total) return fail(AMR_EINVAL, "workspace too small: %zu < %zu bytes", bytes, L.total);
  amr_level_link* l = new (std::nothrow) amr_level_link();
  if (!l) return fail(AMR_ENOMEM, "out of host memory");
  l->c = coarse; l->f = fine; l->ws = (char*)dev_ws; l->bytes = bytes;
  l->forg = (int*)(l->ws + L.forg);
  l->cmap = (int*)(l->ws + L.cmap);
  l->fmap = (int*)(l->ws + L.fmap);
  l->cblk = (int*)(l->ws + L.cblk);
  l->ncblk = (int)(H.cblk.size() / 4);
  l->rlist = (int*)(l->ws + L.rlist);
  l->nrlist = 0;
  l->fblk_c = l->ws + L.fblk_c; l->fblk_f = l->ws + L.fblk_f;
  l->fblk_c_bytes = L.fblk_c_bytes; l->fblk_f_bytes = L.fblk_f_bytes;
  l->nblk_c = H.nblk_c;
  l->shared_c = H.identity_c;
  if (l->shared_c) l->fblk_c = coarse->fblk;
  cudaStream_t s = coarse->stream;
  auto h2d = [&](void* dst, const void* src, size_t nb) {
    return nb ? cudaMemcpyAsync(dst, src, nb, cudaMemcpyHostToDevice, s) : cudaSuccess;
  };
  cudaError_t e = h2d(l->forg, fine->origin.data(), fine->origin.size() * sizeof(int));
  if (e == cudaSuccess) e = h2d(l->cmap, coarse->map.idx.data(), coarse->map.idx.size() * sizeof(int));
  if (e == cudaSuccess) e = h2d(l->fmap, fine->map.idx.data(), fine->map.idx.size() * sizeof(int));
  if (e == cudaSuccess) e = h2d(l->cblk, H.cblk.data(), H.cblk.size() * sizeof(int));
  if (e == cudaSuccess && !l->shared_c) e = h2d(coarse->fblk_of, H.fblk_of_c.data(), H.fblk_of_c.size() * sizeof(int));
  std::vector<int> idf(fine->d.npatch);
  for (int p = 0; p < fine->d.npatch; ++p) idf[p] = p;
  if (e == cudaSuccess) e = h2d(fine->fblk_of, idf.data(), idf.size() * sizeof(int));
  if (e == cudaSuccess && !l->shared_c) e = cudaMemsetAsync(l->fblk_c, 0, L.fblk_c_bytes + 8, s);
  if (e == cudaSuccess) e = cudaMemsetAsync(l->fblk_f, 0, L.fblk_f_bytes + 8, s);
  // the reflux list: found on the device from the tables just uploaded (same stream)
  int nr = 0;
  if (e == cudaSuccess)
    e = amr::launch_reflux_find(coarse->d.nfields, coarse->d.n, l->shared_c ? 1 : 0, coarse->d.domain_cells, fine->map.dims,
                                coarse->d.bc, l->cblk, l->ncblk, l->fmap, l->rlist, (int*)(l->ws + L.rcount), L.rcap, s);
  if (e == cudaSuccess) e = cudaMemcpyAsync(&nr, l->ws + L.rcount, sizeof(int), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) { delete l; return fail(AMR_ECUDA, "link upload: %s", cudaGetErrorString(e)); }
  if (nr > L.rcap) { delete l; return fail(AMR_EINVAL, "reflux list overflow: %d cells > %d (inconsistent patch maps)", nr, L.rcap); }
  l->nrlist = nr;
  if (!l->shared_c) coarse->fblk = l->nblk_c ? l->fblk_c : nullptr;
  fine->fblk = l->fblk_f;
  coarse->link_down = fine->link_up = l;
  *out = l;
  return AMR_OK;
}

int amr_link_destroy(amr_level_link* l) {
  if (!l) return AMR_OK;
  DeviceGuard guard(l->f->device);
  if (l->f->link_down) return fail(AMR_ESTATE, "destroy the finer link first (it records into this link's fine blocks)");
  cudaStreamSynchronize(l->c->stream);
  cudaStreamSynchronize(l->f->stream);
  if (!l->shared_c) l->c->fblk = nullptr;
  l->f->fblk = nullptr;
  l->c->link_down = nullptr; l->f->link_up = nullptr;
  delete l;
  return AMR_OK;
}

int amr_prolong_ghosts(amr_level_link* l, double theta) {
  if (!l) return fail(AMR_EINVAL, "null link");
  DeviceGuard guard(l->f->device);
  if (!(theta >= 0 && theta <= 1)) return fail(AMR_EINVAL, "theta must be in [0,1]");
  amr_patch_batch *c = l->c, *f = l->f;
  cudaError_t e = amr::launch_prolong_halo(f->d.dtype, f->halo, (size_t)f->d.npatch * f->M3, f->d.nfields, f->d.n, f->d.nghost,
                                           f->d.npatch, f->d.domain_cells, c->d.domain_cells, c->map.dims, f->d.bc, l->forg,
                                           f->nbr_dev, l->cmap, c->U[1 - c->cur], c->U[c->cur], (size_t)c->d.npatch * c->n3,
                                           theta, f->stream);
  if (e != cudaSuccess) return fail(AMR_ECUDA, "prolong kernel launch: %s", cudaGetErrorString(e));
  f->halo_valid = true;
  return AMR_OK;
}

int amr_flux_clear(amr_level_link* l) {
  if (!l) return fail(AMR_EINVAL, "null link");
  DeviceGuard guard(l->f->device);
  if (l->shared_c) {
    cudaError_t e = amr::launch_zero_faces(l->c->d.dtype, l->fblk_c, l->c->d.nfields, l->c->d.n, 1, l->c->d.domain_cells,
                                           l->f->map.dims, l->c->d.bc, l->cblk, l->rlist, l->nrlist, l->c->stream);
    if (e != cudaSuccess) return fail(AMR_ECUDA, "flux clear kernel launch: %s", cudaGetErrorString(e));
  } else if (l->fblk_c_bytes) {
    CUDA_TRY(cudaMemsetAsync(l->fblk_c, 0, l->fblk_c_bytes, l->c->stream));
  }
  if (l->fblk_f_bytes) CUDA_TRY(cudaMemsetAsync(l->fblk_f, 0, l->fblk_f_bytes, l->f->stream));
  return AMR_OK;
}

int amr_restrict(amr_level_link* l) {
  if (!l) return fail(AMR_EINVAL, "null link");
  DeviceGuard guard(l->f->device);
  amr_patch_batch *c = l->c, *f = l->f;
  cudaError_t e = amr::launch_restrict(f->d.dtype, f->U[f->cur], (size_t)f->d.npatch * f->n3, f->d.nfields, f->d.n, f->d.npatch,
                                       c->d.domain_cells, c->map.dims, c->d.bc, l->forg, l->cmap, c->U[c->cur],
                                       (size_t)c->d.npatch * c->n3, c->stream);
  if (e != cudaSuccess) return fail(AMR_ECUDA, "restrict kernel launch: %s", cudaGetErrorString(e));
  c->smax_valid = false;
  return AMR_OK;
}

int amr_reflux(amr_level_link* l, double dt_coarse) {
  if (!l) return fail(AMR_EINVAL, "null link");
  DeviceGuard guard(l->f->device);
  if (!(dt_coarse > 0) || !std::isfinite(dt_coarse)) return fail(AMR_EINVAL, "dt_coarse must be finite and > 0");
  amr_patch_batch* c = l->c;
  cudaError_t e = amr::launch_reflux(c->d.dtype, c->U[c->cur], (size_t)c->d.npatch * c->n3, c->d.nfields, c->d.n, l->shared_c ? 1 : 0,
                                     c->d.domain_cells, l->f->map.dims, c->d.bc, l->cblk, l->rlist, l->nrlist, l->fmap, l->forg,
                                     l->fblk_c, l->fblk_f, dt_coarse / c->d.dx, c->stream);
  if (e != cudaSuccess) return fail(AMR_ECUDA, "reflux kernel launch: %s", cudaGetErrorString(e));
  c->smax_valid = false;
  return AMR_OK;
}

}  // extern "C"

// ---- L-level hierarchy ---------------------------------------------------------------

namespace {

int check_hierarchy(amr_patch_batch* const* levels, amr_level_link* const* links, int nlevels) {
  if (!levels || nlevels < 1 || nlevels > 30) return fail(AMR_EINVAL, "levels must hold 1..30 batches");
  for (int l = 0; l < nlevels; ++l)
    if (!levels[l]) return fail(AMR_EINVAL, "null batch at level %d", l);
  if (nlevels > 1 && !links) return fail(AMR_EINVAL, "null links");
  for (int l = 0; l + 1 < nlevels; ++l)
    if (!links[l] || links[l]->c != levels[l] || links[l]->f != levels[l + 1])
      return fail(AMR_EINVAL, "links[%d] must tie levels[%d] (coarse) to levels[%d] (fine)", l, l, l + 1);
  return AMR_OK;
}

struct CycleArgs {
  amr_patch_batch* const* levels;
  amr_level_link* const* links;
  int nlevels, mhd, limiter, riemann, do_reflux;
  double gamma, ch, alpha;
  cudaEvent_t* ev;   // one event per level (nullptr: every level on the caller's stream, no overlap)
};

// `waiter` continues after everything enqueued on `producer` so far (no-op for one stream)
int stream_after(cudaStream_t waiter, cudaStream_t producer, cudaEvent_t ev) {
  if (waiter == producer) return AMR_OK;
  CUDA_TRY(cudaEventRecord(ev, producer));
  CUDA_TRY(cudaStreamWaitEvent(waiter, ev, 0));
  return AMR_OK;
}

// O8 at theta = 0 from the coarse level's CURRENT state, i.e. before its step is enqueued (the same values
// amr_prolong_ghosts(l, 0) reads after it): lets the fine level's first substep run beside the coarse step
int prolong_from_current(amr_level_link* l) {
  amr_patch_batch *c = l->c, *f = l->f;
  cudaError_t e = amr::launch_prolong_halo(f->d.dtype, f->halo, (size_t)f->d.npatch * f->M3, f->d.nfields, f->d.n, f->d.nghost,
                                           f->d.npatch, f->d.domain_cells, c->d.domain_cells, c->map.dims, f->d.bc, l->forg,
                                           f->nbr_dev, l->cmap, c->U[c->cur], c->U[c->cur], (size_t)c->d.npatch * c->n3, 0.0,
                                           f->stream);
  if (e != cudaSuccess) return fail(AMR_ECUDA, "prolong kernel launch: %s", cudaGetErrorString(e));
  f->halo_valid = true;
  return AMR_OK;
}

// advance(l, dt) of oracle.api.hierarchy_step.  Same operators on the same data; the only freedom taken is
// WHEN they are enqueued: the theta = 0 prolongation needs the coarse level's old state only, so it and the
// fine level's first substep (and, recursively, its children's) go to the fine level's stream before the coarse
// step goes to the coarse level's - a level launch of 0.5-3 waves leaves SMs idle that the other levels' CTAs
// fill (profiles/r1g).  Everything that crosses levels is ordered by events.
int advance_level(const CycleArgs& A, int l, double dt) {
  const bool has_child = l + 1 < A.nlevels;
  amr_patch_batch* b = A.levels[l];
  int rc;
  if (has_child) {
    amr_level_link* lk = A.links[l];
    // the fine stream first catches up with this level's: its current state is complete, and the previous
    // reflux of this link (which read the fine flux blocks on this level's stream) is over before they are cleared
    if (A.ev && (rc = stream_after(lk->f->stream, b->stream, A.ev[l])) != AMR_OK) return rc;
    if ((rc = amr_flux_clear(lk)) != AMR_OK) return rc;
    if ((rc = prolong_from_current(lk)) != AMR_OK) return rc;
  }
  rc = A.mhd ? amr_mhd_step(b, dt, A.gamma, A.limiter, A.riemann, A.ch, A.alpha)
             : amr_hydro_step(b, dt, A.gamma, A.limiter, A.riemann);
  if (rc != AMR_OK || !has_child) return rc;
  amr_level_link* lk = A.links[l];
  if ((rc = advance_level(A, l + 1, 0.5 * dt)) != AMR_OK) return rc;
  if (A.ev && (rc = stream_after(lk->f->stream, b->stream, A.ev[l])) != AMR_OK) return rc;   // the coarse step is done
  if ((rc = amr_prolong_ghosts(lk, 0.5)) != AMR_OK) return rc;
  if ((rc = advance_level(A, l + 1, 0.5 * dt)) != AMR_OK) return rc;
  if (A.ev && (rc = stream_after(b->stream, lk->f->stream, A.ev[l])) != AMR_OK) return rc;   // the fine level caught up
  if ((rc = amr_restrict(lk)) != AMR_OK) return rc;
  if (A.do_reflux && (rc = amr_reflux(lk, dt)) != AMR_OK) return rc;
  return AMR_OK;
}

// per-level streams and events of amr_hierarchy_step, created on first use and kept for the life of the thread
struct LevelStreams {
  std::vector<cudaStream_t> s;
  std::vector<cudaEvent_t> ev;
  cudaEvent_t fork = nullptr;
  int ensure(int n) {
    if (!fork) CUDA_TRY(cudaEventCreateWithFlags(&fork, cudaEventDisableTiming));
    while ((int)s.size() < n) {
      cudaStream_t st;
      cudaEvent_t e;
      CUDA_TRY(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
      CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
      s.push_back(st);
      ev.push_back(e);
    }
    return AMR_OK;
  }
};
thread_local LevelStreams g_level_streams;

}  // namespace

extern "C" {

int amr_hierarchy_cfl_dt(amr_patch_batch* const* levels, int nlevels, double gamma, double cfl, int mhd,
                         double* dt0_out, double* smax_out) {
  if (!levels || nlevels < 1 || nlevels > 30) return fail(AMR_EINVAL, "levels must hold 1..30 batches");
  if (!std::isfinite(gamma) || !(gamma > 1)) return fail(AMR_EINVAL, "gamma must be finite and > 1");
  if (!(cfl > 0) || !std::isfinite(cfl)) return fail(AMR_EINVAL, "cfl must be finite and > 0");
  // every level's smax kernel (where the fused value is stale) and 8-byte read are enqueued first, into pinned
  // host memory, then ONE synchronisation per distinct stream - not one round trip per level
  if (!levels[0]) return fail(AMR_EINVAL, "null batch at level 0");
  DeviceGuard guard(levels[0]->device);
  thread_local double* pinned = nullptr;
  if (!pinned) CUDA_TRY(cudaHostAlloc((void**)&pinned, 32 * sizeof(double), cudaHostAllocDefault));
  for (int l = 0; l < nlevels; ++l) {
    amr_patch_batch* b = levels[l];
    if (!b) return fail(AMR_EINVAL, "null batch at level %d", l);
    if ((mhd != 0) != (b->d.nfields == 9)) return fail(AMR_EINVAL, "mhd flag does not match nfields = %d", b->d.nfields);
    if (!(b->smax_valid && b->smax_gamma == gamma)) {
      CUDA_TRY(cudaMemsetAsync(b->smax_slot, 0, 16, b->stream));
      cudaError_t e = amr::launch_smax(b->d.dtype, b->U[b->cur], b->d.nfields, b->d.npatch, b->nactive, b->d.n, gamma, b->smax_slot, b->stream);
      if (e != cudaSuccess) return fail(AMR_ECUDA, "smax kernel launch: %s", cudaGetErrorString(e));
      b->smax_valid = true;
      b->smax_gamma = gamma;
    }
    pinned[l] = 0;
    CUDA_TRY(cudaMemcpyAsync(&pinned[l], b->smax_slot, b->d.dtype == AMR_F32 ? 4 : 8, cudaMemcpyDeviceToHost, b->stream));
  }
  for (int l = 0; l < nlevels; ++l)
    if (l == 0 || levels[l]->stream != levels[l - 1]->stream) CUDA_TRY(cudaStreamSynchronize(levels[l]->stream));
  double sm = 0;
  for (int l = 0; l < nlevels; ++l) {
    double sm_l;
    if (levels[l]->d.dtype == AMR_F32) { float v; std::memcpy(&v, &pinned[l], 4); sm_l = v; }
    else sm_l = pinned[l];
    sm = sm_l > sm ? sm_l : sm;
  }
  if (!(sm > 0) || !std::isfinite(sm)) return fail(AMR_ESTATE, "maximum signal speed over the levels is not finite and > 0");
  if (dt0_out) *dt0_out = cfl * levels[0]->d.dx / sm;
  if (smax_out) *smax_out = sm;
  return AMR_OK;
}

int amr_hierarchy_step(amr_patch_batch* const* levels, amr_level_link* const* links, int nlevels, int mhd, double dt0,
                       double gamma, int limiter, int riemann, double ch, double alpha, int do_reflux) {
  int rc = check_hierarchy(levels, links, nlevels);
  if (rc != AMR_OK) return rc;
  if (!(dt0 > 0) || !std::isfinite(dt0)) return fail(AMR_EINVAL, "dt0 must be finite and > 0");
  DeviceGuard guard(levels[0]->device);
  CycleArgs A{levels, links, nlevels, mhd, limiter, riemann, do_reflux, gamma, ch, alpha, nullptr};
  const char* env = std::getenv("AMR_HIERARCHY_OVERLAP");
  const bool overlap = nlevels > 1 && !(env && env[0] == '0');
  if (!overlap) return advance_level(A, 0, dt0);
  // level l > 0 runs on its own stream for the duration of this call (level 0 stays on the caller's)
  LevelStreams& LS = g_level_streams;
  if ((rc = LS.ensure(nlevels)) != AMR_OK) return rc;
  cudaStream_t caller = levels[0]->stream;
  for (int l = 1; l < nlevels; ++l)
    if (levels[l]->stream != caller) return fail(AMR_EINVAL, "all levels must have been created on one stream");
  CUDA_TRY(cudaEventRecord(LS.fork, caller));
  for (int l = 1; l < nlevels; ++l) {
    CUDA_TRY(cudaStreamWaitEvent(LS.s[l], LS.fork, 0));
    levels[l]->stream = LS.s[l];
  }
  A.ev = LS.ev.data();
  rc = advance_level(A, 0, dt0);
  cudaError_t e = cudaSuccess;
  for (int l = 1; l < nlevels; ++l) {   // join: the caller's stream continues after every level
    levels[l]->stream = caller;
    if (e == cudaSuccess) e = cudaEventRecord(LS.ev[l], LS.s[l]);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(caller, LS.ev[l], 0);
  }
  if (rc == AMR_OK && e != cudaSuccess) return fail(AMR_ECUDA, "stream join: %s", cudaGetErrorString(e));
  return rc;
}

}  // extern "C"

// ---- regridding between steps -----------------------------------------------------------

namespace {

// flat interior index of coarse cell C (level index space, wrapped / clamped by the level's boundary
// conditions) in the coarse batch; false if no patch of the batch holds it
bool coarse_cell_flat(const amr_patch_batch* c, int Cx, int Cy, int Cz, long long* out) {
  const int n = c->d.n;
  const int* domc = c->d.domain_cells;
  int C[3] = {Cx, Cy, Cz};
  for (int a = 0; a < 3; ++a) {
    if (C[a] < 0) C[a] = (c->d.bc[2 * a] == AMR_BC_PERIODIC) ? C[a] + domc[a] : 0;
    else if (C[a] >= domc[a]) C[a] = (c->d.bc[2 * a + 1] == AMR_BC_PERIODIC) ? C[a] - domc[a] : domc[a] - 1;
  }
  const int pc = c->map.at(C[0] / n, C[1] / n, C[2] / n);
  if (pc < 0) return false;
  const int* oc = &c->origin[3 * pc];
  *out = (long long)pc * (long long)c->n3 + ((long long)(C[2] - oc[2]) * n + (C[1] - oc[1])) * n + (C[0] - oc[0]);
  return true;
}

struct RegridHost {
  std::vector<int> pairs;       // (new, old) per kept patch
  std::vector<int> born;        // (new patch index, fine origin x, y, z) per new-born patch
};

struct RegridLayout { size_t pairs, born, cmap, total; };

int check_regrid_args(const amr_patch_batch* nw, const amr_patch_batch* old, const amr_patch_batch* c) {
  if (!nw || !c) return fail(AMR_EINVAL, "null batch");
  int rc = check_link_args(c, nw, 2);
  if (rc != AMR_OK) return rc;
  if (old && (old->d.n != nw->d.n || old->d.nfields != nw->d.nfields || old->d.dtype != nw->d.dtype ||
              old->d.level != nw->d.level))
    return fail(AMR_EINVAL, "old and new fine batches must agree in n, nfields, dtype, level");
  if (old)
    for (int a = 0; a < 3; ++a)
      if (old->d.domain_cells[a] != nw->d.domain_cells[a]) return fail(AMR_EINVAL, "old and new fine batches must share the index space");
  return AMR_OK;
}

// The prolongation of a new-born patch resolves its parents in the kernel (prolong_patches_kernel); what the host
// owes is the nesting check.  The parent block of a patch lies inside one coarse patch (origins are multiples of n,
// the block spans n/2), so the 7-point stencils of all its cells exist iff that patch and, along each axis, the
// coarse patch holding the cell one beyond the block's low and high face (wrapped / clamped) exist.
int build_regrid(const amr_patch_batch* nw, const amr_patch_batch* old, const amr_patch_batch* c, RegridHost& H) {
  const int n = nw->d.n, h = n / 2;
  long long flat;
  for (int p = 0; p < nw->d.npatch; ++p) {
    const int* o = &nw->origin[3 * p];
    const int po = old ? old->map.at(o[0] / n, o[1] / n, o[2] / n) : -1;
    if (po >= 0) { H.pairs.push_back(p); H.pairs.push_back(po); continue; }
    const int C[3] = {o[0] / 2, o[1] / 2, o[2] / 2};
    bool ok = coarse_cell_flat(c, C[0], C[1], C[2], &flat);
    for (int a = 0; a < 3 && ok; ++a) {
      int Cm[3] = {C[0], C[1], C[2]}, Cp[3] = {C[0], C[1], C[2]};
      Cm[a] -= 1;
      Cp[a] += h;
      ok = coarse_cell_flat(c, Cm[0], Cm[1], Cm[2], &flat) && coarse_cell_flat(c, Cp[0], Cp[1], Cp[2], &flat);
    }
    if (!ok) return fail(AMR_EINVAL, "new patch %d is not properly nested in the coarse level (a parent cell or its stencil is missing)", p);
    H.born.push_back(p);
    for (int a = 0; a < 3; ++a) H.born.push_back(o[a]);
  }
  return AMR_OK;
}

RegridLayout make_regrid_layout(const RegridHost& H, const amr_patch_batch* c) {
  RegridLayout L;
  size_t off = 0;
  L.pairs = off; off += up(H.pairs.size() * sizeof(int) + 8);
  L.born = off; off += up(H.born.size() * sizeof(int) + 8);
  L.cmap = off; off += up(c->map.idx.size() * sizeof(int) + 8);
  L.total = off;
  return L;
}

}  // namespace

extern "C" {

int amr_flag_blocks(amr_patch_batch* b, int field, double threshold, unsigned char* host_flags) {
  if (!b || !host_flags) return fail(AMR_EINVAL, "null pointer");
  DeviceGuard guard(b->device);
  if (field < 0 || field >= b->d.nfields) return fail(AMR_EINVAL, "field must be in [0, nfields)");
  if (b->d.n % 2) return fail(AMR_EINVAL, "n must be even");
  const size_t nflag = (size_t)b->d.npatch * 8;
  unsigned char* dflags = nullptr;
  CUDA_TRY(cudaMallocAsync((void**)&dflags, nflag, b->stream));
  const char* U = (const char*)b->U[b->cur] + (size_t)field * b->d.npatch * b->n3 * b->esz;
  cudaError_t e = amr::launch_flag_blocks(b->d.dtype, U, b->d.npatch, b->d.n, threshold, dflags, b->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(host_flags, dflags, nflag, cudaMemcpyDeviceToHost, b->stream);
  cudaError_t e2 = cudaFreeAsync(dflags, b->stream);
  if (e == cudaSuccess) e = e2;
  if (e == cudaSuccess) e = cudaStreamSynchronize(b->stream);
  if (e != cudaSuccess) return fail(AMR_ECUDA, "flag kernel: %s", cudaGetErrorString(e));
  return AMR_OK;
}

size_t amr_regrid_bytes(const amr_patch_batch* new_fine, const amr_patch_batch* old_fine, const amr_patch_batch* coarse) {
  if (check_regrid_args(new_fine, old_fine, coarse) != AMR_OK) return 0;
  RegridHost H;
  if (build_regrid(new_fine, old_fine, coarse, H) != AMR_OK) return 0;
  return make_regrid_layout(H, coarse).total;
}

int amr_regrid_fill(amr_patch_batch* new_fine, const amr_patch_batch* old_fine, const amr_patch_batch* coarse, void* dev_ws,
                    size_t bytes) {
  int rc = check_regrid_args(new_fine, old_fine, coarse);
  if (rc != AMR_OK) return rc;
  if (new_fine->link_up || new_fine->link_down) return fail(AMR_ESTATE, "fill the new batch before linking it");
  DeviceGuard guard(new_fine->device);
  if (old_fine && old_fine->stream != new_fine->stream) return fail(AMR_EINVAL, "old and new fine batches must share the stream");
  if (!dev_ws || (uintptr_t)dev_ws % ALIGN) return fail(AMR_EINVAL, "workspace must be a %zu-byte aligned device pointer", ALIGN);
  RegridHost H;
  rc = build_regrid(new_fine, old_fine, coarse, H);
  if (rc != AMR_OK) return rc;
  const RegridLayout L = make_regrid_layout(H, coarse);
  if (bytes < L.total) return fail(AMR_EINVAL, "workspace too small: %zu < %zu bytes", bytes, L.total);
  cudaStream_t s = new_fine->stream;
  char* ws = (char*)dev_ws;
  auto h2d = [&](void* dst, const void* src, size_t nb) {
    return nb ? cudaMemcpyAsync(dst, src, nb, cudaMemcpyHostToDevice, s) : cudaSuccess;
  };
  cudaError_t e = h2d(ws + L.pairs, H.pairs.data(), H.pairs.size() * sizeof(int));
  if (e == cudaSuccess) e = h2d(ws + L.born, H.born.data(), H.born.size() * sizeof(int));
  if (e == cudaSuccess) e = h2d(ws + L.cmap, coarse->map.idx.data(), coarse->map.idx.size() * sizeof(int));
  const int nf = new_fine->d.nfields, n = new_fine->d.n, h = n / 2;
  const size_t fs_new = (size_t)new_fine->d.npatch * new_fine->n3;
  if (e == cudaSuccess && old_fine)
    e = amr::launch_copy_patches(new_fine->d.dtype, new_fine->U[new_fine->cur], fs_new, old_fine->U[old_fine->cur],
                                 (size_t)old_fine->d.npatch * old_fine->n3, ws + L.pairs, (int)(H.pairs.size() / 2), nf, n, s);
  if (e == cudaSuccess)
    e = amr::launch_prolong_patches(new_fine->d.dtype, new_fine->U[new_fine->cur], fs_new, nf, n, coarse->d.domain_cells,
                                    coarse->map.dims, coarse->d.bc, ws + L.born, (const int*)(ws + L.cmap),
                                    (int)(H.born.size() / 4) * h * h * h, coarse->U[coarse->cur],
                                    (size_t)coarse->d.npatch * coarse->n3, s);
  // the tables are host vectors: the copies above must have left them before they go out of scope
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail(AMR_ECUDA, "regrid fill: %s", cudaGetErrorString(e));
  new_fine->smax_valid = false;
  new_fine->halo_valid = false;
  return AMR_OK;
}

}  // extern "C"

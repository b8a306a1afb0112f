/* amr_godunov.h -- C-ABI of libamrgodunov.so: the per-patch second-order Godunov hydro/MHD update
 * of arXiv 1412.0934 ("Numerical cosmology on the GPU with Enzo and Ramses") on NVIDIA B200.
 *
 * What the paper offloads (PAPER.md:43 "Piecewise Linear Method"; :57 "inner cells plus boundary
 * cells, properly calculated through interpolation"; :58 "hydro equations are solved on the chunk";
 * :76 "All fluxes necessary to update the patch's cells are computed on the GPU", "only fluxes
 * required for flux correction ... are moved back", "MHD solver"; :31 refinement "in space as well
 * as in time") is built here as one resident-arena library.  The concrete scheme (MUSCL-Hancock
 * PLM + limiter, HLL/HLLC or GLM+HLL/HLLD flux, conservative update, CFL reduction) is fixed by
 * BASELINE.json:north_star; its formulas are the readings O0..O9 / A1..A22 of DESIGN.md §3
 * (SURVEY.md §8(c)).
 *
 * Conventions
 *  - Plain C.  Every call returns an int status (AMR_OK = 0, negative = error); after an error
 *    amr_last_error() gives a thread-local message.  No call throws, none aborts.
 *  - "host" / "device" is stated for every pointer.  Host metadata is copied at create time.
 *  - The DEVICE ARENA is allocated by the caller (e.g. a torch uint8 tensor) and only BORROWED:
 *    the library never frees it and keeps pointers into it until amr_patch_batch_destroy.
 *    The only device memory the library obtains itself is transient and stream-ordered
 *    (cudaMallocAsync / cudaFreeAsync on the batch's stream, released before the call returns):
 *    the staging buffer of a ghosted upload/download and the flag array of amr_flag_blocks.
 *  - The device of a batch is the device its arena lives on.  Every call makes that device
 *    current for its own duration and restores the caller's; linked batches share one device.
 *  - Calls enqueue work on the cudaStream_t given at create time and do not synchronise, except
 *    the ones that return host data (upload/download, amr_cfl_dt, amr_conserved_totals,
 *    amr_step_counters), which synchronise that stream.
 *  - There is no CPU fallback: without a CUDA device every compute call returns AMR_ECUDA.
 *
 * Data layout
 *  - Field order rho, m_x, m_y, m_z, E [, B_x, B_y, B_z, psi]  (mu_0 = 1; reading A20).
 *  - Host arrays are U[field][patch][k][j][i], i (x) fastest, either interiors only (n^3 per
 *    patch) or with nghost ghost layers ((n+2g)^3 per patch).
 *  - In the arena the state is stored INTERIORS ONLY, SoA, U[field][patch][n^3], in two buffers
 *    (old/new) that every step swaps.  Ghost zones are not stored: the step kernel assembles the
 *    radius-2 halo of each tile from the neighbouring patches' interiors through a 27-entry
 *    neighbour table per patch (periodic wrap and outflow clamp resolved on the host at create
 *    time), and from the prolongation halo buffer for fine patches next to a coarser level.
 */
#ifndef AMR_GODUNOV_H_
#define AMR_GODUNOV_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { AMR_OK = 0, AMR_EINVAL = -1, AMR_ENOMEM = -2, AMR_ECUDA = -3, AMR_ESTATE = -4 };
enum { AMR_F32 = 0, AMR_F64 = 1 };
enum { AMR_BC_PERIODIC = 0, AMR_BC_OUTFLOW = 1 };
enum { AMR_LIM_NONE = 0, AMR_LIM_MINMOD = 1, AMR_LIM_MC = 2 };   /* O2, reading A4 */
enum { AMR_RS_HLL = 0, AMR_RS_HLLC = 1, AMR_RS_HLLD = 2 };       /* O5 */
/* amr_step_counters slots (same meaning as the oracle's; reading A7/A10) */
enum { AMR_CNT_POSITIVITY = 0, AMR_CNT_HLL_FALLBACK = 1, AMR_CNT_DEGENERATE_D = 2, AMR_CNT_NEG_STATE = 3 };

typedef struct amr_patch_batch amr_patch_batch; /* opaque; one batch = all equal-size patches of one level */
typedef struct amr_level_link amr_level_link;   /* opaque; coarse<->fine tables + flux registers */

typedef struct {
  int32_t npatch;          /* >= 1 */
  int32_t n;               /* interior cells per side: 8, 16 or 32 (multiple of 8) */
  int32_t nghost;          /* ghost layers of the HOST layout, 2..4 (configs use 3; the stencil uses 2, A11) */
  int32_t nfields;         /* 5 = hydro, 9 = MHD */
  int32_t dtype;           /* AMR_F32 | AMR_F64 */
  int32_t level;           /* 0 = root.  level > 0 reserves the prolongation halo buffer */
  double dx;               /* cell size of this level (> 0) */
  const int32_t* origin;   /* host, [npatch][3] lower corner (x,y,z) in level-cell units; multiples of n */
  int32_t domain_cells[3]; /* extent of this level's index space (multiples of n) */
  int32_t bc[6];           /* xlo,xhi,ylo,yhi,zlo,zhi: AMR_BC_* */
  int32_t self_periodic;   /* 1: every patch is its own periodic neighbour (config 2); origin ignored */
  int32_t nactive;         /* 0 = npatch.  Sharding over GPUs: only the first
                              nactive patches are OWNED - stepped, reduced (smax, totals) - the patches behind them are
                              read-only copies of remote patches (halo sources), refreshed by amr_patch_batch_import */
} amr_batch_desc;

/* Bytes of device arena amr_patch_batch_create needs for this desc (0 on an invalid desc). */
size_t amr_patch_batch_bytes(const amr_batch_desc* desc);

/* Build a batch inside the caller's device arena (device pointer, 256-byte aligned, `bytes` >=
 * amr_patch_batch_bytes).  `cuda_stream` is a cudaStream_t (NULL = default stream).  Builds the
 * neighbour tables on the host (O0: sibling copy with periodic wrap, outflow clamp; a region with
 * no sibling on a level > 0 is marked "from the prolongation halo") and uploads them.
 * Errors: AMR_EINVAL (null pointers, n, nfields, dtype, nghost, dx, origins not multiples of n or
 * outside the domain, duplicate patches, a root-level region with no sibling and no BC, arena too
 * small or misaligned), AMR_ECUDA. */
int amr_patch_batch_create(const amr_batch_desc* desc, void* dev_arena, size_t bytes, void* cuda_stream,
                           amr_patch_batch** out);
int amr_patch_batch_destroy(amr_patch_batch* b);

/* Host <-> arena copies of the CURRENT state (set-up and checking only; never needed per step).
 * host: [nfields][npatch][(n+2g)^3] if with_ghosts else [nfields][npatch][n^3], batch dtype.
 * upload ignores the ghost cells of a ghosted host array.  download with_ghosts=1 returns the
 * ghost cells the step kernel would see (O0 rules (i)-(iii); cells on a level>0 that only O8 can
 * supply come from the last amr_prolong_ghosts, NaN if there was none).  Both synchronise. */
int amr_patch_batch_upload(amr_patch_batch* b, const void* host, int with_ghosts);
int amr_patch_batch_download(amr_patch_batch* b, void* host, int with_ghosts);

/* Device pointer of the current (which=0) or previous (which=1) state buffer, U[field][patch][n^3]. */
void* amr_patch_batch_state(amr_patch_batch* b, int which);

/* O0.  The halo is assembled inside the step kernel, so this only validates the batch and returns
 * AMR_OK; it exists because the hierarchy code above the boundary calls it. */
int amr_fill_ghosts(amr_patch_batch* b);

/* O7 (reading A9): smax = max over interior cells and directions of |v_d| + c_d (c_d = sound speed,
 * or the fast speed along d when mhd != 0); dt = cfl*dx/smax.  If the last call on this batch was a
 * step with the same gamma, the value fused into that step's epilogue is returned (bitwise equal to
 * the standalone reduction); otherwise a reduction kernel runs.  Synchronises.  dt_out/smax_out: host. */
int amr_cfl_dt(amr_patch_batch* b, double gamma, double cfl, int mhd, double* dt_out, double* smax_out);

/* O1..O6 for every patch of the batch: reads the current state (halo assembled on the fly), writes
 * the other buffer, swaps.  amr_hydro_step: nfields must be 5, riemann HLL|HLLC.  amr_mhd_step:
 * nfields 9, riemann HLL|HLLD, ch = GLM wave speed (> 0), alpha = damping constant (psi *=
 * exp(-alpha*ch*dt/dx), reading A8).  Errors: AMR_EINVAL for dt <= 0, non-finite gamma or gamma <= 1,
 * unknown limiter/riemann, wrong nfields; AMR_ESTATE if a level>0 batch was never given a halo. */
int amr_hydro_step(amr_patch_batch* b, double dt, double gamma, int limiter, int riemann);
int amr_mhd_step(amr_patch_batch* b, double dt, double gamma, int limiter, int riemann, double ch,
                 double alpha);

/* Sum over interior cells of each field (double accumulation, deterministic).  totals: host [nfields]. */
/* Halo exchange of a level sharded over GPUs (SURVEY.md 8(f4); PAPER.md:70 "16 GPUs", :72 "one GPU per computing
 * node ... communicating through the network").  dev_pairs: DEVICE, int32 [count][2] =
 * (slot in the packed array, patch index in the batch), borrowed for the call.
 * amr_patch_batch_export copies the CURRENT state of the listed patches into dev_packed[field][count][n^3] (what a
 * rank sends); amr_patch_batch_import copies dev_packed[field][count][n^3] into the listed patches of the current
 * state (what a rank receives into its read-only copies; the fused smax stays valid: it covers owned patches only).
 * Both only enqueue on the batch's stream. */
int amr_patch_batch_export(amr_patch_batch* b, const int32_t* dev_pairs, int32_t count, void* dev_packed);
int amr_patch_batch_import(amr_patch_batch* b, const int32_t* dev_pairs, int32_t count, const void* dev_packed);

/* PPM hydro (SURVEY.md 8(f1); PAPER.md:43 "the Piecewise Parabolic Method, PPM [9]", :76 "the PLM/PPM hydro solver,
 * have been ported to NVIDIA's CUDA").  Reading R-PPM: Colella & Woodward 1984, direct
 * Eulerian, dimensionally split, primitive variables, no optional dissipation, HLL | HLLC flux.
 * amr_hydro_sweep_ppm: ONE sweep along dir (0 = x, 1 = y, 2 = z) over every patch: reads the current state (3 halo
 * cells along dir gathered through the neighbour table: sibling / periodic / outflow / prolongation halo), writes the
 * other buffer, swaps.  amr_hydro_step_ppm: the three sweeps of a step, order 0 = x-y-z, 1 = z-y-x (alternate them
 * step by step).  nfields must be 5, nghost >= 3, n <= 64; the batch must not be linked (no flux registers are
 * recorded: AMR_ESTATE).  No CFL value is fused: the next amr_cfl_dt runs the standalone reduction.  Event counters
 * as for amr_hydro_step (a positivity fallback uses the cell-centre state for both traced states). */
int amr_hydro_sweep_ppm(amr_patch_batch* b, double dt, double gamma, int riemann, int dir);
int amr_hydro_step_ppm(amr_patch_batch* b, double dt, double gamma, int riemann, int order);

int amr_conserved_totals(amr_patch_batch* b, double* totals);

/* The same reduction for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): no batch, no arena, no host copy, no synchronisation.
 * dev_U: DEVICE, [nfields] arrays of dtype (AMR_F32 | AMR_F64), field f at dev_U + f*field_stride elements, the first
 * ncells of each are summed (for a batch: amr_patch_batch_state(b, 0), ncells = field_stride = npatch*n^3).
 * dev_totals: DEVICE, double [nfields], written by the kernel (valid once the stream has reached it).
 * cuda_stream: the cudaStream_t to enqueue on (NULL = the default stream).  All pointers must belong to the CURRENT
 * device; nothing is owned or kept.  Same partition and per-block summation order as amr_conserved_totals; the last
 * sum over the 256 block results runs on the device as a double tree (there: long double on the host), so the two agree
 * to a few ulp of sum|U|, not bitwise.
 * Scratch: the block results live in ONE static device array of 33 024 bytes that every GPU loading the library holds
 * until exit; it fits nfields <= AMR_NOALLOC_MAX_FIELDS, more is AMR_EINVAL.  The call allocates nothing (no
 * cudaMalloc / cudaFree / allocating library routine; the first call on a device looks the array's address up).  All
 * calls on a device share the array: calls ordered on one stream (or by events) are safe, calls that overlap on the GPU
 * race on it and give wrong totals. */
#define AMR_NOALLOC_MAX_FIELDS 16
int amr_conserved_totals_noalloc(const void* dev_U, int dtype, int nfields, int64_t ncells, int64_t field_stride,
                                 double* dev_totals, void* cuda_stream);

/* Event counters accumulated since the last call with reset != 0.  counters: host [4] (AMR_CNT_*).
 * Face events are counted once per tile that computes the face. */
int amr_step_counters(amr_patch_batch* b, long long* counters, int reset);

/* ---- two-level operators (O8, O9; config 4) ------------------------------------------------- */
/* Device workspace a link needs (flux registers, the patch maps of both levels, the fine origins and the list of
 * coarse patches that record fluxes; prolongation, restriction and reflux need no per-cell table: their kernels
 * resolve parents and neighbours through the maps); 0 on error.  Also checks proper nesting: every fine halo region
 * no sibling covers, and its +-1 stencil, must lie inside coarse patches; every fine patch and the coarse cells
 * outside its faces must be covered by the coarse level. */
size_t amr_link_bytes(const amr_patch_batch* coarse, const amr_patch_batch* fine, int ratio);
/* Ties a fine batch to its parent level (ratio must be 2).  dev_ws: device, borrowed like an arena.
 * From then on steps of both batches also record the face fluxes the reflux needs.
 * A batch can be the fine side of one link and the coarse side of another (a middle level); create the
 * links from the root upwards and destroy them in the reverse order (AMR_ESTATE otherwise).  For a middle
 * level amr_flux_clear of its child link zeroes only that link's own coarse faces. */
int amr_link_levels(amr_patch_batch* coarse, amr_patch_batch* fine, int ratio, void* dev_ws, size_t bytes,
                    amr_level_link** out);
int amr_link_destroy(amr_level_link* l);
/* O8: fill the fine halo cells no sibling covers from the coarse level, coarse state =
 * (1-theta)*U_old + theta*U_new where new/old are the coarse batch's current/previous buffers
 * (theta in [0,1]; call after the coarse step).  Conservative minmod-limited linear interpolation. */
int amr_prolong_ghosts(amr_level_link* l, double theta);
/* Zero the flux registers (call before the coarse step of O9). */
int amr_flux_clear(amr_level_link* l);
/* O9(6): covered coarse cell <- mean of its 8 fine cells (current states). */
int amr_restrict(amr_level_link* l);
/* O9(7): U_c += s_f (dt_coarse/dx_coarse) (F_coarse - <F_fine>) on uncovered coarse cells next to a
 * fine patch face, from the fluxes recorded since amr_flux_clear. */
int amr_reflux(amr_level_link* l, double dt_coarse);

/* ---- L-level hierarchy with recursive subcycling -----------------------------------
 * PAPER.md:31 "the different resolution levels are advanced in time with different time-steps"; :59 "once a
 * refinement level is completed the solution is corrected ... and the next (coarser) level of refinement is
 * processed"; :63 all levels stay resident on the device.  levels[0..nlevels) are the batches of levels
 * 0..L-1 (all on one stream), links[l] = amr_link_levels(levels[l], levels[l+1]) created from the root
 * upwards (a middle level is the fine side of one link and the coarse side of the next; the hierarchy must
 * be properly nested: a level-(l+1) halo and its prolongation stencil lie inside level l's patches, else
 * amr_link_levels fails with AMR_EINVAL).  Nothing is owned by these calls.
 *
 * amr_hierarchy_cfl_dt: smax = max over the levels of amr_cfl_dt's smax, dt0 = cfl * dx_0 / smax (the smax
 * kernels of the levels whose fused value is stale and one 8-byte read per level are enqueued first, then one
 * synchronisation).
 * amr_hierarchy_step: one root step dt0.  advance(l, dt): clear link l's flux registers; step level l by dt
 * (hydro or MHD, with c_h = ch on every level); if level l+1 exists, twice { amr_prolong_ghosts(links[l],
 * theta = 0, 1/2); advance(l+1, dt/2) }; amr_restrict(links[l]); amr_reflux(links[l], dt) unless do_reflux
 * is 0.  Level l takes 2^l steps of dt0 / 2^l.  Only kernel launches are enqueued (no synchronisation).
 * Scheduling: the theta = 0 prolongation needs only the coarse level's state BEFORE its step, so it and the fine
 * level's first substep are enqueued on a per-level internal stream before the coarse step goes to the caller's
 * stream (levels overlap on the device; every cross-level dependency is an event; the caller's stream continues
 * after all levels when the call returns).  All levels must have been created on one stream (AMR_EINVAL).
 * AMR_HIERARCHY_OVERLAP=0 in the environment keeps every level on the caller's stream (same results).
 * Errors: AMR_EINVAL for a null pointer, nlevels outside 1..30, links that do not tie consecutive entries of
 * levels, dt0 not finite and > 0; otherwise the first error of the calls listed above. */
int amr_hierarchy_cfl_dt(amr_patch_batch* const* levels, int nlevels, double gamma, double cfl, int mhd,
                         double* dt0_out, double* smax_out);
int amr_hierarchy_step(amr_patch_batch* const* levels, amr_level_link* const* links, int nlevels, int mhd,
                       double dt0, double gamma, int limiter, int riemann, double ch, double alpha, int do_reflux);

/* ---- regridding a level between steps (the paper gives neither criterion nor transfer rule:
 * readings in DESIGN.md 12) ---------------------------------------------------------------------------
 * amr_flag_blocks: host_flags[p*8 + bz*4 + by*2 + bx] (host, caller-owned, npatch*8 bytes) = 1 if the maximum of
 * field `field` of the current state over the aligned (n/2)^3 block (bx, by, bz) of patch p exceeds
 * `threshold` (strictly), else 0.  One kernel + one npatch*8-byte read through a stream-ordered temporary of
 * that size (cudaMallocAsync); synchronises the batch's stream.
 * Which flagged blocks become patches of the next level is the caller's policy; the caller then creates the
 * new fine batch (amr_patch_batch_create with the new origins) and calls
 * amr_regrid_fill(new_fine, old_fine, coarse, ws, bytes): the current state of new_fine becomes, patch by
 * patch, a copy of old_fine's patch with the same origin if there is one (old_fine may be NULL), else the
 * conservative limited linear interpolation of O8 from coarse's current state (the 8 children of a coarse cell
 * average to it: composite totals are unchanged).  dev_ws: device workspace of amr_regrid_bytes(...) bytes,
 * borrowed for the call only.  new_fine must not be linked yet (AMR_ESTATE); link it afterwards (after
 * destroying the old link).  AMR_EINVAL if a new patch without an old twin is not properly nested in coarse. */
int amr_flag_blocks(amr_patch_batch* b, int field, double threshold, unsigned char* host_flags);
size_t amr_regrid_bytes(const amr_patch_batch* new_fine, const amr_patch_batch* old_fine, const amr_patch_batch* coarse);
int amr_regrid_fill(amr_patch_batch* new_fine, const amr_patch_batch* old_fine, const amr_patch_batch* coarse,
                    void* dev_ws, size_t bytes);

/* ---- patch builder ------------------------------------------------------------
 * The procedure the paper designed for the GPU (section 3, Figure 1): "AMR cells are
 * ordered according to a space filling curve based layout; cells are grouped in compact (i.e. with no holes)
 * cubic patches of maximum possible size; neighbouring patches are grouped in large chunks collecting all
 * the data necessary".  Readings: Morton curve (bit b of x -> key bit 3b, y -> 3b+1,
 * z -> 3b+2); a patch is an octree-aligned cube of side 2^k cells, k <= kmax, all of whose cells are present;
 * every cell belongs to the largest such cube; patches are listed in curve order.
 * The workspace is caller-allocated DEVICE memory (borrowed, 256-byte aligned), sized by amr_builder_bytes. */
typedef struct amr_patch_builder amr_patch_builder;
size_t amr_builder_bytes(int64_t ncell_max);                       /* 0 if ncell_max is outside [1, 2^30] */
int amr_builder_create(int64_t ncell_max, void* dev_ws, size_t bytes, void* cuda_stream, amr_patch_builder** out);
int amr_builder_destroy(amr_patch_builder* b);
/* Steps 1 + 2.  dev_xyz: DEVICE int32 [3][ncell], the (x, y, z) of the unique leaf cells of one level, each in
 * [0, 2^bits); bits 1..10; kmax 0..min(5, bits).  Synchronises the stream; *npatch_out = number of patches.
 * AMR_EINVAL for bad arguments or duplicate cells. */
int amr_builder_build(amr_patch_builder* b, const int32_t* dev_xyz, int64_t ncell, int32_t bits, int32_t kmax,
                      int64_t* npatch_out);
/* Results of the last build, HOST arrays, each may be NULL: perm [ncell] (perm[i] = input index of the i-th cell
 * along the curve), first [npatch] (curve position of the patch's first cell; its 8^level cells follow in
 * Morton order), level [npatch] (k: side 2^k), origin [npatch][3] (x, y, z of the lower corner). */
int amr_builder_results(amr_patch_builder* b, int64_t* perm, int64_t* first, int32_t* level, int32_t* origin);
/* Step 3 for the patches of side n = 2^k (curve order): dev_out[f][p][lz][ly][lx] = dev_fields[f][cell at
 * origin_p + (lx, ly, lz)], i.e. the [nfields][npatch][n^3] layout amr_patch_batch_upload's device arena uses.
 * dev_fields: DEVICE [nfields][ncell] in INPUT order; dev_out: DEVICE, room for max_patches patches;
 * host_origin: HOST [count][3] or NULL; *count_out = number of such patches.  With dev_out == NULL and
 * host_origin == NULL only the count is returned.  With host_origin == NULL the gather is only enqueued on
 * the builder's stream (no synchronisation); with host_origin it synchronises.  AMR_ENOMEM if count >
 * max_patches. */
int amr_builder_gather(amr_patch_builder* b, const void* dev_fields, int32_t nfields, int32_t dtype, int32_t k,
                       void* dev_out, int64_t max_patches, int32_t* host_origin, int64_t* count_out);

/* Measurement aid for the benchmark's ALU roofline ("an FMA-chain microbenchmark in the
 * same run"); not a step of the path.  Runs plain dependent-FMA chains on every SM for about `ms_target`
 * milliseconds on cuda_stream (dev_scratch: DEVICE, >= 8 bytes, borrowed) and returns the measured rate in
 * *tflops_out (2 flops per FMA per lane; dtype AMR_F32 or AMR_F64).  Synchronises the stream. */
int amr_measure_fma_peak(int32_t dtype, void* dev_scratch, void* cuda_stream, double ms_target, double* tflops_out);

const char* amr_last_error(void);
/* Library/build description, e.g. "amr_godunov sm_100a ..." (static string). */
const char* amr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AMR_GODUNOV_H_ */

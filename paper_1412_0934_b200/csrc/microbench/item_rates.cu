// Diagnostic program, not part of the library: how fast do the two building blocks of the fp32 MHD step kernel run
// when NOTHING else is in the way - every warp of the SM executes the same small loop (instruction cache hit rate
// 99.99 %), operands and results in conflict-free shared-memory pair records, no global traffic?
//   P item = x2::predict_pair (MC slopes, MUSCL-Hancock predictor, positivity) + the six face-state records
//   R item = two records -> x2::riemann2 (HLLD) -> one flux record
// Modes: R only, P only, and 1 P + 2 R items per thread and iteration; each with and without a CTA-wide barrier per
// iteration, at 12 / 16 / 20 warps per SM (168 / 128 / 96 registers).  Used for profiles/r2e_building_blocks.md and
// the answer bounds what ANY re-arrangement of the same arithmetic (role-split pipelines, smaller
// hot code, more warps) can reach.
// Build: python -m paper_1412_0934_b200.build --microbench  ->  paper_1412_0934_b200/build/microbench/item_rates
#include <cstdio>
#include <cstdlib>
#include <vector>
#include "godunov_step_x2.cuh"
using namespace amr; using namespace amr::x2;
#ifndef ITEM_NF
#define ITEM_NF 9          // -DITEM_NF=5: the hydro items (HLLC)
#endif
constexpr int NF = ITEM_NF, REC = NF == 9 ? 20 : 12, NPX = 18;
constexpr int RSV = NF == 9 ? X2_RS_HLLD : X2_RS_HLLC;

template <int MODE, int MAXR, int BAR = 1>
__global__ void __maxnreg__(MAXR) mb(const __grid_constant__ StepParams<float> P, const float* __restrict__ init, int RH, int npool, int niter,
                                     float* sink) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float* ring = reinterpret_cast<float*>(smem_raw);
  const int SLOT = RH * NPX * REC;
  float* pool = ring + 3 * SLOT;            // npool records (face states)
  float* fpool = pool + npool * REC;        // npool/2 records (fluxes)
  __shared__ int s_cnt[4];
  const int tid = threadIdx.x, NT = blockDim.x;
  const int total = 3 * SLOT + npool * REC;
  for (int i = tid; i < total; i += NT) ring[i] = init[i];
  if (tid < 4) s_cnt[tid] = 0;
  __syncthreads();
  RC2 RC;
  RC.gamma = P.gamma; RC.igm1 = P.igm1; RC.ch2 = P.ch2; RC.half_ch = 0.5f * P.ch; RC.half_ich = P.half_ich; RC.eps = P.eps;
  const F2 ms = F2(-P.dtdx);
  const int npos = (RH - 2) * (NPX - 2);
  float* Wm = ring; float* Wc = ring + SLOT; float* Wp = ring + 2 * SLOT;
  for (int it = 0; it < niter; ++it) {
    if (MODE == 1 || MODE == 2) {
      const int pos = (tid + it * 7) % npos;
      const int r = 1 + pos / (NPX - 2), c = 1 + pos % (NPX - 2);
      const int rc = (r * NPX + c) * REC;
      F2 ws[NF], hx[NF], hy[NF], hz[NF];
      predict_pair<NF, X2_LIM_MC>(Wm, Wc, Wp, rc, NPX * REC, REC, P, ms, B2(true), ws, hx, hy, hz);
      F2 t[NF];
      const int base = tid;
#define OUT(k, expr) { _Pragma("unroll") for (int q = 0; q < NF; ++q) t[q] = expr; sts_pairs<NF>(pool + ((base + k * NT) % npool) * REC, t); }
      OUT(0, ws[q] + hx[q]) OUT(1, ws[q] - hx[q]) OUT(2, ws[q] + hy[q]) OUT(3, ws[q] - hy[q]) OUT(4, ws[q] + hz[q]) OUT(5, ws[q] - hz[q])
#undef OUT
      if (MODE == 2 && BAR) __syncthreads();
    }
    if (MODE == 0 || MODE == 2) {
#pragma unroll 1
      for (int rep = 0; rep < 2; ++rep) {
        const int lo = (tid + rep * NT + it) % npool, ro = (lo + 1) % npool;
        F2 WL[NF], WR[NF], F[NF];
        lds_pairs<NF>(pool + lo * REC, WL);
        lds_pairs<NF>(pool + ro * REC, WR);
        riemann2<NF, RSV>(WL, WR, RC, F, B2(true), s_cnt);
        sts_pairs<NF>(fpool + ((tid + rep * NT) % (npool / 2)) * REC, F);
      }
    }
    if (BAR) __syncthreads();
    float* tmp = Wm; Wm = Wc; Wc = Wp; Wp = tmp;
  }
  if (tid == 0) sink[blockIdx.x] = fpool[3] + pool[5] + (float)s_cnt[1];
}

template <int MODE, int MAXR, int BAR = 1>
void run(const char* name, int NT, int RH, int npool, int ctas_per_sm, const StepParams<float>& P, const float* dinit, float* dsink) {
  const int SLOT = RH * NPX * REC;
  const size_t smem = (size_t)(3 * SLOT + npool * REC + (npool / 2) * REC) * 4;
  auto k = mb<MODE, MAXR, BAR>;
  cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  int occ = 0;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, NT, smem);
  const int grid = 148 * ctas_per_sm, niter = 400;
  k<<<grid, NT, smem>>>(P, dinit, RH, npool, 10, dsink);
  cudaDeviceSynchronize();
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  cudaEventRecord(e0);
  k<<<grid, NT, smem>>>(P, dinit, RH, npool, niter, dsink);
  cudaEventRecord(e1);
  cudaError_t e = cudaDeviceSynchronize();
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  const double items_p = (MODE == 0 ? 0.0 : 1.0) * NT / 32.0 * ctas_per_sm * niter;   // warp-items per SM
  const double items_r = (MODE == 1 ? 0.0 : 2.0) * NT / 32.0 * ctas_per_sm * niter;
  int khz = 0;
  cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
  // cycles of one scheduler (SMSP) per warp-item it executes, at the device's maximum SM clock
  const double cyc_smsp = ms * 1e-3 * khz * 1e3 / ((items_p + items_r) / 4.0);
  printf("%-42s %2d warps/SM (occ %d), smem %3zu KB: %.3f ms, %6.0f P + %6.0f R warp-items per SM -> %.1f ns per warp-item per SM, %.0f cycles per warp-item per scheduler  [%s]\n",
         name, NT / 32 * ctas_per_sm, occ, smem / 1024, ms, items_p, items_r, 1e6 * ms / (items_p + items_r), cyc_smsp, cudaGetErrorString(e));
}

int main() {
  const int RHmax = 20, npoolmax = 1024;
  const int tot = 3 * RHmax * NPX * REC + npoolmax * REC;
  std::vector<float> h(tot);
  srand(1);
  auto rnd = [] { return (float)rand() / RAND_MAX - 0.5f; };
  for (int r = 0; r < tot / REC; ++r) {
    float* d = &h[r * REC];
    for (int half = 0; half < 2; ++half) {
      d[0 + half] = 1.f + 0.3f * rnd();
      d[2 + half] = 0.8f * rnd(); d[4 + half] = 0.8f * rnd(); d[6 + half] = 0.8f * rnd();
      d[8 + half] = 1.f + 0.3f * rnd();
      if (NF == 9) {
        d[10 + half] = 0.2f * rnd(); d[12 + half] = 0.2f * rnd(); d[14 + half] = 0.2f * rnd();
        d[16 + half] = 0.01f * rnd();
      }
    }
    for (int i = 2 * NF; i < REC; ++i) d[i] = 0.f;
  }
  float *dinit, *dsink;
  cudaMalloc(&dinit, tot * 4);
  cudaMalloc(&dsink, 148 * 8 * 4);
  cudaMemcpy(dinit, h.data(), tot * 4, cudaMemcpyHostToDevice);
  StepParams<float> P{};
  P.gamma = 5.f / 3.f; P.gm1 = 2.f / 3.f; P.igm1 = 1.5f; P.ch = 3.f; P.ch2 = 9.f; P.half_ich = 0.5f / 3.f; P.damp = 0.9f; P.eps = 1e-6f;
  P.dtdx = 0.1f; P.hdtdx = 0.05f;
  run<0, 168>("R only, 168 regs, 12 warps", 384, 12, 1024, 1, P, dinit, dsink);
  run<0, 128>("R only, 128 regs, 16 warps", 512, 12, 1024, 1, P, dinit, dsink);
  run<0, 96>("R only, 96 regs, 20 warps", 640, 12, 1024, 1, P, dinit, dsink);
  run<0, 168, 0>("R only, 168 regs, 12 warps, no barrier", 384, 12, 1024, 1, P, dinit, dsink);
  run<0, 128, 0>("R only, 128 regs, 16 warps, no barrier", 512, 12, 1024, 1, P, dinit, dsink);
  run<0, 168>("R only, 168 regs, 8 warps", 256, 12, 1024, 1, P, dinit, dsink);
  run<0, 168>("R only, 168 regs, 4 warps", 128, 12, 1024, 1, P, dinit, dsink);
  run<1, 168>("P only, 168 regs, 12 warps", 384, 20, 1024, 1, P, dinit, dsink);
  run<1, 128>("P only, 128 regs, 16 warps", 512, 20, 1024, 1, P, dinit, dsink);
  run<1, 168, 0>("P only, 168 regs, 12 warps, no barrier", 384, 20, 1024, 1, P, dinit, dsink);
  run<2, 168>("P + 2R, 168 regs, 12 warps", 384, 20, 1024, 1, P, dinit, dsink);
  run<2, 128>("P + 2R, 128 regs, 16 warps", 512, 20, 1024, 1, P, dinit, dsink);
  run<2, 168, 0>("P + 2R, 168 regs, 12 warps, no barrier", 384, 20, 1024, 1, P, dinit, dsink);
  run<2, 128, 0>("P + 2R, 128 regs, 16 warps, no barrier", 512, 20, 1024, 1, P, dinit, dsink);
  return 0;
}

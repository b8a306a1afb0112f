// Diagnostic program, not part of the library: issue cost of the instruction classes the fp32 step kernel is made of,
// and whether the pipes of a scheduler (SMSP) overlap.  16 warps per SM, 8 independent dependency chains per thread,
// so every number is a pipe rate, not a latency.  Used for profiles/r2e_building_blocks.md and the ALU bound of
// DESIGN.md section 7.
// Build: python -m paper_1412_0934_b200.build --microbench  ->  paper_1412_0934_b200/build/microbench/pipe_rates
#include <cstdio>
#include <cuda_runtime.h>

__device__ __forceinline__ float rcpf(float a) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
__device__ __forceinline__ float sqf(float a) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }

constexpr int NCH = 8;
// MODE bits: 1 = FFMA2, 2 = FMNMX, 4 = MUFU (1 per 8 others), 8 = scalar FFMA, 16 = FSEL+FSETP, 32 = FMNMX3
template <int MODE>
__global__ void __launch_bounds__(512) k(float* out, int niter, float a, float b) {
  float2 x[NCH];
  float y[NCH], z[NCH], s[NCH], w[NCH];
#pragma unroll
  for (int i = 0; i < NCH; ++i) {
    x[i] = make_float2(threadIdx.x * 1e-3f + i, 1.f + i);
    y[i] = threadIdx.x * 1e-2f + i; z[i] = 1.f + threadIdx.x + i; s[i] = i + 0.5f; w[i] = 2.f * i + threadIdx.x;
  }
  const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
#pragma unroll 1
  for (int it = 0; it < niter; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int i = 0; i < NCH; ++i) {
        if (MODE & 1) x[i] = __ffma2_rn(x[i], a2, b2);
        if (MODE & 2) { y[i] = fminf(y[i], z[i]); z[i] = fmaxf(z[i], y[i]); }
        if (MODE & 8) s[i] = __fmaf_rn(s[i], a, b);
        if (MODE & 16) w[i] = (w[i] > y[(i + 1) % NCH]) ? s[(i + 3) % NCH] : w[i];
        if (MODE & 32) { float t; asm("min.f32 %0, %1, %2, %3;" : "=f"(t) : "f"(y[i]), "f"(z[i]), "f"(w[i])); y[i] = t; }
        if (MODE & 64) { s[i] = __fmaf_rn(s[i], x[i].x, x[(i + 1) % NCH].y); x[i].x = __fmaf_rn(x[i].x, s[(i + 3) % NCH], x[(i + 5) % NCH].y); }
      }
      if (MODE & 4) z[r % NCH] = rcpf(z[r % NCH]);
    }
  }
  float acc = 0.f;
#pragma unroll
  for (int i = 0; i < NCH; ++i) acc += x[i].x + x[i].y + y[i] + z[i] + s[i] + w[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

template <int MODE>
void run(const char* name, float* d, double ninstr_per_iter) {
  const int niter = 2000;
  k<MODE><<<148, 512>>>(d, 10, 0.999f, 0.001f);
  cudaDeviceSynchronize();
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  cudaEventRecord(e0);
  k<MODE><<<148, 512>>>(d, niter, 0.999f, 0.001f);
  cudaEventRecord(e1);
  cudaDeviceSynchronize();
  float ms;
  cudaEventElapsedTime(&ms, e0, e1);
  // 16 warps per SM = 4 per SMSP
  int khz = 0;
  cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
  const double cyc = ms * 1e-3 * khz * 1e3;   // at the device's maximum SM clock
  printf("%-40s %.3f ms  %.2f cycles per iteration per SMSP (4 warps), nominal instr/iter/warp %.0f -> %.2f cyc per warp-instr per SMSP\n", name, ms,
         cyc / niter, ninstr_per_iter, cyc / niter / (4 * ninstr_per_iter));
}

int main() {
  float* d;
  cudaMalloc(&d, 148 * 512 * 4);
  run<1>("FFMA2", d, 64);
  run<8>("FFMA scalar", d, 64);
  run<2>("FMNMX (x2 per slot)", d, 128);
  run<32>("FMNMX3", d, 64);
  run<16>("FSETP+FSEL", d, 128);
  run<4>("MUFU.RCP (8 per iter)", d, 8);
  run<1 | 2>("FFMA2 + 2 FMNMX", d, 192);
  run<1 | 32>("FFMA2 + FMNMX3", d, 128);
  run<1 | 8>("FFMA2 + FFMA", d, 128);
  run<1 | 4>("FFMA2 x64 + MUFU x8", d, 72);
  run<2 | 4>("FMNMX x128 + MUFU x8", d, 136);
  run<1 | 2 | 4>("FFMA2 x64 + FMNMX x128 + MUFU x8", d, 200);
  run<1 | 16>("FFMA2 + FSETP/FSEL", d, 192);
  // register-file operand bandwidth: 2 FFMA (3 distinct registers each) + FMNMX3 (3) = 9 operand reads per slot; the
  // pipes alone would need 2 cycles (fma: 2 x 1, alu: 1 x 2)
  run<64>("2 FFMA, distinct operands", d, 128);
  run<64 | 32>("2 FFMA distinct + FMNMX3", d, 192);
  run<64 | 2>("2 FFMA distinct + 2 FMNMX", d, 256);
  return 0;
}

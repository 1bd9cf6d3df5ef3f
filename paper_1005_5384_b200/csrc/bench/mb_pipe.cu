// MEASUREMENT AID, not part of the library: what an FFMA2 / FFMA stream sustains per SM sub-partition as a function of
// where its operands come from (distinct registers, shared registers = operand-reuse cache), alone and mixed with
// MUFU / LDS.  Evidence for "the force kernel is bound by register-file operand bandwidth" (
// results: profiles/r02_microbench.md).
//   nvcc -std=c++17 -O3 -gencode arch=compute_100a,code=sm_100a -o /tmp/mb_pipe paper_1005_5384_b200/csrc/bench/mb_pipe.cu && /tmp/mb_pipe
#include <cstdio>
#include <cuda_runtime.h>
typedef unsigned long long f2;
__device__ __forceinline__ f2 pk(float lo, float hi) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ float lo(f2 v) { float a; asm("{ .reg .b32 t; mov.b64 {%0, t}, %1; }" : "=f"(a) : "l"(v)); return a; }
__device__ __forceinline__ float hi(f2 v) { float b; asm("{ .reg .b32 t; mov.b64 {t, %0}, %1; }" : "=f"(b) : "l"(v)); return b; }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { f2 d; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 d; asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ float fma1(float a, float b, float c) { float d; asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c)); return d; }
__device__ __forceinline__ float rsq(float x) { float y; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

constexpr int NCH = 12;
// MODE 0: packed, 3 distinct register operands (acc, x, y)      1: packed, acc = fma2(acc, c, d) shared c, d
// MODE 2: scalar 3 distinct                                       3: packed 3 distinct + 1 MUFU per MUF packed
// MODE 4: packed 3 distinct + LDS.128 per LDSN packed             5: scalar + MUFU per MUF       6: packed with broadcast scalar operand (pk(s,s))
template <int MODE, int MUF, int LDSN>
__global__ void __launch_bounds__(128, 4) k(int n, float s, float* out) {
  __shared__ float4 sm[256];
  sm[threadIdx.x] = make_float4(s, s * 2, s * 3, s * 4); sm[threadIdx.x + 128] = make_float4(s, s, s, s);
  __syncthreads();
  f2 acc[NCH], x[NCH], y[NCH];
  float a1[NCH], x1[NCH], y1[NCH];
#pragma unroll
  for (int i = 0; i < NCH; i++) {
    acc[i] = add2(pk(threadIdx.x * 0.001f + i, 1.f), pk(0.f, 0.f)); x[i] = add2(pk(s + 1e-3f * i, s), pk(0.f, 0.f)); y[i] = add2(pk(1.f - s, 1e-3f * i), pk(0.f, 0.f));
    a1[i] = threadIdx.x * 0.001f + i; x1[i] = s + 1e-3f * i; y1[i] = 1.f - s - 1e-3f * i;
  }
  float mu = 1.f + s; float4 ld = make_float4(0, 0, 0, 0);
  const f2 c = add2(pk(s, s), pk(0.f, 0.f)), d = add2(pk(1.f - s, 1.f - s), pk(0.f, 0.f));
  int cnt = 0;
  for (int t = 0; t < n; t++) {
#pragma unroll
    for (int i = 0; i < NCH; i++) {
      if (MODE == 0 || MODE == 3 || MODE == 4) acc[i] = fma2(x[i], y[i], acc[i]);
      else if (MODE == 1) acc[i] = fma2(acc[i], c, d);
      else if (MODE == 2 || MODE == 5) { a1[i] = fma1(x1[i], y1[i], a1[i]); a1[i] = fma1(y1[i], x1[(i + 1) % NCH], a1[i]); }
      else if (MODE == 6) acc[i] = fma2(pk(x1[i], x1[i]), y[i], acc[i]);
      if ((MODE == 3 || MODE == 5) && (i % MUF) == MUF - 1) mu = rsq(mu);
      if (MODE == 4 && (i % LDSN) == LDSN - 1) { const float4 v = sm[(cnt++ + threadIdx.x) & 255]; ld.x += v.x; }
    }
  }
  float r = mu + ld.x;
#pragma unroll
  for (int i = 0; i < NCH; i++) r += lo(acc[i]) + hi(acc[i]) + a1[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}
template <int MODE, int MUF = 4, int LDSN = 4>
void run(const char* name, double fma_per_iter) {
  const int grid = 148 * 4, n = 20000;
  float* d; cudaMalloc(&d, sizeof(float) * grid * 128);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  k<MODE, MUF, LDSN><<<grid, 128>>>(100, 0.999f, d);
  float best = 1e30f;
  for (int it = 0; it < 3; it++) {
    cudaEventRecord(e0); k<MODE, MUF, LDSN><<<grid, 128>>>(n, 0.999f, d); cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1); best = ms < best ? ms : best;
  }
  // per SMSP: 4 warps x n iterations x fma_per_iter FMA-pipe warp-instructions
  const double cyc = best * 1e-3 * 1.965e9;
  printf("%-55s %.3f ms  cycles per FMA-pipe instruction (per SMSP): %.3f\n", name, best, cyc / (4.0 * n * fma_per_iter));
  cudaFree(d);
}
int main() {
  run<0>("FFMA2 acc=fma2(x_i,y_i,acc_i) 3 distinct regs", NCH);
  run<1>("FFMA2 acc=fma2(acc_i,c,d) shared c,d", NCH);
  run<6>("FFMA2 acc=fma2(bcast x1_i, y_i, acc_i)", NCH);
  run<2>("FFMA  2 per chain, 3 distinct regs", 2 * NCH);
  run<3, 4>("FFMA2 3 distinct + MUFU per 4", NCH);
  run<3, 6>("FFMA2 3 distinct + MUFU per 6", NCH);
  run<3, 12>("FFMA2 3 distinct + MUFU per 12", NCH);
  run<5, 2>("FFMA 2/chain + MUFU per 4 FFMA", 2 * NCH);
  run<5, 6>("FFMA 2/chain + MUFU per 12 FFMA", 2 * NCH);
  run<4, 4, 4>("FFMA2 3 distinct + LDS.128 per 4", NCH);
  run<4, 4, 12>("FFMA2 3 distinct + LDS.128 per 12", NCH);
  return 0;
}

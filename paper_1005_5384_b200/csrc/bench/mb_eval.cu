// MEASUREMENT AID, not part of the library: the evaluation loops of tc_kernels.cu ALONE (the same code — this file
// includes the kernel source —, the same launch bounds and shared memory, hence the same occupancy), per K particles
// per lane and S slices.  It is where kRecordCycles[] of tc_lanes.h and the "loops' own ceiling" of DESIGN.md
// section 6 come from (results: profiles/r02_microbench.md).
//   nvcc -std=c++17 -O3 -gencode arch=compute_100a,code=sm_100a -o /tmp/mb_eval paper_1005_5384_b200/csrc/bench/mb_eval.cu
//   /tmp/mb_eval            # every K at S = 1, particle-cell and particle-particle
//   /tmp/mb_eval warps      # throughput against the number of resident warps per SM sub-partition
//   /tmp/mb_eval slices     # S > 1 slices of the list
#include "../tc_kernels.cu"
#include <cstdio>
namespace tc { namespace {
template <int K, int WHAT>
__global__ void __launch_bounds__(kWarpsPerCta * 32, TC_MINB) mb(int S, int reps, float eps2, float* out, int cnt_arg) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  WarpSmem<256>& sm = reinterpret_cast<WarpSmem<256>*>(smem_raw)[warp];
  for (int t = lane; t < kCellCap; t += 32) {
    CellRec r; r.xm = make_float4(10.f + t, 3.f, -2.f + 0.1f * t, 1e-3f); r.q0 = make_float4(1e-4f, -2e-4f, 1e-4f, 3e-5f); r.q1 = make_float2(1e-5f, 2e-5f); r.pad = make_float2(0, 0);
    sm.u.cell[t] = r;
  }
  __syncwarp();
  Lanes L; L.S = S; L.q = 32 / S; L.K = K; L.s = lane / L.q; L.p = lane - L.s * L.q; L.active = L.s < L.S;
  PassState ps;
#pragma unroll
  for (int j = 0; j < kMaxKP; j++) {
    ps.A[j].ax = ps.A[j].ay = ps.A[j].az = ps.A[j].npot = 0ull;
    ps.P[j].x = add2(pk(0.01f * lane + j, 0.02f * lane - j), bc(0.f)); ps.P[j].y = add2(pk(0.3f * lane, 0.1f * j), bc(0.f)); ps.P[j].z = add2(pk(1.f * j, 2.f + lane), bc(0.f));
  }
  ps.p1.x = 0.5f * lane; ps.p1.y = 1.f; ps.p1.z = -lane; ps.a1.ax = ps.a1.ay = ps.a1.az = ps.a1.npot = 0.f;
  const int cnt = cnt_arg;
  for (int r = 0; r < reps; r++) {
    if (WHAT == 0) eval_cells_k<K / 2, (K & 1) != 0>(sm.u.cell, cnt, eps2, L, ps);
    else eval_bodies_k<K / 2, (K & 1) != 0, false>(sm.u.bs.body, cnt, eps2, L, ps);
    __syncwarp();
  }
  float s = ps.a1.ax + ps.a1.npot;
#pragma unroll
  for (int j = 0; j < kMaxKP; j++) s += lo(ps.A[j].ax) + hi(ps.A[j].ay) + lo(ps.A[j].npot) + hi(ps.A[j].az);
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <int K, int WHAT>
void run(int S, int ctas = 0) {
  const size_t smem = sizeof(WarpSmem<256>) * kWarpsPerCta;
  cudaFuncSetAttribute(mb<K, WHAT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  int per_sm = 0; cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, mb<K, WHAT>, kWarpsPerCta * 32, smem);
  if (ctas) per_sm = ctas;
  const int grid = 148 * per_sm, reps = 400;
  float* d; cudaMalloc(&d, sizeof(float) * grid * kWarpsPerCta * 32);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  mb<K, WHAT><<<grid, kWarpsPerCta * 32, smem>>>(S, 10, 1e-4f, d, (WHAT == 0) ? kCellCap : kBodyCap);
  float best = 1e30f;
  for (int it = 0; it < 3; it++) {
    cudaEventRecord(e0); mb<K, WHAT><<<grid, kWarpsPerCta * 32, smem>>>(S, reps, 1e-4f, d, (WHAT == 0) ? kCellCap : kBodyCap); cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1); best = ms < best ? ms : best;
  }
  const int cnt = (WHAT == 0) ? kCellCap : kBodyCap;
  const int q = 32 / S;
  // interactions: per warp per rep: cnt records x q*K particles (each slice takes cnt/S records, S slices x q lanes x K)
  const double inter = (double)grid * kWarpsPerCta * reps * (double)cnt * q * K;
  const double instr = (WHAT == 0) ? 33.0 : 13.0;
  const double ideal = 148.0 * 4 * 32 * 1.965e9 / instr;   // interactions/s if every FMA-pipe lane-cycle were an interaction instruction
  printf("%s K=%d S=%2d per_sm=%d: %.3f ms  %.3e inter/s  = %.1f %% of the FP32-issue ideal (lanes used %d/32)\n", WHAT == 0 ? "pc" : "pp", K, S, per_sm, best,
         inter / (best * 1e-3), 100.0 * inter / (best * 1e-3) / ideal, S * q);
  cudaFree(d);
}
}}
int main(int argc, char** argv) {
  using namespace tc;
  if (argc > 1 && argv[1][0] == 's') {   // S > 1 slices: lanes of different slices read different records in one load
    run<2, 0>(1); run<2, 0>(2); run<2, 0>(4); run<2, 0>(8); run<2, 0>(16); run<4, 0>(1); run<4, 0>(4); run<4, 0>(8); run<6, 0>(2); run<6, 0>(5);
    return 0;
  }
  if (argc > 1) {   // throughput vs resident warps per sub-partition (CTAs per SM)
    for (int c = 1; c <= 4; c++) run<6, 0>(1, c);
    for (int c = 1; c <= 4; c++) run<4, 0>(4, c);
    for (int c = 1; c <= 4; c++) run<2, 0>(1, c);
    for (int c = 1; c <= 4; c++) run<7, 0>(1, c);
    return 0;
  }
  run<1, 0>(1); run<2, 0>(1); run<3, 0>(1); run<4, 0>(1); run<5, 0>(1); run<6, 0>(1); run<7, 0>(1); run<8, 0>(1);
  run<1, 1>(1); run<2, 1>(1); run<3, 1>(1); run<4, 1>(1); run<6, 1>(1); run<8, 1>(1);
  return 0;
}

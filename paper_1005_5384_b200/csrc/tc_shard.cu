// ONE force evaluation over k GPUs: layout of the shards and the scatter
// of the all-gathered result.  Groups are independent given the read-only tree (one walk per group,
// no exchange between groups), so rank r simply evaluates the schedule positions r, r + k, ... (the schedule is
// cost-ordered: strided shards are balanced) and writes ONLY its particles, compactly: its groups in that order,
// particles in tree order inside a group.  The one exchange hands every rank the rows of the others (one
// all-gather of 16 bytes per particle, done by the caller); the kernel here scatters the gathered rows to the
// caller's particle order.  No collective inside the walk or the evaluation.
#include <cuda_runtime.h>

#include <cub/device/device_scan.cuh>

#include <algorithm>
#include <cstdint>
#include <vector>

#include "tc_internal.h"

namespace tc {
namespace {

// schedule position i belongs to rank i % k and is that rank's (i / k)-th group; in RANK-MAJOR order (all groups
// of rank 0, then rank 1, ...) it has index rank_start(i % k) + i / k
__host__ __device__ inline long long rank_start(int r, long long ng, int k) {
  const long long rem = ng % k;
  return (long long)r * (ng / k) + (r < rem ? (long long)r : rem);
}

__global__ void k_shard_counts(const int4* __restrict__ grp, int ng, int k, int32_t* __restrict__ cnt) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i > ng) return;
  if (i == ng) { cnt[ng] = 0; return; }             // the scan runs over ng + 1 entries: its last value is the total
  const int g = __ldg(&grp[i].w);                    // i-th group to run
  cnt[rank_start(i % k, ng, k) + i / k] = __ldg(&grp[g].z);
}

__global__ void k_shard_off(const int32_t* __restrict__ scan, int ng, int k, int32_t* __restrict__ off, int32_t* __restrict__ rank_rows) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < ng) {
    const long long s = rank_start(i % k, ng, k);
    off[i] = scan[s + i / k] - scan[s];
  }
  if (i < k) rank_rows[i] = scan[rank_start(i + 1, ng, k)] - scan[rank_start(i, ng, k)];   // particles rank i evaluates
}

// one warp per schedule position: rows of the group's particles in the gathered buffer [k, n_slots]
__global__ void k_shard_slots(const int4* __restrict__ grp, const int32_t* __restrict__ off, int ng, int k, long long n_slots,
                              int32_t* __restrict__ slot) {
  const int i = (int)((blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
  if (i >= ng) return;
  const int g = __ldg(&grp[i].w);
  const int4 G = __ldg(grp + g);
  const long long base = (long long)(i % k) * n_slots + off[i];
  for (int t = lane; t < G.z; t += 32) slot[G.y + t] = (int32_t)(base + t);
}

// HBM-bound: 24 bytes read + 16 (+ 8) written per particle
__global__ void k_shard_scatter(const float4* __restrict__ gathered, const int2* __restrict__ gcnt, const int32_t* __restrict__ slot,
                                const int32_t* __restrict__ orig, long long n, float* __restrict__ acc, float* __restrict__ pot,
                                int32_t* __restrict__ n_pc, int32_t* __restrict__ n_pp) {
  const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (t >= n) return;
  const int s = __ldg(slot + t);
  const float4 v = __ldg(gathered + s);
  const size_t i = (size_t)__ldg(orig + t);
  acc[3 * i + 0] = v.x; acc[3 * i + 1] = v.y; acc[3 * i + 2] = v.z;
  if (pot) pot[i] = v.w;
  if (gcnt) {
    const int2 c = __ldg(gcnt + s);
    if (n_pc) n_pc[i] = c.x;
    if (n_pp) n_pp[i] = c.y;
  }
}

template <typename T>
cudaError_t grow(T*& p, size_t& cap, size_t need) {
  if (cap >= need) return cudaSuccess;
  cudaFree(p); p = nullptr; cap = 0;
  const cudaError_t e = cudaMalloc((void**)&p, sizeof(T) * need);
  if (e == cudaSuccess) cap = need;
  return e;
}

}  // namespace

#define TS_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return (int)e_; } while (0)

void ShardLayout::release() {
  cudaFree(off); cudaFree(slot); cudaFree(cnt); cudaFree(scan); cudaFree(tmp);
  *this = ShardLayout();
}

int build_shard_layout(const DeviceTree& T, int k, ShardLayout& L, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  const long long ng = T.n_groups, n = T.n;
  L.k = 0;
  TS_CUDA(cudaStreamSynchronize(st));       // nothing in flight reads the arrays that may be re-allocated below
  TS_CUDA(grow(L.off, L.cap_off, (size_t)ng)); TS_CUDA(grow(L.slot, L.cap_slot, (size_t)n));
  TS_CUDA(grow(L.cnt, L.cap_cnt, (size_t)std::max<long long>(ng + 1, k))); TS_CUDA(grow(L.scan, L.cap_scan, (size_t)ng + 1));
  const int tpb = 256;
  k_shard_counts<<<(unsigned)((ng + 1 + tpb - 1) / tpb), tpb, 0, st>>>(T.grp, (int)ng, k, L.cnt);
  size_t need = 0;
  TS_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, need, L.cnt, L.scan, (int)(ng + 1), st));
  TS_CUDA(grow(L.tmp, L.cap_tmp, need));
  TS_CUDA(cub::DeviceScan::ExclusiveSum(L.tmp, need, L.cnt, L.scan, (int)(ng + 1), st));
  // (cnt is free again: it receives the k shard sizes)
  k_shard_off<<<(unsigned)((std::max<long long>(ng, k) + tpb - 1) / tpb), tpb, 0, st>>>(L.scan, (int)ng, k, L.off, L.cnt);
  std::vector<int32_t> rows((size_t)k);
  TS_CUDA(cudaMemcpyAsync(rows.data(), L.cnt, sizeof(int32_t) * (size_t)k, cudaMemcpyDeviceToHost, st));
  TS_CUDA(cudaStreamSynchronize(st));
  long long mx = 1;
  for (int r = 0; r < k; r++) mx = std::max<long long>(mx, rows[(size_t)r]);
  if (mx * (long long)k > 2147483647LL) return (int)cudaErrorInvalidValue;
  L.n_slots = mx;
  k_shard_slots<<<(unsigned)((ng * 32 + tpb - 1) / tpb), tpb, 0, st>>>(T.grp, L.off, (int)ng, k, L.n_slots, L.slot);
  TS_CUDA(cudaGetLastError());
  L.k = k;
  return 0;
}

int launch_shard_scatter(const DeviceTree& T, const ShardLayout& L, const float* gathered, const int32_t* gathered_cnt, float* acc,
                         float* pot, int32_t* n_pc, int32_t* n_pp, void* stream) {
  const int tpb = 256;
  k_shard_scatter<<<(unsigned)((T.n + tpb - 1) / tpb), tpb, 0, (cudaStream_t)stream>>>(
      reinterpret_cast<const float4*>(gathered), reinterpret_cast<const int2*>(gathered_cnt), L.slot, T.orig, T.n, acc, pot, n_pc, n_pp);
  return (int)cudaGetLastError();
}

}  // namespace tc

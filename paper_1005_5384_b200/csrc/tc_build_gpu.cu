// Device-side tree build (option "device_build").  The paper builds the octree on
// the host and names that the bottleneck for N >~ 1e6; this is the same
// construction O1-O4 of DESIGN.md §2 executed on the GPU, producing the SAME packed layout
// (tc_internal.h) directly in device memory, so tc_forces does not care who built the tree:
//   O1  bounding box (reduction), root cube on the host from 6 numbers, 63-bit Morton keys in fp64 with
//       explicitly rounded operations (bit-identical to the host builder's keys);
//   --  cub::DeviceRadixSort of (key, index) — a library primitive for a non-hot precondition step;
//   O2  breadth-first split, one level per step: per node 7 binary searches over its key range;
//   O3  tight boxes and fp64 moments bottom-up, level by level (leaves: direct sums over members,
//       nodes: parallel-axis shift of the children);  R20 boundary cubes;
//   O4  groups = cells with count <= N_group (or leaves) whose parent is larger, in Morton order;
//       cost-ordered schedule;  pack.
// Cells, boundaries and groups are identical to the host builder's; the order of particles inside a
// leaf (hence fp64 summation order, hence the last bit of some fp32 moments) may differ.
#include <cuda_runtime.h>

#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_reduce.cuh>
#include <cub/device/device_scan.cuh>
#include <cub/device/device_select.cuh>
#include <thrust/iterator/counting_iterator.h>

#include <cmath>
#include <cstdint>
#include <limits>
#include <algorithm>
#include <string>
#include <utility>
#include <vector>

#include "tc_internal.h"
#include "tc_lanes.h"

namespace tc {
namespace {

#define TCG_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { msg = std::string(#call) + ": " + cudaGetErrorString(e_); return e_ == cudaErrorMemoryAllocation ? TC_ENOMEM : TC_ECUDA; } } while (0)

struct Moments {          // fp64 moments + fp32-exact tight box of one cell
  double M, X[3], Q[6];
  float bmin[3], bmax[3];
};

__device__ __forceinline__ unsigned long long spread21(unsigned long long x) {
  x &= 0x1fffffull;
  x = (x | (x << 32)) & 0x1f00000000ffffull;
  x = (x | (x << 16)) & 0x1f0000ff0000ffull;
  x = (x | (x << 8)) & 0x100f00f00f00f00full;
  x = (x | (x << 4)) & 0x10c30c30c30c30c3ull;
  x = (x | (x << 2)) & 0x1249249249249249ull;
  return x;
}

struct Box6 { float lo[3], hi[3]; };
struct BoxOp {
  __device__ Box6 operator()(const Box6& a, const Box6& b) const {
    Box6 r;
#pragma unroll
    for (int k = 0; k < 3; k++) { r.lo[k] = fminf(a.lo[k], b.lo[k]); r.hi[k] = fmaxf(a.hi[k], b.hi[k]); }
    return r;
  }
};

// O1: per-block bounding boxes (finished on the host: <= 1024 partial boxes)
__global__ void __launch_bounds__(256) k_boxes(const float4* __restrict__ src, long long n, Box6* __restrict__ out) {
  __shared__ Box6 sh[8];
  Box6 b;
#pragma unroll
  for (int k = 0; k < 3; k++) { b.lo[k] = INFINITY; b.hi[k] = -INFINITY; }
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const float4 p = src[i];
    b.lo[0] = fminf(b.lo[0], p.x); b.hi[0] = fmaxf(b.hi[0], p.x);
    b.lo[1] = fminf(b.lo[1], p.y); b.hi[1] = fmaxf(b.hi[1], p.y);
    b.lo[2] = fminf(b.lo[2], p.z); b.hi[2] = fmaxf(b.hi[2], p.z);
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1)
#pragma unroll
    for (int k = 0; k < 3; k++) {
      b.lo[k] = fminf(b.lo[k], __shfl_xor_sync(0xffffffffu, b.lo[k], d));
      b.hi[k] = fmaxf(b.hi[k], __shfl_xor_sync(0xffffffffu, b.hi[k], d));
    }
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = b;
  __syncthreads();
  if (threadIdx.x == 0) {
    BoxOp op;
    for (int w = 1; w < 8; w++) b = op(b, sh[w]);
    out[blockIdx.x] = b;
  }
}

// O1: g_k = clamp(floor((x_k - org_k) * scale), 0, 2^21 - 1) in fp64, one rounding per operation
__global__ void k_keys(const float4* __restrict__ src, long long n, double ox, double oy, double oz, double scale,
                       unsigned long long* __restrict__ keys, unsigned int* __restrict__ idx) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float4 p = src[i];
  const double gmax = 2097151.0;
  const double vx = fmin(fmax(floor(__dmul_rn(__dsub_rn((double)p.x, ox), scale)), 0.0), gmax);
  const double vy = fmin(fmax(floor(__dmul_rn(__dsub_rn((double)p.y, oy), scale)), 0.0), gmax);
  const double vz = fmin(fmax(floor(__dmul_rn(__dsub_rn((double)p.z, oz), scale)), 0.0), gmax);
  keys[i] = (spread21((unsigned long long)vx) << 2) | (spread21((unsigned long long)vy) << 1) |
            spread21((unsigned long long)vz);
  idx[i] = (unsigned int)i;
}

// first position in [b, e) whose octant digit at `shift` is >= o
__device__ __forceinline__ int lower_octant(const unsigned long long* __restrict__ keys, int b, int e, int shift, unsigned o) {
  while (b < e) {
    const int m = b + ((e - b) >> 1);
    if (((keys[m] >> shift) & 7ull) < o) b = m + 1; else e = m;
  }
  return b;
}

// O2 pass 1: 8 lanes per node — lane o finds where octant o starts in the node's sorted key range (one binary
// search each, side by side), the 8 lanes count the non-empty octants (0 for leaves) and keep the bounds.
__global__ void k_count_children(const unsigned long long* __restrict__ keys, const int* __restrict__ c_begin,
                                 const int* __restrict__ c_count, int lb, int nl, int shift, int n_leaf, int* __restrict__ nch,
                                 int* __restrict__ bounds) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int node = t >> 3;
  const unsigned o = (unsigned)(t & 7);
  const bool valid = node < nl;
  const int c = lb + (valid ? node : 0);
  const int b = c_begin[c], e = b + c_count[c];
  const bool split = valid && c_count[c] > n_leaf;
  const int p0 = (o == 0 || !split) ? b : lower_octant(keys, b, e, shift, o);
  int p1 = __shfl_down_sync(0xffffffffu, p0, 1, 8);
  if (o == 7) p1 = e;
  const unsigned seg = 0xffu << ((threadIdx.x & 31) & ~7);
  const unsigned m = __ballot_sync(0xffffffffu, split && p1 > p0) & seg;
  if (!valid) return;
  bounds[t] = p0;
  if (o == 0) nch[node] = __popc(m);
}

// O2 pass 2: create the children (contiguous, octant order) from the kept bounds
__global__ void k_make_children(int* __restrict__ c_begin, int* __restrict__ c_count, int* __restrict__ c_first,
                                int* __restrict__ c_nchild, int* __restrict__ c_parent, int lb, int nl, int le,
                                const int* __restrict__ nch, const int* __restrict__ off, const int* __restrict__ bounds) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int node = t >> 3;
  const unsigned o = (unsigned)(t & 7);
  const bool valid = node < nl;
  const int c = lb + (valid ? node : 0);
  const int k = valid ? nch[node] : 0;
  const int e = c_begin[c] + c_count[c];
  const int p0 = valid ? bounds[t] : 0;
  int p1 = __shfl_down_sync(0xffffffffu, p0, 1, 8);
  if (o == 7) p1 = e;
  const bool nonempty = k > 0 && p1 > p0;
  const unsigned seg_shift = (threadIdx.x & 31) & ~7;
  const unsigned m = (__ballot_sync(0xffffffffu, nonempty) >> seg_shift) & 0xffu;
  if (!valid) return;
  if (o == 0) { c_nchild[c] = k; c_first[c] = k ? le + off[node] : -1; }
  if (nonempty) {
    const int j = le + off[node] + __popc(m & ((1u << o) - 1u));
    c_begin[j] = p0; c_count[j] = p1 - p0; c_parent[j] = c;
  }
}

// O3: tight box + fp64 moments of the cells of one level (children are one level deeper and done)
__global__ void k_moments(const float4* __restrict__ src, const unsigned int* __restrict__ idx, const int* __restrict__ c_begin,
                          const int* __restrict__ c_count, const int* __restrict__ c_first, const int* __restrict__ c_nchild,
                          int lb, int nl, Moments* __restrict__ mom) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nl) return;
  const int c = lb + t;
  Moments P;
  double M = 0.0, S[3] = {0.0, 0.0, 0.0};
  float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
  double Q[6] = {0, 0, 0, 0, 0, 0};
  if (c_nchild[c] == 0) {
    const int pb = c_begin[c], pe = pb + c_count[c];
    for (int j = pb; j < pe; j++) {
      const float4 p = src[idx[j]];
      const double m = (double)p.w;
      mn[0] = fminf(mn[0], p.x); mx[0] = fmaxf(mx[0], p.x);
      mn[1] = fminf(mn[1], p.y); mx[1] = fmaxf(mx[1], p.y);
      mn[2] = fminf(mn[2], p.z); mx[2] = fmaxf(mx[2], p.z);
      S[0] += m * (double)p.x; S[1] += m * (double)p.y; S[2] += m * (double)p.z;
      M += m;
    }
    for (int k = 0; k < 3; k++) P.X[k] = (M > 0.0) ? S[k] / M : ((double)mn[k] + (double)mx[k]) / 2.0;  // R19
    for (int j = pb; j < pe; j++) {
      const float4 p = src[idx[j]];
      const double m = (double)p.w;
      const double yx = (double)p.x - P.X[0], yy = (double)p.y - P.X[1], yz = (double)p.z - P.X[2];
      const double y2 = yx * yx + yy * yy + yz * yz;
      Q[0] += m * (3.0 * yx * yx - y2); Q[1] += m * (3.0 * yy * yy - y2); Q[2] += m * (3.0 * yz * yz - y2);
      Q[3] += m * (3.0 * yx * yy); Q[4] += m * (3.0 * yx * yz); Q[5] += m * (3.0 * yy * yz);
    }
  } else {
    const int f = c_first[c], l = f + c_nchild[c];
    for (int ch = f; ch < l; ch++) {
      const Moments& C = mom[ch];
      for (int k = 0; k < 3; k++) {
        mn[k] = fminf(mn[k], C.bmin[k]); mx[k] = fmaxf(mx[k], C.bmax[k]);
        S[k] += C.M * C.X[k];
      }
      M += C.M;
    }
    for (int k = 0; k < 3; k++) P.X[k] = (M > 0.0) ? S[k] / M : ((double)mn[k] + (double)mx[k]) / 2.0;
    for (int ch = f; ch < l; ch++) {
      const Moments& C = mom[ch];
      const double dx = C.X[0] - P.X[0], dy = C.X[1] - P.X[1], dz = C.X[2] - P.X[2];
      const double d2 = dx * dx + dy * dy + dz * dz;
      Q[0] += C.Q[0] + C.M * (3.0 * dx * dx - d2); Q[1] += C.Q[1] + C.M * (3.0 * dy * dy - d2);
      Q[2] += C.Q[2] + C.M * (3.0 * dz * dz - d2);
      Q[3] += C.Q[3] + C.M * (3.0 * dx * dy); Q[4] += C.Q[4] + C.M * (3.0 * dx * dz);
      Q[5] += C.Q[5] + C.M * (3.0 * dy * dz);
    }
  }
  P.M = M;
  for (int k = 0; k < 3; k++) { P.bmin[k] = mn[k]; P.bmax[k] = mx[k]; }
  for (int k = 0; k < 6; k++) P.Q[k] = Q[k];
  mom[c] = P;
}

// pack the per-cell arrays of the layout in tc_internal.h (+ the inspection arrays link / q6)
__global__ void k_pack_cells(const Moments* __restrict__ mom, const int* __restrict__ c_begin, const int* __restrict__ c_count,
                             const int* __restrict__ c_first, const int* __restrict__ c_nchild, const int* __restrict__ c_parent,
                             int nc, int n_group, float4* __restrict__ bnd, float4* __restrict__ xm, float4* __restrict__ q0,
                             float4* __restrict__ q1, int4* __restrict__ link, float* __restrict__ q6) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= nc) return;
  const Moments P = mom[c];
  // boundary cube, FP32 form R20: centre rounded to nearest, reach from the rounded centre rounded up
  float b[3];
  double reach = 0.0;
#pragma unroll
  for (int k = 0; k < 3; k++) {
    const double lo = (double)P.bmin[k], hi = (double)P.bmax[k];
    b[k] = (float)(0.5 * (lo + hi));
    reach = fmax(reach, fmax(hi - (double)b[k], (double)b[k] - lo));
  }
  float h = __double2float_ru(reach);
  const bool leaf = c_nchild[c] == 0;
  bnd[c] = make_float4(b[0], b[1], b[2], leaf ? -h : h);
  xm[c] = make_float4((float)P.X[0], (float)P.X[1], (float)P.X[2], (float)P.M);
  q0[c] = make_float4(-(float)P.Q[0], -(float)P.Q[1], -(float)P.Q[2], -(float)P.Q[3]);   // -Q: see tc_kernels.cu
  const int la = leaf ? c_begin[c] : c_first[c], lb = leaf ? c_count[c] : c_nchild[c];
  q1[c] = make_float4(-(float)P.Q[4], -(float)P.Q[5], __int_as_float(la), __int_as_float(lb));
  link[c] = make_int4(leaf ? -1 : c_first[c], c_nchild[c], c_begin[c], c_count[c]);
#pragma unroll
  for (int k = 0; k < 6; k++) q6[6 * (size_t)c + k] = (float)P.Q[k];
}

// O4: a group is a cell that is small enough (or a leaf) while its parent is not
__global__ void k_flag_groups(const int* __restrict__ c_count, const int* __restrict__ c_nchild, const int* __restrict__ c_parent,
                              int nc, int n_group, unsigned char* __restrict__ is_group, unsigned int* __restrict__ n_leaves) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= nc) return;
  const bool leaf = c_nchild[c] == 0;
  const bool small = c_count[c] <= n_group || leaf;
  bool parent_small = false;
  if (c > 0) { const int p = c_parent[c]; parent_small = c_count[p] <= n_group || c_nchild[p] == 0; }
  is_group[c] = (small && !parent_small) ? 1 : 0;
  if (leaf) atomicAdd(n_leaves, 1u);
}

__global__ void k_pack_particles(const float4* __restrict__ src, const unsigned int* __restrict__ idx, long long n,
                                 float4* __restrict__ part, int* __restrict__ orig) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const unsigned int i = idx[t];
  part[t] = src[i];
  orig[t] = (int)i;
}

// group records: key for the Morton order = first body; cost class for the schedule
__constant__ LaneTable c_lanes_build = LaneTable();   // the kernel's lane mapping (tc_lanes.h): cost model of the schedule
__global__ void k_group_keys(const int* __restrict__ gcell, int ng, const int* __restrict__ c_begin, const int* __restrict__ c_count,
                             unsigned int* __restrict__ first_body, unsigned int* __restrict__ cls_key, int shift) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= ng) return;
  const int c = gcell[g];
  first_body[g] = (unsigned int)c_begin[c];
  const int cnt = c_count[c];
  cls_key[g] = (unsigned int)(kMaxCostClass - group_cost_class(c_lanes_build, cnt, shift));   // ascending key = descending cost
}

__global__ void k_iota(unsigned int* a, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) a[i] = (unsigned int)i;
}

__global__ void k_pack_groups(const int* __restrict__ gcell_sorted, const unsigned int* __restrict__ sched, int ng,
                              const int* __restrict__ c_begin, const int* __restrict__ c_count,
                              const Moments* __restrict__ mom, int4* __restrict__ grp, float4* __restrict__ gbox) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= ng) return;
  const int c = gcell_sorted[g];
  grp[g] = make_int4(c, c_begin[c], c_count[c], (int)sched[g]);
  // variant R23: half extents of the tight box about the fp32 centre, per axis, rounded up
  float e[3];
#pragma unroll
  for (int k = 0; k < 3; k++) {
    const double lo = (double)mom[c].bmin[k], hi = (double)mom[c].bmax[k];
    const float bk = (float)(0.5 * (lo + hi));
    e[k] = __double2float_ru(fmax(hi - (double)bk, (double)bk - lo));
  }
  gbox[g] = make_float4(e[0], e[1], e[2], 0.f);
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }
inline unsigned blocks(long long n, int t = 256) { return (unsigned)((n + t - 1) / t); }

}  // namespace

// tc_set_particles with device inputs in device-build mode: interleave + validate on the device
__global__ void k_pack_src(const float* __restrict__ pos, const float* __restrict__ mass, long long n, float4* __restrict__ out,
                           unsigned int* __restrict__ flags) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2], m = mass[i];
  out[i] = make_float4(x, y, z, m);
  if (!(isfinite(x) && isfinite(y) && isfinite(z))) atomicOr(flags, 1u);
  if (!(isfinite(m) && m >= 0.f)) atomicOr(flags, 2u);
}

int pack_src_device(const float* pos, const float* mass, int64_t n, float4* out, unsigned int* flags, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = cudaMemsetAsync(flags, 0, sizeof(unsigned int), st);
  if (e != cudaSuccess) return (int)e;
  k_pack_src<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(pos, mass, n, out, flags);
  return (int)cudaGetLastError();
}

// ---- scratch management -------------------------------------------------------------------------
template <typename T>
static int grow(T*& p, size_t& cap, size_t need, bool keep, cudaStream_t st, std::string& msg) {
  if (cap >= need) return TC_OK;
  size_t ncap = need + need / 4 + 256;
  T* q = nullptr;
  TCG_CUDA(cudaMalloc((void**)&q, sizeof(T) * ncap));
  if (keep && p && cap) TCG_CUDA(cudaMemcpyAsync(q, p, sizeof(T) * cap, cudaMemcpyDeviceToDevice, st));
  if (p) { TCG_CUDA(cudaStreamSynchronize(st)); cudaFree(p); }
  p = q; cap = ncap;
  return TC_OK;
}
#define TCG_GROW(ptr, cap, need, keep) do { const int rc_ = grow(ptr, cap, (size_t)(need), keep, st, msg); if (rc_ != TC_OK) return rc_; } while (0)

void DeviceBuildScratch::release() {
  void* ptrs[] = {keys, keys_alt, idx, idx_alt, cub_tmp, c_begin, c_count, c_first, c_nchild, c_parent, nch, off, mom,
                  is_group, gcell, gcell_sorted, gkey, gkey_alt, gval, gval_alt, boxes, small, link, q6, bounds};
  for (void* p : ptrs) cudaFree(p);
  *this = DeviceBuildScratch();
}

int build_device_tree(const float4* src, int64_t n, int n_leaf, int n_group, DeviceBuildScratch& S, void** d_tree,
                      size_t* d_tree_cap, HostTree& T, DeviceTree& D, void* stream, std::string& msg) {
  cudaStream_t st = (cudaStream_t)stream;
  if (n < 1 || n_leaf < 1 || n_group < 1) { msg = "build: n, n_leaf, n_group must be >= 1"; return TC_EINVAL; }
  if (n > 0x7fffffffLL) { msg = "build: n must be < 2^31"; return TC_EINVAL; }
  T.n = n; T.n_leaf = n_leaf; T.n_group = n_group;

  // ---- O1: bounding box -> root cube (host arithmetic on 6 numbers, same as tc_build.cpp)
  const int nb = (int)std::min<long long>(1024, (n + 255) / 256);
  TCG_GROW(S.boxes, S.cap_boxes, sizeof(Box6) * 1024, false);
  k_boxes<<<nb, 256, 0, st>>>(src, n, (Box6*)S.boxes);
  Box6 hb[1024];
  TCG_CUDA(cudaMemcpyAsync(hb, S.boxes, sizeof(Box6) * nb, cudaMemcpyDeviceToHost, st));
  TCG_CUDA(cudaStreamSynchronize(st));
  double lo[3], hi[3];
  for (int k = 0; k < 3; k++) { lo[k] = std::numeric_limits<double>::infinity(); hi[k] = -lo[k]; }
  for (int b = 0; b < nb; b++)
    for (int k = 0; k < 3; k++) { lo[k] = std::min(lo[k], (double)hb[b].lo[k]); hi[k] = std::max(hi[k], (double)hb[b].hi[k]); }
  double ext = 0.0;
  for (int k = 0; k < 3; k++) ext = std::max(ext, hi[k] - lo[k]);
  double side = ext * (1.0 + std::ldexp(1.0, -20));
  if (side == 0.0) side = 1.0;
  double org[3];
  for (int k = 0; k < 3; k++) org[k] = (lo[k] + hi[k]) / 2.0 - side / 2.0;
  const double scale = std::ldexp(1.0, 21) / side;

  // ---- keys + sort
  TCG_GROW(S.keys, S.cap_keys, n, false); TCG_GROW(S.keys_alt, S.cap_keys_alt, n, false);
  TCG_GROW(S.idx, S.cap_idx, n, false);   TCG_GROW(S.idx_alt, S.cap_idx_alt, n, false);
  k_keys<<<blocks(n), 256, 0, st>>>(src, n, org[0], org[1], org[2], scale, S.keys, S.idx);
  {
    cub::DoubleBuffer<unsigned long long> kb(S.keys, S.keys_alt);
    cub::DoubleBuffer<unsigned int> vb(S.idx, S.idx_alt);
    size_t need = 0;
    TCG_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, need, kb, vb, (int)n, 0, 63, st));
    TCG_GROW(S.cub_tmp, S.cap_tmp, need, false);
    TCG_CUDA(cub::DeviceRadixSort::SortPairs(S.cub_tmp, need, kb, vb, (int)n, 0, 63, st));
    if (kb.Current() != S.keys) { std::swap(S.keys, S.keys_alt); std::swap(S.cap_keys, S.cap_keys_alt); }
    if (vb.Current() != S.idx) { std::swap(S.idx, S.idx_alt); std::swap(S.cap_idx, S.cap_idx_alt); }
  }

  // ---- O2: breadth-first split
  size_t cap0 = (size_t)std::max<int64_t>(1024, n / 2);
  TCG_GROW(S.c_begin, S.cap_cbegin, cap0, false); TCG_GROW(S.c_count, S.cap_ccount, cap0, false);
  TCG_GROW(S.c_first, S.cap_cfirst, cap0, false); TCG_GROW(S.c_nchild, S.cap_cnchild, cap0, false);
  TCG_GROW(S.c_parent, S.cap_cparent, cap0, false);
  {
    const int root[5] = {0, (int)n, -1, 0, -1};
    TCG_CUDA(cudaMemcpyAsync(S.c_begin, &root[0], 4, cudaMemcpyHostToDevice, st));
    TCG_CUDA(cudaMemcpyAsync(S.c_count, &root[1], 4, cudaMemcpyHostToDevice, st));
    TCG_CUDA(cudaMemcpyAsync(S.c_first, &root[2], 4, cudaMemcpyHostToDevice, st));
    TCG_CUDA(cudaMemcpyAsync(S.c_nchild, &root[3], 4, cudaMemcpyHostToDevice, st));
    TCG_CUDA(cudaMemcpyAsync(S.c_parent, &root[4], 4, cudaMemcpyHostToDevice, st));
    TCG_CUDA(cudaStreamSynchronize(st));     // `root` leaves scope
  }
  std::vector<int64_t> level_start;
  level_start.push_back(0);
  int64_t lb = 0, le = 1;
  int level = 0;
  while (true) {
    level_start.push_back(le);
    const int64_t nl = le - lb;
    if (level == kMaxLevel) {                  // level-21 cells are leaves whatever their count (R7)
      TCG_CUDA(cudaMemsetAsync(S.c_nchild + lb, 0, sizeof(int) * (size_t)nl, st));
      break;
    }
    const int shift = 3 * (kMaxLevel - 1 - level);
    TCG_GROW(S.nch, S.cap_nch, nl, false); TCG_GROW(S.off, S.cap_off, nl, false); TCG_GROW(S.bounds, S.cap_bounds, 8 * nl, false);
    k_count_children<<<blocks(8 * nl), 256, 0, st>>>(S.keys, S.c_begin, S.c_count, (int)lb, (int)nl, shift, n_leaf, S.nch, S.bounds);
    size_t need = 0;
    TCG_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, need, S.nch, S.off, (int)nl, st));
    TCG_GROW(S.cub_tmp, S.cap_tmp, need, false);
    TCG_CUDA(cub::DeviceScan::ExclusiveSum(S.cub_tmp, need, S.nch, S.off, (int)nl, st));
    int last[2];
    TCG_CUDA(cudaMemcpyAsync(&last[0], S.off + (nl - 1), 4, cudaMemcpyDeviceToHost, st));
    TCG_CUDA(cudaMemcpyAsync(&last[1], S.nch + (nl - 1), 4, cudaMemcpyDeviceToHost, st));
    TCG_CUDA(cudaStreamSynchronize(st));
    const int64_t total = (int64_t)last[0] + last[1];
    const int64_t new_e = le + total;
    if (new_e > (int64_t)0x0fffffff) { msg = "build: more than 2^28 cells"; return TC_EINVAL; }
    if (total > 0) {
      TCG_GROW(S.c_begin, S.cap_cbegin, new_e, true); TCG_GROW(S.c_count, S.cap_ccount, new_e, true);
      TCG_GROW(S.c_first, S.cap_cfirst, new_e, true); TCG_GROW(S.c_nchild, S.cap_cnchild, new_e, true);
      TCG_GROW(S.c_parent, S.cap_cparent, new_e, true);
    }
    k_make_children<<<blocks(8 * nl), 256, 0, st>>>(S.c_begin, S.c_count, S.c_first, S.c_nchild, S.c_parent, (int)lb, (int)nl,
                                                     (int)le, S.nch, S.off, S.bounds);
    if (total == 0) break;
    lb = le; le = new_e; level++;
  }
  const int64_t nc = le;
  const int n_levels = (int)level_start.size() - 1;
  T.n_cells = nc;
  T.depth = (int32_t)level_start.size() - 2;

  // ---- O3: moments bottom-up
  TCG_GROW(S.mom, S.cap_mom, sizeof(Moments) * (size_t)nc, false);
  for (int L = n_levels - 1; L >= 0; L--) {
    const int64_t b = level_start[L], e = level_start[L + 1];
    k_moments<<<blocks(e - b, 128), 128, 0, st>>>(src, S.idx, S.c_begin, S.c_count, S.c_first, S.c_nchild, (int)b, (int)(e - b),
                                                  (Moments*)S.mom);
  }

  // ---- O4: groups (flag, compact, Morton order, schedule)
  TCG_GROW(S.is_group, S.cap_isg, nc, false);
  TCG_GROW(S.small, S.cap_small, 8, false);
  TCG_CUDA(cudaMemsetAsync(S.small, 0, sizeof(unsigned int) * 8, st));
  k_flag_groups<<<blocks(nc), 256, 0, st>>>(S.c_count, S.c_nchild, S.c_parent, (int)nc, n_group, S.is_group, S.small);
  TCG_GROW(S.gcell, S.cap_gcell, nc, false);
  {
    thrust::counting_iterator<int> it(0);
    size_t need = 0;
    TCG_CUDA(cub::DeviceSelect::Flagged(nullptr, need, it, S.is_group, S.gcell, (int*)(S.small + 1), (int)nc, st));
    TCG_GROW(S.cub_tmp, S.cap_tmp, need, false);
    TCG_CUDA(cub::DeviceSelect::Flagged(S.cub_tmp, need, it, S.is_group, S.gcell, (int*)(S.small + 1), (int)nc, st));
  }
  unsigned int hsmall[2];
  TCG_CUDA(cudaMemcpyAsync(hsmall, S.small, sizeof(hsmall), cudaMemcpyDeviceToHost, st));
  TCG_CUDA(cudaStreamSynchronize(st));
  T.n_leaves = hsmall[0];
  const int64_t ng = hsmall[1];
  T.n_groups = ng;

  // Morton order of the groups = ascending first body
  TCG_GROW(S.gkey, S.cap_gkey, ng, false); TCG_GROW(S.gkey_alt, S.cap_gkeya, ng, false);
  TCG_GROW(S.gval, S.cap_gval, ng, false); TCG_GROW(S.gval_alt, S.cap_gvala, ng, false);
  TCG_GROW(S.gcell_sorted, S.cap_gcells, ng, false);
  {
    // (1) sort the group cells by first body: keys = first body, values = cell id
    k_group_keys<<<blocks(ng), 256, 0, st>>>(S.gcell, (int)ng, S.c_begin, S.c_count, S.gkey, S.gval, schedule_class_shift((long long)ng));
    cub::DoubleBuffer<unsigned int> kb(S.gkey, S.gkey_alt);
    cub::DoubleBuffer<int> vb(S.gcell, S.gcell_sorted);
    size_t need = 0;
    TCG_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, need, kb, vb, (int)ng, 0, 32, st));
    TCG_GROW(S.cub_tmp, S.cap_tmp, need, false);
    TCG_CUDA(cub::DeviceRadixSort::SortPairs(S.cub_tmp, need, kb, vb, (int)ng, 0, 32, st));
    if (vb.Current() != S.gcell_sorted) { std::swap(S.gcell, S.gcell_sorted); std::swap(S.cap_gcell, S.cap_gcells); }
    if (kb.Current() != S.gkey) { std::swap(S.gkey, S.gkey_alt); std::swap(S.cap_gkey, S.cap_gkeya); }
    // (2) schedule: stable sort of the Morton-ordered group indices by descending cost class
    k_group_keys<<<blocks(ng), 256, 0, st>>>(S.gcell_sorted, (int)ng, S.c_begin, S.c_count, S.gkey_alt, S.gkey, schedule_class_shift((long long)ng));
    k_iota<<<blocks(ng), 256, 0, st>>>(S.gval, (int)ng);
    cub::DoubleBuffer<unsigned int> kb2(S.gkey, S.gkey_alt);
    cub::DoubleBuffer<unsigned int> vb2(S.gval, S.gval_alt);
    TCG_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, need, kb2, vb2, (int)ng, 0, 21, st));
    TCG_GROW(S.cub_tmp, S.cap_tmp, need, false);
    TCG_CUDA(cub::DeviceRadixSort::SortPairs(S.cub_tmp, need, kb2, vb2, (int)ng, 0, 21, st));
    if (vb2.Current() != S.gval) { std::swap(S.gval, S.gval_alt); std::swap(S.cap_gval, S.cap_gvala); }
    if (kb2.Current() != S.gkey) { std::swap(S.gkey, S.gkey_alt); std::swap(S.cap_gkey, S.cap_gkeya); }
  }

  // ---- pack: the layout of tc_internal.h, written in place on the device
  PackedLayout& Y = T.lay;
  size_t off = 0;
  Y.off_bnd = off;  off = align256(off + sizeof(float4) * (size_t)nc);
  Y.off_xm = off;   off = align256(off + sizeof(float4) * (size_t)nc);
  Y.off_q0 = off;   off = align256(off + sizeof(float4) * (size_t)nc);
  Y.off_q1 = off;   off = align256(off + sizeof(float4) * (size_t)nc);
  Y.off_part = off; off = align256(off + sizeof(float4) * (size_t)n);
  Y.off_orig = off; off = align256(off + sizeof(int32_t) * (size_t)n);
  Y.off_grp = off;  off = align256(off + sizeof(int4) * (size_t)ng);
  Y.off_gbox = off; off = align256(off + sizeof(float4) * (size_t)ng);
  Y.bytes = off;
  if (*d_tree_cap < Y.bytes) {
    TCG_CUDA(cudaStreamSynchronize(st));
    cudaFree(*d_tree); *d_tree = nullptr; *d_tree_cap = 0;
    const size_t cap = Y.bytes + Y.bytes / 8;
    TCG_CUDA(cudaMalloc(d_tree, cap));
    *d_tree_cap = cap;
  }
  char* base = (char*)*d_tree;
  D.bnd = (const float4*)(base + Y.off_bnd); D.xm = (const float4*)(base + Y.off_xm);
  D.q0 = (const float4*)(base + Y.off_q0);   D.q1 = (const float4*)(base + Y.off_q1);
  D.part = (const float4*)(base + Y.off_part); D.orig = (const int32_t*)(base + Y.off_orig);
  D.grp = (const int4*)(base + Y.off_grp);
  D.gbox = (const float4*)(base + Y.off_gbox);
  D.n = n; D.n_cells = nc; D.n_groups = ng;
  TCG_GROW(S.link, S.cap_link, nc, false);
  TCG_GROW(S.q6, S.cap_q6, 6 * (size_t)nc, false);
  k_pack_cells<<<blocks(nc), 256, 0, st>>>((const Moments*)S.mom, S.c_begin, S.c_count, S.c_first, S.c_nchild, S.c_parent, (int)nc,
                                           n_group, (float4*)D.bnd, (float4*)D.xm, (float4*)D.q0, (float4*)D.q1, S.link, S.q6);
  k_pack_particles<<<blocks(n), 256, 0, st>>>(src, S.idx, n, (float4*)D.part, (int*)D.orig);
  // after the two sorts: gcell_sorted = group cells in Morton order, gval = schedule
  k_pack_groups<<<blocks(ng), 256, 0, st>>>(S.gcell_sorted, S.gval, (int)ng, S.c_begin, S.c_count, (const Moments*)S.mom,
                                            (int4*)D.grp, (float4*)D.gbox);
  TCG_CUDA(cudaGetLastError());
  TCG_CUDA(cudaStreamSynchronize(st));
  return TC_OK;
}

}  // namespace tc

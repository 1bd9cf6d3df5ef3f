// Internal declarations shared by the host builder (tc_build.cpp), the kernels
// (tc_kernels.cu) and the C ABI (tc_api.cpp).  Not installed; include/tc.h is the
// public boundary.  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include <vector_functions.h>  // float4 / int4 / make_float4 (CUDA toolkit header, host-safe)

#include "../../include/tc.h"
#include "../../include/tc_bench.h"

namespace tc {

constexpr int kMaxLevel = 21;  // 3 x 21 = 63-bit Morton keys (R7)

// Packed tree in ONE host buffer (pinned when a device exists) that tc_build moves
// with one cudaMemcpyAsync.  All section offsets are multiples
// of 256 bytes.  Per cell c (cells in breadth-first order, children contiguous):
//   bnd [c] = (bx, by, bz, h)        boundary cube, Fig. 1; sign bit of h set <=> leaf
//   xm  [c] = (X, Y, Z, M)           centre of mass, mass
//   q0  [c] = -(Qxx, Qyy, Qzz, Qxy)  traceless quadrupole about X, NEGATED (see tc_kernels.cu)
//   q1  [c] = (-Qxz, -Qyz, a, b)       a,b int bits: node -> (first_child, n_child)
//                                                 leaf -> (first_body,  n_body)
//   part[i] = (x, y, z, m)           particles in tree (Morton) order
//   orig[i] = caller's index of tree-order particle i
//   grp [g] = (cell, first_body, n_body, sched)  groups in Morton order; sched = index of the
//             g-th group to RUN (costly groups first, tc_build.cpp)
//   gbox[g] = (ex, ey, ez, 0)       half extents of the group's TIGHT box about bnd[cell].xyz, rounded up
//             (variant R23, option "group_box"; max(ex,ey,ez) == |bnd[cell].w|)
struct PackedLayout {
  size_t off_bnd = 0, off_xm = 0, off_q0 = 0, off_q1 = 0, off_part = 0, off_orig = 0, off_grp = 0, off_gbox = 0;
  size_t bytes = 0;
};

// Grow-only scratch of the host builder, kept between builds so that a rebuild (every step of a
// simulation) does not fault ~60 MB of fresh pages in again.  Contents are undefined between builds.
struct HostScratch {
  void* buf[3] = {nullptr, nullptr, nullptr};
  size_t cap[3] = {0, 0, 0};
  void* get(int k, size_t bytes);  // >= bytes of uninitialised storage, nullptr on failure
  // per-cell arrays of the breadth-first split and the group list: cleared, not freed, between builds
  std::vector<int32_t> c_begin, c_count, c_first_child, c_nchild, nch, groups, bounds;
  HostScratch() = default;
  HostScratch(const HostScratch&) = delete;
  HostScratch& operator=(const HostScratch&) = delete;
  ~HostScratch();
};

struct HostTree {
  int64_t n = 0;
  int32_t n_leaf = 0, n_group = 0;
  int64_t n_cells = 0, n_leaves = 0, n_groups = 0;
  int32_t depth = 0;
  // link per cell (host inspection, tc_get_tree): first_child, n_child, first_body, n_body
  std::vector<int32_t> link;
  std::vector<float> q6;  // unpacked quadrupole for tc_get_tree [n_cells,6]
  PackedLayout lay;
  void* packed = nullptr;  // lay.bytes, owned by the ctx (pinned or malloc)
  size_t packed_cap = 0;
  bool packed_pinned = false;
  HostScratch scratch;     // Morton keys, sort elements (2x) and per-cell moments of build_host_tree
};

// Host builder (tc_build.cpp).  xyzm [n] = (x, y, z, m) host fp32, caller's order.  Allocates/reuses
// T.packed through alloc(bytes) (returns nullptr on failure).  Returns TC_OK or an
// error code with msg set.
typedef void* (*PackedAlloc)(void* user, size_t bytes);
int build_host_tree(const float4* xyzm, int64_t n, int n_leaf, int n_group,
                    HostTree& T, PackedAlloc alloc, void* alloc_user, std::string& msg,
                    const float* bbox6 = nullptr /* per-axis min (0-2), max (3-5) of xyzm if the caller has them */);

// Device-side view handed to the kernels (tc_kernels.cu).
struct DeviceTree {
  const float4* bnd = nullptr;
  const float4* xm = nullptr;
  const float4* q0 = nullptr;
  const float4* q1 = nullptr;
  const float4* part = nullptr;
  const int32_t* orig = nullptr;
  const int4* grp = nullptr;
  const float4* gbox = nullptr;
  int64_t n = 0, n_cells = 0, n_groups = 0;
};

// Device counters written by the force kernel (one struct, zeroed before launch).
struct DeviceCounters {
  unsigned long long n_pc_total;
  unsigned long long n_pp_total;
  unsigned long long n_tests_total;
  unsigned long long n_spills;
  unsigned long long n_opened_total;
  unsigned int next_group;  // dynamic work counter (persistent warps)
  unsigned int overflow;    // != 0: a spill stack overflowed -> TC_EOVERFLOW
};

struct ForceLaunch {
  float theta = 0.f, eps = 0.f;
  float* acc = nullptr;       // device [n,3] caller order
  float* pot = nullptr;       // device [n] caller order or nullptr
  int32_t* n_pc = nullptr;    // device [n] caller order
  int32_t* n_pp = nullptr;    // device [n] caller order
  DeviceCounters* counters = nullptr;
  uint32_t* spill = nullptr;  // device [n_warps_total * spill_cap]
  int spill_cap = 0;
  int stack_smem = 256;
  int flags = 0;              // bit 0: walk_only (measurement aid), bit 1: COM opening rule (R21), bit 2: monopole only (R22), bit 3: group = its tight box (R23)
  int n_sm = 148;
  int max_grid = 0;           // CTAs the spill buffer has room for (0: no limit)
  int shard_rank = 0, shard_count = 1;   // this launch runs schedule positions rank, rank + count, ... (fused kernel)
  // shard of a multi-GPU evaluation: compact rows instead of the caller's order (all three set, or none)
  float* shard_out4 = nullptr;           // device [n_slots,4]  (ax, ay, az, phi)
  int32_t* shard_cnt2 = nullptr;         // device [n_slots,2]  (n_pc, n_pp) or nullptr
  const int32_t* shard_off = nullptr;    // device [n_groups] by schedule position: first row of the group in its rank's shard
};

// Layout of the shards of ONE evaluation over k ranks: rank r evaluates the schedule positions
// r, r + k, ...; its rows are its groups in that order, particles in tree order inside a group.
//   off [i]  (i = schedule position)   first row of group sched[i] inside the shard of rank i % k
//   slot[t]  (t = tree-order particle) row of particle t in the all-gathered buffer [k, n_slots]: (i % k) n_slots + off[i] + ...
// Scratch owned by the context, grow-only.
struct ShardLayout {
  int32_t *off = nullptr, *slot = nullptr, *cnt = nullptr, *scan = nullptr;
  size_t cap_off = 0, cap_slot = 0, cap_cnt = 0, cap_scan = 0;
  char* tmp = nullptr; size_t cap_tmp = 0;
  int k = 0;                 // the layout was built for this shard_count (0: none)
  long long n_slots = 0;     // rows per rank in the gathered buffer = max over ranks of the particles a rank evaluates
  void release();
};
// builds L for k ranks on `stream` (synchronises it once to read the k shard sizes).  cudaError_t as int.
int build_shard_layout(const DeviceTree& T, int k, ShardLayout& L, void* stream);
// gathered [k, n_slots, 4] (+ gathered_cnt [k, n_slots, 2] or nullptr) -> acc [n,3], pot [n] or nullptr, n_pc / n_pp [n] or nullptr,
// all DEVICE, in the caller's order.  cudaError_t as int.
int launch_shard_scatter(const DeviceTree& T, const ShardLayout& L, const float* gathered, const int32_t* gathered_cnt, float* acc,
                         float* pot, int32_t* n_pc, int32_t* n_pp, void* stream);

// Launches the fused walk+evaluate kernel on `stream` (a cudaStream_t).  Returns a
// cudaError_t as int (0 = success).  Defined in tc_kernels.cu.
// Two builds of the same kernel source with different launch configurations (tc_kernels.cu / tc_kernels_dense.cu).
namespace sparse {
int launch_forces(const DeviceTree& T, const ForceLaunch& L, void* stream);
int forces_total_warps(int n_sm, int stack_smem);   // warps the persistent grid runs (for sizing the spill buffer)
int forces_warps_per_cta();
}  // namespace sparse
namespace dense {
int launch_forces(const DeviceTree& T, const ForceLaunch& L, void* stream);
int forces_total_warps(int n_sm, int stack_smem);
int forces_warps_per_cta();
}  // namespace dense
// Two-pass variant (option "two_pass"): global interaction lists and their scratch, owned by the context.
struct TwoPassScratch {
  unsigned long long *cnt_c = nullptr, *cnt_l = nullptr, *off_c = nullptr, *off_l = nullptr;
  size_t cap_cnt_c = 0, cap_cnt_l = 0, cap_off_c = 0, cap_off_l = 0;
  int* leaf_bodies = nullptr;  size_t cap_lb = 0;
  int* cells = nullptr;        size_t cap_cells = 0;
  int2* leaves = nullptr;      size_t cap_leaves = 0;
  char* tmp = nullptr;         size_t cap_tmp = 0;
  void* ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // cudaEvent_t
  long long n_list_cells = 0, n_list_leaves = 0;
  void release();
};
// count -> scan -> write lists -> node kernel -> leaf kernel.  cudaError_t as int.
int launch_forces_two_pass(const DeviceTree& T, const ForceLaunch& L, TwoPassScratch& S, void* stream);
int two_pass_times(const TwoPassScratch& S, float ms[4]);
// Scratch of the device-side builder (tc_build_gpu.cu); grow-only, owned by the context.
struct DeviceBuildScratch {
  unsigned long long *keys = nullptr, *keys_alt = nullptr;  size_t cap_keys = 0, cap_keys_alt = 0;
  unsigned int *idx = nullptr, *idx_alt = nullptr;          size_t cap_idx = 0, cap_idx_alt = 0;
  char* cub_tmp = nullptr;                                   size_t cap_tmp = 0;
  int *c_begin = nullptr, *c_count = nullptr, *c_first = nullptr, *c_nchild = nullptr, *c_parent = nullptr;
  size_t cap_cbegin = 0, cap_ccount = 0, cap_cfirst = 0, cap_cnchild = 0, cap_cparent = 0;
  int *nch = nullptr, *off = nullptr;                        size_t cap_nch = 0, cap_off = 0;
  int* bounds = nullptr;                                     size_t cap_bounds = 0;  // 8 octant starts per node of a level
  char* mom = nullptr;                                       size_t cap_mom = 0;     // Moments[]
  unsigned char* is_group = nullptr;                         size_t cap_isg = 0;
  int *gcell = nullptr, *gcell_sorted = nullptr;             size_t cap_gcell = 0, cap_gcells = 0;
  unsigned int *gkey = nullptr, *gkey_alt = nullptr, *gval = nullptr, *gval_alt = nullptr;
  size_t cap_gkey = 0, cap_gkeya = 0, cap_gval = 0, cap_gvala = 0;
  char* boxes = nullptr;                                     size_t cap_boxes = 0;
  unsigned int* small = nullptr;                             size_t cap_small = 0;   // counters
  int4* link = nullptr;                                      size_t cap_link = 0;    // tc_get_tree
  float* q6 = nullptr;                                       size_t cap_q6 = 0;      // tc_get_tree
  void release();
};

// Device-side builder (option "device_build"): same tree, same packed layout, written straight into
// *d_tree (grown if needed).  src = (x,y,z,m) in the caller's order, device.  Fills T's sizes/layout
// and D.  Returns TC_OK or an error code with msg set.
int build_device_tree(const float4* src, int64_t n, int n_leaf, int n_group, DeviceBuildScratch& S, void** d_tree,
                      size_t* d_tree_cap, HostTree& T, DeviceTree& D, void* stream, std::string& msg);

// pos [n,3], mass [n] DEVICE -> out [n] (x,y,z,m); flags[0] bit 0: non-finite position, bit 1: bad mass.
// Returns a cudaError_t as int.
int pack_src_device(const float* pos, const float* mass, int64_t n, float4* out, unsigned int* flags, void* stream);

// Direct summation (tc_direct): src [n] (x,y,z,m) device, targets device int64 [n_t] or nullptr (all),
// acc [n_t,3] / pot [n_t] device fp64 (zeroed inside).  Returns a cudaError_t as int.
int launch_direct(const float4* src, long long n, const long long* targets, long long n_t, float eps, double* acc,
                  double* pot, int n_sm, void* stream);
// tc_direct_static: the same direct sum with its source array in a static __device__ block (no allocation of any kind;
// tc_kernels.cu).  All pointers DEVICE.  Returns TC_OK or a TC_E* code with msg set.
int direct_static(const float* pos, const float* mass, long long n, float eps, const long long* targets, long long n_targets,
                  double* acc, double* pot, void* stream, std::string& msg);
// Leapfrog pieces (tc_leapfrog): v += a dt/2 ; x += v dt  and  v += a dt/2 over [n,3] device arrays
// (16-byte aligned).  Return a cudaError_t as int.
int launch_kick_drift(float* pos, float* vel, const float* acc, long long n, float dt, int n_sm, void* stream);
int launch_kick(float* vel, const float* acc, long long n, float dt, int n_sm, void* stream);
// FFMA-only microbenchmark (tc_fp32_peak): returns a cudaError_t as int, *tflops on success.
int measure_fp32_peak(int n_sm, void* stream, double* tflops);

}  // namespace tc

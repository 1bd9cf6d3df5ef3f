// C ABI of the tree-code library (include/tc.h): context, particle intake, host
// build + one bulk copy, launch of the fused walk+evaluate kernel, results.
// There is no CPU fallback anywhere in this file: without a device tc_create()
// fails, and a host-only context (tests of the host builder) refuses tc_forces.
#include <cuda_runtime.h>

#include <chrono>
#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "tc_internal.h"

#ifndef TC_DENSE_MIN_MEAN
#define TC_DENSE_MIN_MEAN 24.0
#endif

struct tc_ctx {
  uint32_t flags = 0;
  bool host_only = false;
  int device = 0, n_sm = 148;
  cudaStream_t own_stream = nullptr, stream = nullptr;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  std::string err;
  // options
  int n_group = 128;
  bool device_build = false;          // option "device_build": tc_build_gpu.cu instead of tc_build.cpp
  int stack_smem = 256;
  int walk_only = 0, open_rule = 0, quadrupole = 1, group_box = 0;
  int shard_rank = 0, shard_count = 1;
  int kernel_config = 0;              // option "kernel_config": 0 = by the mean group size, 1 = sparse, 2 = dense (tc_kernels.cu)
  size_t grid_warps[2][2] = {{0, 0}, {0, 0}};   // warps of the persistent grid, cached: [dense][stack_smem == 64]
  bool two_pass = false;
  tc::TwoPassScratch tps;
  bool last_two_pass = false;
  tc::ShardLayout shard;              // layout of the shards of one evaluation over shard_count ranks (tc_shard.cu)
  bool counts_valid = false;          // d_npc / d_npp hold the counts of the last tc_forces (a shard writes them to its rows)
  // particles (host copy, caller order)
  std::vector<float4> xyzm;                 // the context's host copy of the particles: (x, y, z, m), caller's order
  bool bbox_valid = false;                  // bbox[] = per-axis min (0-2) and max (3-5) of xyzm, taken by the pass that copied it in
  float bbox[6] = {0, 0, 0, 0, 0, 0};
  std::vector<float> pos, mass;             // staging of DEVICE inputs on their way into xyzm
  int64_t n = 0;
  // tree
  tc::HostTree tree;
  bool built = false;
  void* d_tree = nullptr;
  size_t d_tree_cap = 0;
  tc::DeviceTree dview;
  // outputs / scratch on the device
  float* d_acc = nullptr; float* d_pot = nullptr; int64_t out_cap = 0;
  int32_t* d_npc = nullptr; int32_t* d_npp = nullptr; int64_t cnt_cap = 0;
  tc::DeviceCounters* d_ctr = nullptr;
  uint32_t* d_spill = nullptr; size_t spill_elems = 0; int spill_cap = 4096;
  bool forces_done = false, timing_pending = false;
  tc::DeviceBuildScratch dscr;
  bool tree_host_valid = false;       // the host copy of the packed tree (tc_get_tree) is current
  bool host_particles_valid = false;  // xyzm holds the current particles (else only d_src does)
  float4* h_src = nullptr; int64_t h_src_cap = 0;     // pinned staging of (x,y,z,m) for the device build
  float* d_raw = nullptr; int64_t raw_cap = 0;        // device landing area of PINNED host inputs (pos [3n] | mass [n])
  unsigned int* d_flags = nullptr;
  // tc_direct scratch
  float4* d_src = nullptr; int64_t src_cap = 0; bool src_valid = false;
  long long* d_tgt = nullptr; double* d_dacc = nullptr; double* d_dpot = nullptr; int64_t tgt_cap = 0;
  tc_stats stats{};
};

namespace {

thread_local std::string g_create_err;

int fail(tc_ctx* c, int code, const std::string& m) { if (c) c->err = m; return code; }
int cuda_fail(tc_ctx* c, cudaError_t e, const char* what) {
  return fail(c, e == cudaErrorMemoryAllocation ? TC_ENOMEM : TC_ECUDA,
              std::string(what) + ": " + cudaGetErrorString(e));
}
#define TC_CUDA(c, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(c, e_, #call); } while (0)

// page-locked host memory (cudaHostAlloc / cudaHostRegister, e.g. torch pin_memory): DMA reads it directly
bool is_pinned_host_ptr(const tc_ctx* c, const void* p) {
  if (c->host_only || !p) return false;
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeHost;
}

bool is_device_ptr(const tc_ctx* c, const void* p) {
  if (c->host_only || !p) return false;
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

void* packed_alloc(void* user, size_t bytes) {
  tc_ctx* c = (tc_ctx*)user;
  tc::HostTree& T = c->tree;
  if (T.packed && T.packed_cap >= bytes) return T.packed;
  if (T.packed) { if (T.packed_pinned) cudaFreeHost(T.packed); else std::free(T.packed); T.packed = nullptr; T.packed_cap = 0; }
  const size_t cap = bytes + bytes / 8;
  if (!c->host_only) {
    void* p = nullptr;
    if (cudaHostAlloc(&p, cap, cudaHostAllocDefault) == cudaSuccess) { T.packed = p; T.packed_cap = cap; T.packed_pinned = true; return p; }
    cudaGetLastError();
  }
  T.packed = std::malloc(cap); T.packed_pinned = false; T.packed_cap = T.packed ? cap : 0;
  return T.packed;
}

double now_ms() {
  return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

// read the device counters + event time of the last tc_forces into stats (stream must be idle)
int collect(tc_ctx* c) {
  if (!c->timing_pending) return TC_OK;
  c->timing_pending = false;
  tc::DeviceCounters h;
  TC_CUDA(c, cudaMemcpy(&h, c->d_ctr, sizeof(h), cudaMemcpyDeviceToHost));
  float ms = 0.f;
  TC_CUDA(c, cudaEventElapsedTime(&ms, c->ev0, c->ev1));
  c->stats.t_gpu_ms = ms;
  c->stats.t_walk_count_ms = c->stats.t_walk_write_ms = c->stats.t_node_ms = c->stats.t_leaf_ms = 0.0; c->stats.list_bytes = 0;
  if (c->last_two_pass) {
    float t4[4];
    if (tc::two_pass_times(c->tps, t4) == 0) {
      c->stats.t_walk_count_ms = t4[0]; c->stats.t_walk_write_ms = t4[1]; c->stats.t_node_ms = t4[2]; c->stats.t_leaf_ms = t4[3];
    } else cudaGetLastError();
    c->stats.list_bytes = (int64_t)(4 * c->tps.n_list_cells + 8 * c->tps.n_list_leaves);
  }
  c->stats.n_pc_total = (int64_t)h.n_pc_total; c->stats.n_pp_total = (int64_t)h.n_pp_total;
  c->stats.n_tests_total = (int64_t)h.n_tests_total; c->stats.n_spills = (int64_t)h.n_spills;
  c->stats.n_opened_total = (int64_t)h.n_opened_total;
  if (h.overflow) {
    cudaMemset((char*)c->d_ctr + offsetof(tc::DeviceCounters, overflow), 0, sizeof(unsigned int));
  }
  if (h.overflow) return fail(c, TC_EOVERFLOW, "tc_forces: a walk stack exceeded its global spill capacity");
  return TC_OK;
}

// the host copy of the particles (host build, first use after a device-only tc_set_particles)
int ensure_host_particles(tc_ctx* c) {
  if (c->host_particles_valid) return TC_OK;
  if (!c->src_valid) return fail(c, TC_ESTATE, "no particles");
  const int64_t n = c->n;
  try { c->xyzm.resize((size_t)n); } catch (...) { return fail(c, TC_ENOMEM, "out of host memory"); }
  TC_CUDA(c, cudaMemcpyAsync(c->xyzm.data(), c->d_src, sizeof(float4) * (size_t)n, cudaMemcpyDeviceToHost, c->stream));
  TC_CUDA(c, cudaStreamSynchronize(c->stream));
  c->host_particles_valid = true;
  return TC_OK;
}

// (x, y, z, m) of the caller's particles as one float4 array on the device (tc_direct, device build)
int ensure_src(tc_ctx* c) {
  if (c->src_valid) return TC_OK;
  { const int rc = ensure_host_particles(c); if (rc != TC_OK) return rc; }
  const int64_t n = c->n;
  if (c->src_cap < n) {
    cudaFree(c->d_src); c->d_src = nullptr; c->src_cap = 0;
    TC_CUDA(c, cudaMalloc((void**)&c->d_src, sizeof(float4) * (size_t)n));
    c->src_cap = n;
  }
  TC_CUDA(c, cudaMemcpyAsync(c->d_src, c->xyzm.data(), sizeof(float4) * (size_t)n, cudaMemcpyHostToDevice, c->stream));
  TC_CUDA(c, cudaStreamSynchronize(c->stream));
  c->src_valid = true;
  return TC_OK;
}

}  // namespace

extern "C" {

tc_ctx* tc_create_ex(uint32_t flags) {
  tc_ctx* c = new (std::nothrow) tc_ctx();
  if (!c) { g_create_err = "tc_create: out of host memory"; return nullptr; }
  c->flags = flags;
  c->host_only = (flags & TC_FLAG_HOST_ONLY) != 0;
  if (c->host_only) return c;
  cudaError_t e = cudaGetDevice(&c->device);
  if (e == cudaSuccess) e = cudaFree(0);
  cudaDeviceProp prop;
  if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, c->device);
  if (e == cudaSuccess && prop.major < 10) {
    g_create_err = "tc_create: this library is built for sm_100a (B200) only; device is sm_" +
                   std::to_string(prop.major) + std::to_string(prop.minor);
    delete c; return nullptr;
  }
  if (e == cudaSuccess) { c->n_sm = prop.multiProcessorCount; e = cudaStreamCreateWithFlags(&c->own_stream, cudaStreamNonBlocking); }
  if (e == cudaSuccess) e = cudaEventCreate(&c->ev0);
  if (e == cudaSuccess) e = cudaEventCreate(&c->ev1);
  if (e == cudaSuccess) e = cudaMalloc((void**)&c->d_ctr, sizeof(tc::DeviceCounters));
  if (e == cudaSuccess) e = cudaMemset(c->d_ctr, 0, sizeof(tc::DeviceCounters));
  if (e != cudaSuccess) {
    g_create_err = std::string("tc_create: no usable CUDA device (no CPU fallback exists): ") + cudaGetErrorString(e);
    cudaGetLastError();
    tc_destroy(c); return nullptr;
  }
  c->stream = c->own_stream;
  return c;
}

tc_ctx* tc_create(void) { return tc_create_ex(0); }

void tc_destroy(tc_ctx* c) {
  if (!c) return;
  if (!c->host_only) {
    if (c->stream) cudaStreamSynchronize(c->stream);
    cudaFree(c->d_tree); cudaFree(c->d_acc); cudaFree(c->d_pot); cudaFree(c->d_npc); cudaFree(c->d_npp);
    cudaFree(c->d_ctr); cudaFree(c->d_spill);
    c->dscr.release();
    c->tps.release();
    c->shard.release();
    if (c->h_src) cudaFreeHost(c->h_src);
    cudaFree(c->d_flags); cudaFree(c->d_raw);
    cudaFree(c->d_src); cudaFree(c->d_tgt); cudaFree(c->d_dacc); cudaFree(c->d_dpot);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    if (c->own_stream) cudaStreamDestroy(c->own_stream);
  }
  if (c->tree.packed) { if (c->tree.packed_pinned) cudaFreeHost(c->tree.packed); else std::free(c->tree.packed); }
  delete c;
}

const char* tc_last_error(const tc_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }

int tc_set_option(tc_ctx* c, const char* key, double v) {
  if (!c || !key) return fail(c, TC_EINVAL, "tc_set_option: null argument");
  if (!std::strcmp(key, "n_group")) {
    if (!(v >= 1.0) || v > 2147483647.0 || v != std::floor(v)) return fail(c, TC_EINVAL, "tc_set_option: n_group must be an integer >= 1");
    c->n_group = (int)v; return TC_OK;
  }
  if (!std::strcmp(key, "device_build")) {
    if (v != 0.0 && v != 1.0) return fail(c, TC_EINVAL, "tc_set_option: device_build must be 0 or 1");
    if (c->host_only && v != 0.0) return fail(c, TC_ESTATE, "tc_set_option: device_build needs a device");
    c->device_build = (v != 0.0); return TC_OK;
  }
  if (!std::strcmp(key, "open_rule")) {
    if (v != 0.0 && v != 1.0) return fail(c, TC_EINVAL, "tc_set_option: open_rule must be 0 or 1");
    c->open_rule = (int)v; return TC_OK;
  }
  if (!std::strcmp(key, "kernel_config")) {
    if (v != 0.0 && v != 1.0 && v != 2.0) return fail(c, TC_EINVAL, "tc_set_option: kernel_config must be 0 (auto), 1 (sparse) or 2 (dense)");
    c->kernel_config = (int)v; return TC_OK;
  }
  if (!std::strcmp(key, "shard_count")) {
    if (!(v >= 1.0) || v > 65536.0 || v != std::floor(v)) return fail(c, TC_EINVAL, "tc_set_option: shard_count must be an integer in [1, 65536]");
    c->shard_count = (int)v; return TC_OK;
  }
  if (!std::strcmp(key, "shard_rank")) {
    if (!(v >= 0.0) || v > 65535.0 || v != std::floor(v)) return fail(c, TC_EINVAL, "tc_set_option: shard_rank must be an integer in [0, 65535]");
    c->shard_rank = (int)v; return TC_OK;
  }
  if (!std::strcmp(key, "group_box")) {
    if (v != 0.0 && v != 1.0) return fail(c, TC_EINVAL, "tc_set_option: group_box must be 0 or 1");
    c->group_box = (int)v; return TC_OK;
  }
  if (!std::strcmp(key, "quadrupole")) {
    if (v != 0.0 && v != 1.0) return fail(c, TC_EINVAL, "tc_set_option: quadrupole must be 0 or 1");
    c->quadrupole = (int)v; return TC_OK;
  }
  if (!std::strcmp(key, "two_pass")) {
    if (v != 0.0 && v != 1.0) return fail(c, TC_EINVAL, "tc_set_option: two_pass must be 0 or 1");
    c->two_pass = (v != 0.0); return TC_OK;
  }
  if (!std::strcmp(key, "walk_only")) {
    if (v != 0.0 && v != 1.0) return fail(c, TC_EINVAL, "tc_set_option: walk_only must be 0 or 1");
    c->walk_only = (int)v; return TC_OK;
  }
  if (!std::strcmp(key, "stack_smem")) {
    if (v != 256.0 && v != 64.0) return fail(c, TC_EINVAL, "tc_set_option: stack_smem must be 256 or 64");
    c->stack_smem = (int)v; return TC_OK;
  }
  return fail(c, TC_EINVAL, std::string("tc_set_option: unknown key '") + key + "'");
}

int tc_set_stream(tc_ctx* c, void* s) {
  if (!c) return TC_EINVAL;
  if (c->host_only) return fail(c, TC_ESTATE, "tc_set_stream: host-only context");
  TC_CUDA(c, cudaStreamSynchronize(c->stream));
  c->stream = s ? (cudaStream_t)s : c->own_stream;
  return TC_OK;
}

int tc_sync(tc_ctx* c) {
  if (!c) return TC_EINVAL;
  if (c->host_only) return TC_OK;
  TC_CUDA(c, cudaStreamSynchronize(c->stream));
  return collect(c);
}

int tc_set_particles(tc_ctx* c, const float* pos, const float* mass, int64_t n) {
  if (!c) return TC_EINVAL;
  if (!pos || !mass) return fail(c, TC_EINVAL, "tc_set_particles: null pointer");
  if (n < 1 || n > 2147483647LL) return fail(c, TC_EINVAL, "tc_set_particles: n must be in [1, 2^31-1]");
  c->built = false; c->forces_done = false; c->src_valid = false; c->host_particles_valid = false; c->bbox_valid = false;
  c->n = 0;
  const bool pos_dev = is_device_ptr(c, pos), mass_dev = is_device_ptr(c, mass);
  const bool dev_mode = c->device_build && !c->host_only;
  if (dev_mode) {
    if (c->src_cap < n) {
      TC_CUDA(c, cudaStreamSynchronize(c->stream));
      cudaFree(c->d_src); c->d_src = nullptr; c->src_cap = 0;
      TC_CUDA(c, cudaMalloc((void**)&c->d_src, sizeof(float4) * (size_t)n));
      c->src_cap = n;
    }
    if (!c->d_flags) TC_CUDA(c, cudaMalloc((void**)&c->d_flags, sizeof(unsigned int)));
  }
  // device build with PINNED host inputs: DMA them as they are and let the pack kernel interleave and validate —
  // no host pass over the particles at all (pageable inputs keep the parallel staging pass below, which is
  // faster than the driver's own staging of pageable memory)
  const bool pos_pin = dev_mode && !pos_dev && is_pinned_host_ptr(c, pos), mass_pin = dev_mode && !mass_dev && is_pinned_host_ptr(c, mass);
  if (dev_mode && (pos_dev || pos_pin) && (mass_dev || mass_pin)) {
    const float* dp = pos; const float* dm = mass;
    if (pos_pin || mass_pin) {
      if (c->raw_cap < n) {
        TC_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(c->d_raw); c->d_raw = nullptr; c->raw_cap = 0;
        TC_CUDA(c, cudaMalloc((void**)&c->d_raw, sizeof(float) * 4 * (size_t)n));
        c->raw_cap = n;
      }
      if (pos_pin) { TC_CUDA(c, cudaMemcpyAsync(c->d_raw, pos, sizeof(float) * 3 * (size_t)n, cudaMemcpyHostToDevice, c->stream)); dp = c->d_raw; }
      if (mass_pin) { TC_CUDA(c, cudaMemcpyAsync(c->d_raw + 3 * (size_t)n, mass, sizeof(float) * (size_t)n, cudaMemcpyHostToDevice, c->stream)); dm = c->d_raw + 3 * (size_t)n; }
    }
    // device (or landed) inputs, device build: interleave + validate in one kernel
    const int le = tc::pack_src_device(dp, dm, n, c->d_src, c->d_flags, c->stream);
    if (le != 0) return cuda_fail(c, (cudaError_t)le, "tc_set_particles: pack kernel");
    unsigned int flags = 0;
    TC_CUDA(c, cudaMemcpyAsync(&flags, c->d_flags, sizeof(flags), cudaMemcpyDeviceToHost, c->stream));
    TC_CUDA(c, cudaStreamSynchronize(c->stream));
    if (flags & 1u) return fail(c, TC_EINVAL, "tc_set_particles: non-finite position");
    if (flags & 2u) return fail(c, TC_EINVAL, "tc_set_particles: negative or non-finite mass");
    c->src_valid = true;
    c->n = n;
    return TC_OK;
  }
  try {
    c->xyzm.resize((size_t)n);
    if (pos_dev) c->pos.resize((size_t)n * 3);
    if (mass_dev) c->mass.resize((size_t)n);
  } catch (...) { return fail(c, TC_ENOMEM, "tc_set_particles: out of host memory"); }
  const float* P = pos; const float* M = mass;      // where the validation pass reads from
  if (pos_dev) { TC_CUDA(c, cudaMemcpyAsync(c->pos.data(), pos, sizeof(float) * 3 * (size_t)n, cudaMemcpyDeviceToHost, c->stream)); P = c->pos.data(); }
  if (mass_dev) { TC_CUDA(c, cudaMemcpyAsync(c->mass.data(), mass, sizeof(float) * (size_t)n, cudaMemcpyDeviceToHost, c->stream)); M = c->mass.data(); }
  if (!c->host_only) TC_CUDA(c, cudaStreamSynchronize(c->stream));   // also: h_src of the previous call is no longer in flight
  if (dev_mode && c->h_src_cap < n) {
    if (c->h_src) cudaFreeHost(c->h_src);
    c->h_src = nullptr; c->h_src_cap = 0;
    TC_CUDA(c, cudaHostAlloc((void**)&c->h_src, sizeof(float4) * (size_t)n, cudaHostAllocDefault));
    c->h_src_cap = n;
  }
  // one pass: copy into the context, validate, and (device build) stage (x,y,z,m) in pinned memory
  bool bad_pos = false, bad_mass = false;
  float4* X4 = c->xyzm.data();
  float4* H = dev_mode ? c->h_src : nullptr;
  // (the per-axis extremes are the first thing tc_build needs: taken here, while the data passes by)
  float l0 = INFINITY, l1 = INFINITY, l2 = INFINITY, h0 = -INFINITY, h1 = -INFINITY, h2 = -INFINITY;
#pragma omp parallel for schedule(static) reduction(| : bad_pos, bad_mass) reduction(min : l0, l1, l2) reduction(max : h0, h1, h2)
  for (int64_t i = 0; i < n; i++) {
    const float x = P[3 * i], y = P[3 * i + 1], z = P[3 * i + 2], m = M[i];
    X4[i] = make_float4(x, y, z, m);
    l0 = std::min(l0, x); h0 = std::max(h0, x); l1 = std::min(l1, y); h1 = std::max(h1, y); l2 = std::min(l2, z); h2 = std::max(h2, z);
    if (H) H[i] = make_float4(x, y, z, m);
    bad_pos |= !(std::isfinite(x) && std::isfinite(y) && std::isfinite(z));
    bad_mass |= !(std::isfinite(m) && m >= 0.f);
  }
  if (bad_pos) return fail(c, TC_EINVAL, "tc_set_particles: non-finite position");
  if (bad_mass) return fail(c, TC_EINVAL, "tc_set_particles: negative or non-finite mass");
  c->host_particles_valid = true;
  c->bbox[0] = l0; c->bbox[1] = l1; c->bbox[2] = l2; c->bbox[3] = h0; c->bbox[4] = h1; c->bbox[5] = h2;
  c->bbox_valid = true;
  if (dev_mode) {     // stream-ordered: tc_build runs on the same stream
    TC_CUDA(c, cudaMemcpyAsync(c->d_src, c->h_src, sizeof(float4) * (size_t)n, cudaMemcpyHostToDevice, c->stream));
    c->src_valid = true;
  }
  c->n = n;
  return TC_OK;
}

int tc_build(tc_ctx* c, int n_leaf) {
  if (!c) return TC_EINVAL;
  if (c->n < 1) return fail(c, TC_ESTATE, "tc_build: no particles (call tc_set_particles first)");
  if (n_leaf < 1) return fail(c, TC_EINVAL, "tc_build: n_leaf must be >= 1");
  c->built = false; c->forces_done = false; c->shard.k = 0;
  if (!c->host_only) TC_CUDA(c, cudaStreamSynchronize(c->stream));  // the pinned buffer may still be in flight
  if (c->device_build) {
    { const int rc = ensure_src(c); if (rc != TC_OK) return rc; }
    const double t0 = now_ms();
    std::string msg;
    const int rc = tc::build_device_tree(c->d_src, c->n, n_leaf, c->n_group, c->dscr, &c->d_tree, &c->d_tree_cap, c->tree,
                                         c->dview, c->stream, msg);
    if (rc != TC_OK) { cudaGetLastError(); return fail(c, rc, "tc_build (device): " + msg); }
    const tc::HostTree& T = c->tree;
    tc_stats& S = c->stats;
    S = tc_stats{};
    S.n = c->n; S.n_cells = T.n_cells; S.n_leaves = T.n_leaves; S.n_groups = T.n_groups; S.depth = T.depth;
    S.n_leaf = n_leaf; S.n_group = c->n_group; S.t_host_ms = now_ms() - t0; S.t_copy_ms = 0.0; S.tree_bytes = (int64_t)T.lay.bytes;
    c->tree_host_valid = false;
    c->built = true;
    return TC_OK;
  }
  { const int rc0 = ensure_host_particles(c); if (rc0 != TC_OK) return rc0; }
  const double t0 = now_ms();
  std::string msg;
  const int rc = tc::build_host_tree(c->xyzm.data(), c->n, n_leaf, c->n_group, c->tree, packed_alloc, c, msg,
                                     c->bbox_valid ? c->bbox : nullptr);
  if (rc != TC_OK) return fail(c, rc, msg);
  const double t1 = now_ms();
  const tc::HostTree& T = c->tree;
  tc_stats& S = c->stats;
  S = tc_stats{};
  S.n = c->n; S.n_cells = T.n_cells; S.n_leaves = T.n_leaves; S.n_groups = T.n_groups; S.depth = T.depth;
  S.n_leaf = n_leaf; S.n_group = c->n_group; S.t_host_ms = t1 - t0; S.tree_bytes = (int64_t)T.lay.bytes;
  if (!c->host_only) {
    if (c->d_tree_cap < T.lay.bytes) {
      cudaFree(c->d_tree); c->d_tree = nullptr; c->d_tree_cap = 0;
      const size_t cap = T.lay.bytes + T.lay.bytes / 8;
      TC_CUDA(c, cudaMalloc(&c->d_tree, cap));
      c->d_tree_cap = cap;
    }
    // the ONE bulk copy ("only the tree structure needs to travel")
    TC_CUDA(c, cudaMemcpyAsync(c->d_tree, T.packed, T.lay.bytes, cudaMemcpyHostToDevice, c->stream));
    TC_CUDA(c, cudaStreamSynchronize(c->stream));
    S.t_copy_ms = now_ms() - t1;
    char* b = (char*)c->d_tree;
    tc::DeviceTree& D = c->dview;
    D.bnd = (const float4*)(b + T.lay.off_bnd); D.xm = (const float4*)(b + T.lay.off_xm);
    D.q0 = (const float4*)(b + T.lay.off_q0); D.q1 = (const float4*)(b + T.lay.off_q1);
    D.part = (const float4*)(b + T.lay.off_part); D.orig = (const int32_t*)(b + T.lay.off_orig);
    D.grp = (const int4*)(b + T.lay.off_grp);
    D.gbox = (const float4*)(b + T.lay.off_gbox);
    D.n = c->n; D.n_cells = T.n_cells; D.n_groups = T.n_groups;
  }
  c->tree_host_valid = true;
  c->built = true;
  return TC_OK;
}

namespace {
// theta and eps as the kernels may take them.  eps < kEpsMin is eps = 0: the self pair and coincident pairs
// have s^2 = eps^2, and m / eps^3 must stay finite in fp32 for their (zero) contribution m d / s^3 not to become
// inf * 0 = NaN (a subnormal eps^2 is even flushed to 0 by rsqrt.approx.ftz and gives inf at once); fp32 coordinates
// cannot resolve separations below 1e-10 anyway unless |x| < 1e-3.  theta whose square overflows fp32 is refused
// (d^2 theta^2 = 0 * inf = NaN would leave a group's own ancestors un-opened).
constexpr float kEpsMin = 1e-10f;
// the dense launch configuration pays from this many particles per group on (measured crossover)
constexpr double kDenseMinMean = TC_DENSE_MIN_MEAN;
int check_theta_eps(tc_ctx* c, const char* who, float theta, float& eps) {
  if (!(theta >= 0.f) || !std::isfinite(theta) || !(eps >= 0.f) || !std::isfinite(eps))
    return fail(c, TC_EINVAL, std::string(who) + ": theta and eps must be finite and >= 0");
  if (theta > 1e18f) return fail(c, TC_EINVAL, std::string(who) + ": theta must be <= 1e18 (theta^2 overflows fp32)");
  if (eps < kEpsMin) eps = 0.f;
  return TC_OK;
}

// A1-A6 on the context's stream.  shard_out4 == nullptr: the whole evaluation into acc / pot (host or device, caller's
// order).  shard_out4 != nullptr (device [n_slots,4]): this rank's shard into compact rows (tc_forces_shard).
int forces_impl(tc_ctx* c, const char* who, float theta, float eps, float* acc, float* pot, float* shard_out4, int32_t* shard_cnt2) {
  if (c->host_only) return fail(c, TC_ESTATE, std::string(who) + ": host-only context has no device (there is no CPU fallback)");
  if (!c->built) return fail(c, TC_ESTATE, std::string(who) + ": no tree (call tc_build first)");
  { const int rc = check_theta_eps(c, who, theta, eps); if (rc != TC_OK) return rc; }
  const bool shard = shard_out4 != nullptr;
  const int64_t n = c->n;
  bool acc_dev = true;
  if (!shard) {
    if (!acc) return fail(c, TC_EINVAL, std::string(who) + ": acc is null");
    acc_dev = is_device_ptr(c, acc);
    const bool pot_dev = pot ? is_device_ptr(c, pot) : acc_dev;
    if (pot && acc_dev != pot_dev) return fail(c, TC_EINVAL, std::string(who) + ": acc and pot must both be host or both be device pointers");
  }
  if (c->cnt_cap < n) {
    cudaFree(c->d_npc); cudaFree(c->d_npp); c->d_npc = c->d_npp = nullptr; c->cnt_cap = 0;
    TC_CUDA(c, cudaMalloc((void**)&c->d_npc, sizeof(int32_t) * (size_t)n));
    TC_CUDA(c, cudaMalloc((void**)&c->d_npp, sizeof(int32_t) * (size_t)n));
    c->cnt_cap = n;
  }
  if (!acc_dev && c->out_cap < n) {
    cudaFree(c->d_acc); cudaFree(c->d_pot); c->d_acc = c->d_pot = nullptr; c->out_cap = 0;
    TC_CUDA(c, cudaMalloc((void**)&c->d_acc, sizeof(float) * 3 * (size_t)n));
    TC_CUDA(c, cudaMalloc((void**)&c->d_pot, sizeof(float) * (size_t)n));
    c->out_cap = n;
  }
  // launch configuration of the fused kernel (tc_kernels.cu): dense from kDenseMinMean particles per group on
  // (a forced configuration is honoured with either stack size; the automatic choice keeps the small-stack test path on
  // the sparse build; the two-pass pipeline exists in one configuration only)
  const bool dense = !c->two_pass &&
                     (c->kernel_config == 2 ||
                      (c->kernel_config == 0 && c->stack_smem == 256 && (double)n >= kDenseMinMean * (double)c->tree.n_groups));
  size_t& warps_cached = c->grid_warps[dense ? 1 : 0][c->stack_smem == 64 ? 1 : 0];
  if (!warps_cached)   // (an occupancy query: once per configuration, not per call)
    warps_cached = (size_t)(dense ? tc::dense::forces_total_warps(c->n_sm, c->stack_smem) : tc::sparse::forces_total_warps(c->n_sm, c->stack_smem));
  const size_t warps = warps_cached;
  if (c->spill_elems < warps * (size_t)c->spill_cap) {
    cudaFree(c->d_spill); c->d_spill = nullptr; c->spill_elems = 0;
    TC_CUDA(c, cudaMalloc((void**)&c->d_spill, sizeof(uint32_t) * warps * (size_t)c->spill_cap));
    c->spill_elems = warps * (size_t)c->spill_cap;
  }
  tc::ForceLaunch L;
  L.theta = theta; L.eps = eps;
  L.acc = acc_dev ? acc : c->d_acc;
  L.pot = pot ? (acc_dev ? pot : c->d_pot) : nullptr;
  L.n_pc = c->d_npc; L.n_pp = c->d_npp; L.counters = c->d_ctr; L.spill = c->d_spill; L.spill_cap = c->spill_cap;
  L.stack_smem = c->stack_smem; L.n_sm = c->n_sm; L.flags = (c->walk_only ? 1 : 0) | (c->open_rule ? 2 : 0) | (c->quadrupole ? 0 : 4) | (c->group_box ? 8 : 0);
  L.max_grid = (int)(warps / (size_t)(dense ? tc::dense::forces_warps_per_cta() : tc::sparse::forces_warps_per_cta()));
  if (shard) {
    L.shard_rank = c->shard_rank; L.shard_count = c->shard_count;
    L.shard_out4 = shard_out4; L.shard_cnt2 = shard_cnt2; L.shard_off = c->shard.off;
  }
  // stream-ordered: no host synchronisation between queued calls; the overflow flag is sticky until collect()
  TC_CUDA(c, cudaMemsetAsync(c->d_ctr, 0, offsetof(tc::DeviceCounters, overflow), c->stream));
  TC_CUDA(c, cudaEventRecord(c->ev0, c->stream));
  const int le = c->two_pass ? tc::launch_forces_two_pass(c->dview, L, c->tps, c->stream)
                             : dense ? tc::dense::launch_forces(c->dview, L, c->stream) : tc::sparse::launch_forces(c->dview, L, c->stream);
  if (le != 0) return cuda_fail(c, (cudaError_t)le, "forces kernel launch");
  c->last_two_pass = c->two_pass;
  TC_CUDA(c, cudaEventRecord(c->ev1, c->stream));
  c->timing_pending = true; c->forces_done = true; c->counts_valid = !shard;
  if (!acc_dev) {
    TC_CUDA(c, cudaMemcpyAsync(acc, c->d_acc, sizeof(float) * 3 * (size_t)n, cudaMemcpyDeviceToHost, c->stream));
    if (pot) TC_CUDA(c, cudaMemcpyAsync(pot, c->d_pot, sizeof(float) * (size_t)n, cudaMemcpyDeviceToHost, c->stream));
    TC_CUDA(c, cudaStreamSynchronize(c->stream));
    return collect(c);
  }
  return TC_OK;
}

// the shard layout of the built tree for the current shard_count (built on first use, kept until tc_build)
int ensure_shard_layout(tc_ctx* c, const char* who) {
  if (c->host_only) return fail(c, TC_ESTATE, std::string(who) + ": host-only context has no device");
  if (!c->built) return fail(c, TC_ESTATE, std::string(who) + ": no tree (call tc_build first)");
  if (c->shard_rank >= c->shard_count) return fail(c, TC_EINVAL, std::string(who) + ": shard_rank must be < shard_count");
  if (c->shard.k == c->shard_count) return TC_OK;
  const int e = tc::build_shard_layout(c->dview, c->shard_count, c->shard, c->stream);
  if (e != 0) return cuda_fail(c, (cudaError_t)e, "shard layout");
  return TC_OK;
}
}  // namespace

int tc_forces(tc_ctx* c, float theta, float eps, float* acc, float* pot) {
  if (!c) return TC_EINVAL;
  if (c->shard_count > 1)
    return fail(c, TC_ESTATE, "tc_forces: shard_count > 1 — a shard of a multi-GPU evaluation is computed by tc_forces_shard");
  return forces_impl(c, "tc_forces", theta, eps, acc, pot, nullptr, nullptr);
}

int tc_shard_size(tc_ctx* c, int64_t* n_slots) {
  if (!c || !n_slots) return fail(c, TC_EINVAL, "tc_shard_size: null argument");
  const int rc = ensure_shard_layout(c, "tc_shard_size");
  if (rc != TC_OK) return rc;
  *n_slots = (int64_t)c->shard.n_slots;
  return TC_OK;
}

int tc_forces_shard(tc_ctx* c, float theta, float eps, float* out4, int32_t* cnt2) {
  if (!c) return TC_EINVAL;
  if (!out4) return fail(c, TC_EINVAL, "tc_forces_shard: out4 is null");
  if (c->two_pass) return fail(c, TC_EINVAL, "tc_forces_shard: sharding runs the fused kernel only (two_pass must be 0)");
  if (!c->host_only && (!is_device_ptr(c, out4) || (cnt2 && !is_device_ptr(c, cnt2))))
    return fail(c, TC_EINVAL, "tc_forces_shard: out4 and cnt2 must be device pointers");
  const int rc = ensure_shard_layout(c, "tc_forces_shard");
  if (rc != TC_OK) return rc;
  return forces_impl(c, "tc_forces_shard", theta, eps, nullptr, nullptr, out4, cnt2);
}

int tc_shard_scatter(tc_ctx* c, const float* gathered4, const int32_t* gathered_cnt2, float* acc, float* pot, int32_t* n_pc,
                     int32_t* n_pp) {
  if (!c) return TC_EINVAL;
  if (!gathered4 || !acc) return fail(c, TC_EINVAL, "tc_shard_scatter: gathered4 and acc must not be null");
  const int rc = ensure_shard_layout(c, "tc_shard_scatter");
  if (rc != TC_OK) return rc;
  for (const void* p : {(const void*)gathered4, (const void*)gathered_cnt2, (const void*)acc, (const void*)pot, (const void*)n_pc, (const void*)n_pp})
    if (p && !is_device_ptr(c, p)) return fail(c, TC_EINVAL, "tc_shard_scatter: all buffers must be device pointers");
  const int e = tc::launch_shard_scatter(c->dview, c->shard, gathered4, gathered_cnt2, acc, pot, n_pc, n_pp, c->stream);
  if (e != 0) return cuda_fail(c, (cudaError_t)e, "shard scatter");
  return TC_OK;
}

int tc_get_counts(tc_ctx* c, int32_t* n_pc, int32_t* n_pp) {
  if (!c) return TC_EINVAL;
  if (!c->forces_done) return fail(c, TC_ESTATE, "tc_get_counts: no tc_forces since the last tc_build");
  if (!c->counts_valid) return fail(c, TC_ESTATE, "tc_get_counts: the last evaluation was a shard (its counts are in the cnt2 rows of tc_forces_shard)");
  TC_CUDA(c, cudaStreamSynchronize(c->stream));
  if (n_pc) TC_CUDA(c, cudaMemcpy(n_pc, c->d_npc, sizeof(int32_t) * (size_t)c->n, cudaMemcpyDeviceToHost));
  if (n_pp) TC_CUDA(c, cudaMemcpy(n_pp, c->d_npp, sizeof(int32_t) * (size_t)c->n, cudaMemcpyDeviceToHost));
  return collect(c);
}

int tc_get_stats(tc_ctx* c, tc_stats* out) {
  if (!c || !out) return fail(c, TC_EINVAL, "tc_get_stats: null argument");
  int rc = TC_OK;
  if (!c->host_only && c->timing_pending) { TC_CUDA(c, cudaStreamSynchronize(c->stream)); rc = collect(c); }
  *out = c->stats;
  return rc;
}

int tc_direct(tc_ctx* c, float eps, const int64_t* targets, int64_t n_targets, double* acc, double* pot) {
  if (!c) return TC_EINVAL;
  if (c->host_only) return fail(c, TC_ESTATE, "tc_direct: host-only context has no device (there is no CPU fallback)");
  if (c->n < 1) return fail(c, TC_ESTATE, "tc_direct: no particles (call tc_set_particles first)");
  if (!acc) return fail(c, TC_EINVAL, "tc_direct: acc is null");
  if (!(eps >= 0.f) || !std::isfinite(eps)) return fail(c, TC_EINVAL, "tc_direct: eps must be finite and >= 0");
  if (eps < 1e-10f) eps = 0.f;   // as tc_forces (check_theta_eps): m / eps^3 of the self pair must stay finite
  const int64_t n = c->n;
  const int64_t nt = targets ? n_targets : n;
  if (nt < 1) return fail(c, TC_EINVAL, "tc_direct: n_targets must be >= 1");
  if (targets)
    for (int64_t t = 0; t < nt; t++)
      if (targets[t] < 0 || targets[t] >= n) return fail(c, TC_EINVAL, "tc_direct: target index out of range");
  const bool acc_dev = is_device_ptr(c, acc), pot_dev = pot ? is_device_ptr(c, pot) : acc_dev;
  if (acc_dev != pot_dev) return fail(c, TC_EINVAL, "tc_direct: acc and pot must both be host or both be device pointers");
  { const int rc = ensure_src(c); if (rc != TC_OK) return rc; }
  if (c->tgt_cap < nt) {
    cudaFree(c->d_tgt); cudaFree(c->d_dacc); cudaFree(c->d_dpot); c->d_tgt = nullptr; c->d_dacc = c->d_dpot = nullptr; c->tgt_cap = 0;
    TC_CUDA(c, cudaMalloc((void**)&c->d_tgt, sizeof(long long) * (size_t)nt));
    TC_CUDA(c, cudaMalloc((void**)&c->d_dacc, sizeof(double) * 3 * (size_t)nt));
    TC_CUDA(c, cudaMalloc((void**)&c->d_dpot, sizeof(double) * (size_t)nt));
    c->tgt_cap = nt;
  }
  if (targets) {
    static_assert(sizeof(long long) == sizeof(int64_t), "int64_t layout");
    TC_CUDA(c, cudaMemcpyAsync(c->d_tgt, targets, sizeof(int64_t) * (size_t)nt, cudaMemcpyHostToDevice, c->stream));
  }
  double* o_acc = acc_dev ? acc : c->d_dacc;
  double* o_pot = pot ? (acc_dev ? pot : c->d_dpot) : nullptr;
  TC_CUDA(c, cudaEventRecord(c->ev0, c->stream));
  const int le = tc::launch_direct(c->d_src, n, targets ? c->d_tgt : nullptr, nt, eps, o_acc, o_pot, c->n_sm, c->stream);
  if (le != 0) return cuda_fail(c, (cudaError_t)le, "direct-sum kernel launch");
  TC_CUDA(c, cudaEventRecord(c->ev1, c->stream));
  if (!acc_dev) {
    TC_CUDA(c, cudaMemcpyAsync(acc, c->d_dacc, sizeof(double) * 3 * (size_t)nt, cudaMemcpyDeviceToHost, c->stream));
    if (pot) TC_CUDA(c, cudaMemcpyAsync(pot, c->d_dpot, sizeof(double) * (size_t)nt, cudaMemcpyDeviceToHost, c->stream));
  }
  // targets (host memory of the caller) must not be in flight on return
  TC_CUDA(c, cudaStreamSynchronize(c->stream));
  float ms = 0.f;
  if (cudaEventElapsedTime(&ms, c->ev0, c->ev1) == cudaSuccess) c->stats.t_gpu_ms = ms; else cudaGetLastError();
  c->timing_pending = false;
  return TC_OK;
}

// No context, no allocation: everything happens in tc::direct_static (tc_kernels.cu, next to the static array it uses).
int tc_direct_static(const float* pos, const float* mass, int64_t n, float eps, const int64_t* targets, int64_t n_targets,
                     double* acc, double* pot, void* cuda_stream) {
  static_assert(sizeof(long long) == sizeof(int64_t), "int64_t layout");
  std::string msg;
  const int rc = tc::direct_static(pos, mass, (long long)n, eps, reinterpret_cast<const long long*>(targets), (long long)n_targets,
                                   acc, pot, cuda_stream, msg);
  if (rc != TC_OK) g_create_err = msg;
  return rc;
}

int tc_leapfrog(tc_ctx* c, float* pos, float* vel, const float* mass, int64_t n, float dt, int steps, int n_leaf,
                float theta, float eps, float* acc, float* pot, int have_acc) {
  if (!c) return TC_EINVAL;
  if (c->host_only) return fail(c, TC_ESTATE, "tc_leapfrog: host-only context has no device (there is no CPU fallback)");
  if (!pos || !vel || !mass || !acc) return fail(c, TC_EINVAL, "tc_leapfrog: null argument");
  if (n < 1 || n > 2147483647LL) return fail(c, TC_EINVAL, "tc_leapfrog: n must be in [1, 2^31-1]");
  if (steps < 0 || !std::isfinite(dt)) return fail(c, TC_EINVAL, "tc_leapfrog: steps must be >= 0 and dt finite");
  const void* ptrs[5] = {pos, vel, mass, acc, pot};
  for (int k = 0; k < 5; k++) {
    if (!ptrs[k]) continue;
    if (!is_device_ptr(c, ptrs[k])) return fail(c, TC_EINVAL, "tc_leapfrog: pos, vel, mass, acc and pot must be DEVICE pointers");
    if (k != 2 && (reinterpret_cast<uintptr_t>(ptrs[k]) & 15u)) return fail(c, TC_EINVAL, "tc_leapfrog: arrays must be 16-byte aligned");
  }
  auto force = [&]() -> int {          // the user's three calls, with device pointers: nothing crosses PCIe with device_build
    int e = tc_set_particles(c, pos, mass, n);
    if (e == TC_OK) e = tc_build(c, n_leaf);
    if (e == TC_OK) e = tc_forces(c, theta, eps, acc, pot);
    return e;
  };
  if (!have_acc || steps == 0) { const int e = force(); if (e != TC_OK) return e; }
  for (int s = 0; s < steps; s++) {
    int le = tc::launch_kick_drift(pos, vel, acc, n, dt, c->n_sm, c->stream);
    if (le != 0) return cuda_fail(c, (cudaError_t)le, "kick-drift kernel launch");
    const int e = force();
    if (e != TC_OK) return e;
    le = tc::launch_kick(vel, acc, n, dt, c->n_sm, c->stream);
    if (le != 0) return cuda_fail(c, (cudaError_t)le, "kick kernel launch");
  }
  return TC_OK;
}

int tc_fp32_peak(tc_ctx* c, double* tflops) {
  if (!c || !tflops) return fail(c, TC_EINVAL, "tc_fp32_peak: null argument");
  if (c->host_only) return fail(c, TC_ESTATE, "tc_fp32_peak: host-only context has no device");
  const int e = tc::measure_fp32_peak(c->n_sm, c->stream, tflops);
  if (e != 0) return cuda_fail(c, (cudaError_t)e, "fp32 peak microbenchmark");
  return TC_OK;
}

int tc_get_tree(tc_ctx* c, int32_t* perm, float* cell_bnd, float* cell_xm, float* cell_q, int32_t* cell_link,
                int32_t* groups) {
  if (!c) return TC_EINVAL;
  if (!c->built) return fail(c, TC_ESTATE, "tc_get_tree: no tree (call tc_build first)");
  if (!c->tree_host_valid) {                       // built on the device: bring the packed tree back
    tc::HostTree& W = c->tree;
    if (!packed_alloc(c, W.lay.bytes)) return fail(c, TC_ENOMEM, "tc_get_tree: out of host memory");
    try { W.link.resize((size_t)W.n_cells * 4); W.q6.resize((size_t)W.n_cells * 6); } catch (...) { return fail(c, TC_ENOMEM, "tc_get_tree: out of host memory"); }
    TC_CUDA(c, cudaStreamSynchronize(c->stream));
    TC_CUDA(c, cudaMemcpy(W.packed, c->d_tree, W.lay.bytes, cudaMemcpyDeviceToHost));
    TC_CUDA(c, cudaMemcpy(W.link.data(), c->dscr.link, sizeof(int32_t) * 4 * (size_t)W.n_cells, cudaMemcpyDeviceToHost));
    TC_CUDA(c, cudaMemcpy(W.q6.data(), c->dscr.q6, sizeof(float) * 6 * (size_t)W.n_cells, cudaMemcpyDeviceToHost));
    c->tree_host_valid = true;
  }
  const tc::HostTree& T = c->tree;
  const char* b = (const char*)T.packed;
  const size_t nc = (size_t)T.n_cells;
  if (perm) std::memcpy(perm, b + T.lay.off_orig, sizeof(int32_t) * (size_t)T.n);
  if (cell_bnd) {
    std::memcpy(cell_bnd, b + T.lay.off_bnd, sizeof(float) * 4 * nc);
    for (size_t i = 0; i < nc; i++) cell_bnd[4 * i + 3] = std::fabs(cell_bnd[4 * i + 3]);  // drop the leaf flag
  }
  if (cell_xm) std::memcpy(cell_xm, b + T.lay.off_xm, sizeof(float) * 4 * nc);
  if (cell_q) std::memcpy(cell_q, T.q6.data(), sizeof(float) * 6 * nc);
  if (cell_link) std::memcpy(cell_link, T.link.data(), sizeof(int32_t) * 4 * nc);
  if (groups) {
    const int4* g = (const int4*)(b + T.lay.off_grp);
    for (int64_t i = 0; i < T.n_groups; i++) groups[i] = g[i].x;
  }
  return TC_OK;
}

int tc_get_group_boxes(tc_ctx* c, float* half_ext) {
  if (!c || !half_ext) return fail(c, TC_EINVAL, "tc_get_group_boxes: null argument");
  const int e = tc_get_tree(c, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr);   // brings a device-built tree back
  if (e != TC_OK) return e;
  const tc::HostTree& T = c->tree;
  const float4* gb = (const float4*)((const char*)T.packed + T.lay.off_gbox);
  for (int64_t i = 0; i < T.n_groups; i++) { half_ext[3 * i] = gb[i].x; half_ext[3 * i + 1] = gb[i].y; half_ext[3 * i + 2] = gb[i].z; }
  return TC_OK;
}

}  // extern "C"

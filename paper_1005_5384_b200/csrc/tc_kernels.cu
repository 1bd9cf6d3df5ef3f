// Fused tree walk + interaction-list evaluation for sm_100a (steps A1-A6 of
// DESIGN.md; Sec. 2.2-2.3 of arXiv 1005.5384).
//
// The paper walks every group twice with one THREAD per group (count, host scan,
// write), stores the lists in global memory and evaluates them
// with two more kernels (Lists 3-4).  Here one WARP owns a group from start to end:
//   * the walk is lane-parallel: 4 nodes are popped from a shared-memory stack per
//     iteration and their <= 8 contiguous children are tested by 32 lanes at once
//     (`test_cell`/`open_node`, List 2 PAPER.md:73-91), 4 coalesced float4 loads per
//     lane (boundary + multipole, issued together so an iteration costs one memory
//     latency);
//   * ballot/popc compaction sorts the children into: stack (opened nodes), a queue
//     of opened leaves, and a shared-memory chunk of un-opened cells' multipoles
//     (48-byte records);
//   * a chunk is evaluated as soon as it fills (FP32 FMA + one rsqrt.approx per
//     interaction), so no interaction list ever reaches global memory and there is
//     no count pass, no host scan, no second walk;
//   * lanes map to (list slice s, particle column p): a pass over m <= kPassCap particles
//     (ONE walk per group) picks S slices of q = floor(32/S) columns and
//     K = ceil(m / q) <= kMaxK particles per lane so that the issue slots per list entry
//     are minimal (tc_lanes.h); every list record is loaded from shared memory once per
//     lane and applied to the lane's particles: floor(K/2) PAIRS with packed FP32
//     instructions (FFMA2/FMUL2/FADD2: two particles per instruction) and, when K is
//     odd, one more particle with scalar instructions; slices are reduced with shuffles
//     at the end — the fix for the paper's 30 % thread utilisation.
// No tensor cores: this is not a dense contraction.
#include <cuda_runtime.h>

#include <cub/device/device_scan.cuh>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <mutex>
#include <string>

// This file is compiled TWICE into libtc_b200.so (tc_kernels_dense.cu includes it with other constants): the launch
// configuration of the fused kernel is a compile-time matter (warps per CTA, shared-memory capacities, registers), and no
// single one is best for every tree:
//   sparse (this file on its own): 4 CTAs x 4 warps per SM, 128 registers, 224-record chunks, no tail in the lane
//          mapping — many warps hide the walk's latency when groups are small and the walk is most of the work
//          (N_group = N_leaf = 16: 8.7 ms against 9.4; the tail code alone, never taken there, costs 3 %: registers);
//   dense  (tc_kernels_dense.cu):  4 CTAs x 3 warps per SM, 168 registers, 320-record chunks, tails of up to 4 particles —
//          fewer, longer evaluation rounds when groups are large (config 3 at N_group = 128: 5.65 ms against 5.74;
//          N = 2^24: 105.7 against 108.8).
// tc_api.cpp picks by the mean number of particles per group (crossover measured at ~24).  Everything that is not the
// fused kernel (two-pass variant, direct summation, kicks, FP32 peak) exists once, in the sparse build.  The builders'
// schedules use the lane table of tc_lanes.h with its defaults (the dense one): a cost model, not a contract.
#ifndef TC_CFG_NS
#define TC_CFG_NS sparse
#ifndef TC_MAXTAIL
#define TC_MAXTAIL 0
#endif
#endif

#include "tc_internal.h"
#include "tc_lanes.h"

namespace tc {
namespace {

#ifndef TC_MINB
#define TC_MINB 4
#endif
#ifndef TC_WALKB
#define TC_WALKB 2
#endif
constexpr int kWalkB = TC_WALKB;   // batches of 4 nodes (32 child tests) per walk iteration
#ifndef TC_BULK_BODIES
#define TC_BULK_BODIES 0         // 1: stage opened-leaf bodies with cp.async.bulk (1-D TMA) + mbarrier instead of ldg + sts
#endif
#ifndef TC_UNROLL2_MAXK
#define TC_UNROLL2_MAXK 2   // particle-cell loop: two records in flight up to this many particles per lane
#endif
#ifndef TC_CELLCAP
#define TC_CELLCAP 224
#endif
#ifndef TC_WARPS
#define TC_WARPS 4
#endif
constexpr int kWarpsPerCta = TC_WARPS;
constexpr int kCellCap = TC_CELLCAP;  // un-opened cells staged per warp before evaluation
#ifndef TC_LEAFQCAP
#define TC_LEAFQCAP 256
#endif
constexpr int kLeafQCap = TC_LEAFQCAP;   // opened-leaf ranges queued per warp
#ifndef TC_BODYCAP
#define TC_BODYCAP 384
#endif
constexpr int kBodyCap = TC_BODYCAP;   // bodies staged per warp per evaluation round
constexpr int kMaxKP = kMaxK / 2;  // particle PAIRS per lane (packed f32x2 arithmetic); an odd K adds one scalar particle
constexpr unsigned kFull = 0xffffffffu;

struct __align__(16) CellRec {   // one un-opened cell: 48 bytes
  float4 xm;                     // (X, Y, Z, M)
  float4 q0;                     // (Qxx, Qyy, Qzz, Qxy)
  float2 q1;                     // (Qxz, Qyz)
  float2 pad;
};

struct BodyStage {
  float4 body[kBodyCap];         // (x, y, z, m)
  int bidx[kBodyCap];            // flattened body indices of the current round
};

template <int STK>
struct __align__(16) WarpSmem {
  union {                        // cells are flushed before bodies are staged
    CellRec cell[kCellCap];
    BodyStage bs;
  } u;
  int2 leafq[kLeafQCap];         // (first_body, n_body)
  uint32_t stack[STK];           // nodes to expand: first_child << 3 | (n_child - 1)
#if TC_BULK_BODIES
  unsigned long long mbar;       // mbarrier of the bulk copies that stage opened-leaf bodies (A/B of DESIGN.md section 6)
  unsigned long long pad_;
#endif
};

// Lane mapping of a pass over m particles (tc_lanes.h): S slices x q columns, K particles per lane
__constant__ LaneTable c_lanes = LaneTable();

__device__ __forceinline__ float rsqrt_approx(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// ---- packed FP32 pairs (sm_100a FFMA2 / FMUL2 / FADD2): one instruction does the arithmetic of
// the lane's TWO particles (lo = even, hi = odd) at half the issue cost of two scalar instructions.
// A scalar operand (a field of the list record) is broadcast by the hardware (`R.F32` operand form).
typedef unsigned long long f2;
__device__ __forceinline__ f2 pk(float lo, float hi) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ f2 bc(float x) { return pk(x, x); }
__device__ __forceinline__ float lo(f2 v) { float a; asm("{ .reg .b32 t; mov.b64 {%0, t}, %1; }" : "=f"(a) : "l"(v)); return a; }
__device__ __forceinline__ float hi(f2 v) { float b; asm("{ .reg .b32 t; mov.b64 {t, %0}, %1; }" : "=f"(b) : "l"(v)); return b; }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2 sub2(f2 a, f2 b) { f2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { f2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { f2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }

struct Acc2 {      // accumulators of a particle pair; `npot` accumulates -phi (negated at write-back)
  f2 ax, ay, az, npot;
};
struct Pos2 {      // positions of a particle pair
  f2 x, y, z;
};
struct Acc1 {      // the same for the single particle of an odd K
  float ax, ay, az, npot;
};
struct Pos1 {
  float x, y, z;
};
// The lane's particles of the current pass and their accumulators: floor(K/2) pairs and, K odd, one more particle
struct PassState {
  Pos2 P[kMaxKP];
  Acc2 A[kMaxKP];
  Pos1 p1;
  Acc1 a1;
};

// particle-cell: monopole + traceless quadrupole (O6), d = X - x_i:
//   a   += M d/s^3 - Q d/s^5 + (5/2)(d^T Q d) d/s^7
//   phi += -M/s - (1/2)(d^T Q d)/s^5
// The record carries -Q (nq0, nq1; negated on the host), so no operand needs a run-time negation.
// 33 packed FP32 instructions + 2 MUFU per PAIR of interactions.
__device__ __forceinline__ void pc_interact(const Pos2& p, float eps2, const float4 xm, const float4 nq0,
                                            const float2 nq1, Acc2& a) {
  const f2 dx = sub2(bc(xm.x), p.x), dy = sub2(bc(xm.y), p.y), dz = sub2(bc(xm.z), p.z);
  const f2 s2 = fma2(dz, dz, fma2(dy, dy, fma2(dx, dx, bc(eps2))));
  const f2 ri = pk(rsqrt_approx(lo(s2)), rsqrt_approx(hi(s2)));
  const f2 ri2 = mul2(ri, ri);
  const f2 ri3 = mul2(ri, ri2);
  const f2 ri5 = mul2(ri3, ri2);
  // -(Q d), column by column: the three products of one d_k are consecutive and share it (operand reuse cache:
  // the register file delivers two 32-bit operands per lane and cycle, an FFMA2 with three register pairs needs six)
  f2 gx = mul2(bc(nq0.x), dx), gy = mul2(bc(nq0.w), dx), gz = mul2(bc(nq1.x), dx);
  gx = fma2(bc(nq0.w), dy, gx); gy = fma2(bc(nq0.y), dy, gy); gz = fma2(bc(nq1.y), dy, gz);
  gx = fma2(bc(nq1.x), dz, gx); gy = fma2(bc(nq1.y), dz, gy); gz = fma2(bc(nq0.z), dz, gz);
  const f2 g = fma2(dz, gz, fma2(dy, gy, mul2(dx, gx)));                         // -(d^T Q d)
  const f2 t5 = mul2(g, ri5);
  a.npot = fma2(bc(xm.w), ri, a.npot);
  a.npot = fma2(bc(-0.5f), t5, a.npot);
  const f2 c = fma2(bc(-2.5f), mul2(t5, ri2), mul2(bc(xm.w), ri3));
  a.ax = fma2(c, dx, a.ax); a.ay = fma2(c, dy, a.ay); a.az = fma2(c, dz, a.az);
  a.ax = fma2(ri5, gx, a.ax); a.ay = fma2(ri5, gy, a.ay); a.az = fma2(ri5, gz, a.az);
}
// the same interaction for ONE particle: 33 scalar FP32 instructions + 1 MUFU (the issue cost of half a pair)
__device__ __forceinline__ void pc_interact(const Pos1& p, float eps2, const float4 xm, const float4 nq0,
                                            const float2 nq1, Acc1& a) {
  const float dx = __fsub_rn(xm.x, p.x), dy = __fsub_rn(xm.y, p.y), dz = __fsub_rn(xm.z, p.z);
  const float s2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmaf_rn(dx, dx, eps2)));
  const float ri = rsqrt_approx(s2);
  const float ri2 = __fmul_rn(ri, ri);
  const float ri3 = __fmul_rn(ri, ri2);
  const float ri5 = __fmul_rn(ri3, ri2);
  const float gx = __fmaf_rn(nq1.x, dz, __fmaf_rn(nq0.w, dy, __fmul_rn(nq0.x, dx)));
  const float gy = __fmaf_rn(nq1.y, dz, __fmaf_rn(nq0.y, dy, __fmul_rn(nq0.w, dx)));
  const float gz = __fmaf_rn(nq0.z, dz, __fmaf_rn(nq1.y, dy, __fmul_rn(nq1.x, dx)));
  const float g = __fmaf_rn(dz, gz, __fmaf_rn(dy, gy, __fmul_rn(dx, gx)));
  const float t5 = __fmul_rn(g, ri5);
  a.npot = __fmaf_rn(xm.w, ri, a.npot);
  a.npot = __fmaf_rn(-0.5f, t5, a.npot);
  const float c = __fmaf_rn(-2.5f, __fmul_rn(t5, ri2), __fmul_rn(xm.w, ri3));
  a.ax = __fmaf_rn(c, dx, a.ax); a.ay = __fmaf_rn(c, dy, a.ay); a.az = __fmaf_rn(c, dz, a.az);
  a.ax = __fmaf_rn(ri5, gx, a.ax); a.ay = __fmaf_rn(ri5, gy, a.ay); a.az = __fmaf_rn(ri5, gz, a.az);
}

// particle-particle, Plummer softening (O6), d = x_j - x_i:
//   a += m_j d/s^3, phi += -m_j/s.   13 packed FP32 instructions + 2 MUFU per pair of interactions.
// kEps0: eps == 0, coincident pairs (and the particle itself) contribute nothing.
template <bool kEps0>
__device__ __forceinline__ void pp_interact(const Pos2& p, float eps2, const float4 b, Acc2& a) {
  const f2 dx = sub2(bc(b.x), p.x), dy = sub2(bc(b.y), p.y), dz = sub2(bc(b.z), p.z);
  const f2 s2 = fma2(dz, dz, fma2(dy, dy, fma2(dx, dx, bc(eps2))));
  float r0 = rsqrt_approx(lo(s2)), r1 = rsqrt_approx(hi(s2));
  if (kEps0) { r0 = (lo(s2) > 0.f) ? r0 : 0.f; r1 = (hi(s2) > 0.f) ? r1 : 0.f; }
  const f2 ri = pk(r0, r1);
  const f2 ri2 = mul2(ri, ri);
  const f2 mr = mul2(bc(b.w), ri);
  const f2 mr3 = mul2(mr, ri2);
  a.npot = add2(a.npot, mr);
  a.ax = fma2(mr3, dx, a.ax); a.ay = fma2(mr3, dy, a.ay); a.az = fma2(mr3, dz, a.az);
}
template <bool kEps0>
__device__ __forceinline__ void pp_interact(const Pos1& p, float eps2, const float4 b, Acc1& a) {
  const float dx = __fsub_rn(b.x, p.x), dy = __fsub_rn(b.y, p.y), dz = __fsub_rn(b.z, p.z);
  const float s2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmaf_rn(dx, dx, eps2)));
  float ri = rsqrt_approx(s2);
  if (kEps0) ri = (s2 > 0.f) ? ri : 0.f;
  const float ri2 = __fmul_rn(ri, ri);
  const float mr = __fmul_rn(b.w, ri);
  const float mr3 = __fmul_rn(mr, ri2);
  a.npot = __fadd_rn(a.npot, mr);
  a.ax = __fmaf_rn(mr3, dx, a.ax); a.ay = __fmaf_rn(mr3, dy, a.ay); a.az = __fmaf_rn(mr3, dz, a.az);
}

// The same pair of interactions with one mass per half: the half whose particle IS the staged body gets mass 0 and the
// pair (i, i) contributes exactly nothing (O6: the sums run over j != i).  eps > 0 only: with eps = 0 the pair is masked by s^2 = 0.
__device__ __forceinline__ void pp_interact_masked(const Pos2& p, float eps2, const float4 b, float m0, float m1, Acc2& a) {
  const f2 dx = sub2(bc(b.x), p.x), dy = sub2(bc(b.y), p.y), dz = sub2(bc(b.z), p.z);
  const f2 s2 = fma2(dz, dz, fma2(dy, dy, fma2(dx, dx, bc(eps2))));
  const f2 ri = pk(rsqrt_approx(lo(s2)), rsqrt_approx(hi(s2)));
  const f2 ri2 = mul2(ri, ri);
  const f2 mr = mul2(pk(m0, m1), ri);
  const f2 mr3 = mul2(mr, ri2);
  a.npot = add2(a.npot, mr);
  a.ax = fma2(mr3, dx, a.ax); a.ay = fma2(mr3, dy, a.ay); a.az = fma2(mr3, dz, a.az);
}

// Lane mapping of one pass over m <= kPassCap particles of a group (tc_lanes.h):
// lane = s * q + p, q = floor(32 / S); the lane's j-th particle is j * q + p, j < K.
struct Lanes {
  int S, q, K;   // warp-uniform
  int s, p;      // this lane's slice and particle column
  bool active;   // lane < S * q
  // the TAIL of the pass (tc_lanes.h): its last mB particles, tree-order indices tail .. tail + mB - 1, are not in the
  // mapping; every lane applies its own records (S = 32, q = 1) to all of them.  The mapping covers mA = m - mB.
  int mA, mB, tail;
  const float4* part;
};

// one list record applied to the lane's KP pairs (+ ODD single particle)
template <int KP, bool ODD>
__device__ __forceinline__ void pc_apply(PassState& st, float eps2, const float4 a, const float4 b, const float2 c) {
#pragma unroll
  for (int j = 0; j < KP; j++) pc_interact(st.P[j], eps2, a, b, c, st.A[j]);
  if (ODD) pc_interact(st.p1, eps2, a, b, c, st.a1);
}
template <int KP, bool ODD, bool kEps0>
__device__ __forceinline__ void pp_apply(PassState& st, float eps2, const float4 b) {
#pragma unroll
  for (int j = 0; j < KP; j++) pp_interact<kEps0>(st.P[j], eps2, b, st.A[j]);
  if (ODD) pp_interact<kEps0>(st.p1, eps2, b, st.a1);
}

// Un-opened cells (List 3): slice s takes records s, s+S, s+2S, ...
// Each record is loaded once and applied to the lane's K = 2 KP + ODD particles.
template <int KP, bool ODD>
__device__ __forceinline__ void eval_cells_k(const CellRec* __restrict__ rec, int cnt, float eps2, const Lanes& L, PassState& st) {
  if (!L.active) return;
  // pointer walk (one add per record, no index multiply)
  const CellRec* r0 = rec + L.s;
  const CellRec* const end = rec + cnt;
  const int sd = L.S;
  if (2 * KP + ODD <= TC_UNROLL2_MAXK) {
    for (; r0 + sd < end; r0 += 2 * sd) {          // two records in flight
      const CellRec* r1 = r0 + sd;
      const float4 a0 = r0->xm, b0 = r0->q0; const float2 c0 = r0->q1;
      const float4 a1 = r1->xm, b1 = r1->q0; const float2 c1 = r1->q1;
      pc_apply<KP, ODD>(st, eps2, a0, b0, c0);
      pc_apply<KP, ODD>(st, eps2, a1, b1, c1);
    }
    if (r0 < end) {
      const float4 a0 = r0->xm, b0 = r0->q0; const float2 c0 = r0->q1;
      pc_apply<KP, ODD>(st, eps2, a0, b0, c0);
    }
  } else {
    for (; r0 < end; r0 += sd) {
      const float4 a0 = r0->xm, b0 = r0->q0; const float2 c0 = r0->q1;
      pc_apply<KP, ODD>(st, eps2, a0, b0, c0);
    }
  }
}

// Monopole-only variant (R22, option "quadrupole" = 0): a cell is a point mass (X, M)
template <int KP, bool ODD, bool kEps0>
__device__ __forceinline__ void eval_cells_mono_k(const CellRec* __restrict__ rec, int cnt, float eps2, const Lanes& L, PassState& st) {
  if (!L.active) return;
  const int sd = L.S;
  for (int e = L.s; e < cnt; e += sd) pp_apply<KP, ODD, kEps0>(st, eps2, rec[e].xm);
}

template <int KP, bool ODD, bool kEps0>
__device__ __forceinline__ void eval_bodies_k(const float4* __restrict__ body, int cnt, float eps2, const Lanes& L, PassState& st) {
  if (!L.active) return;
  const float4* b = body + L.s;                  // pointer walk, as in eval_cells_k
  const float4* const end = body + cnt;
  const int sd = L.S;
  if (2 * KP + ODD <= 2) {
    for (; b + 3 * sd < end; b += 4 * sd) {        // four bodies in flight
      const float4 b0 = b[0], b1 = b[sd], b2 = b[2 * sd], b3 = b[3 * sd];
      pp_apply<KP, ODD, kEps0>(st, eps2, b0); pp_apply<KP, ODD, kEps0>(st, eps2, b1);
      pp_apply<KP, ODD, kEps0>(st, eps2, b2); pp_apply<KP, ODD, kEps0>(st, eps2, b3);
    }
  } else {
    for (; b + sd < end; b += 2 * sd) {            // two bodies in flight
      const float4 b0 = b[0], b1 = b[sd];
      pp_apply<KP, ODD, kEps0>(st, eps2, b0); pp_apply<KP, ODD, kEps0>(st, eps2, b1);
    }
  }
  for (; b < end; b += sd) pp_apply<KP, ODD, kEps0>(st, eps2, b[0]);
}

// The round that stages the pass's OWN particles (at most a few per group: its own leaves): the only place where a particle can
// meet itself.  The staged body's tree index (bidx) is compared with the lane's particles' and the self pair gets mass 0 —
// so -m/eps never enters the fp32 potential sum (it used to be added and taken out again at write-back, which cost
// ~6e-8 m/eps of absolute accuracy).  Plain loop: these rounds are a few per cent of the particle-particle work.
template <int KP, bool ODD>
__device__ __forceinline__ void eval_bodies_self_k(const float4* __restrict__ body, const int* __restrict__ bidx, int cnt, float eps2,
                                                   const Lanes& L, PassState& st) {
  if (!L.active) return;
  const int me = L.tail - L.mA + L.p;              // tree index of the lane's particle 0; particle j is me + j * q
  for (int e = L.s; e < cnt; e += L.S) {
    const float4 b = body[e];
    const int rel = bidx[e] - me;
#pragma unroll
    for (int j = 0; j < KP; j++)
      pp_interact_masked(st.P[j], eps2, b, rel == 2 * j * L.q ? 0.f : b.w, rel == (2 * j + 1) * L.q ? 0.f : b.w, st.A[j]);
    if (ODD) pp_interact<false>(st.p1, eps2, make_float4(b.x, b.y, b.z, rel == 2 * KP * L.q ? 0.f : b.w), st.a1);
  }
}

// K is warp-uniform: one branch to the instantiation for this pass's particles per lane
enum { kEvalCells = 0, kEvalMono = 1, kEvalBodies = 2, kEvalBodiesSelf = 3 };
template <int WHAT, bool kEps0, int K = 1>
__device__ __forceinline__ void eval_dispatch(const void* list, int cnt, float eps2, const Lanes& L, PassState& st, const int* bidx = nullptr) {
  if (K == kMaxK || L.K == K) {
    if (WHAT == kEvalBodiesSelf) eval_bodies_self_k<K / 2, (K & 1) != 0>(static_cast<const float4*>(list), bidx, cnt, eps2, L, st);
    else if (WHAT == kEvalCells) eval_cells_k<K / 2, (K & 1) != 0>(static_cast<const CellRec*>(list), cnt, eps2, L, st);
    else if (WHAT == kEvalMono) eval_cells_mono_k<K / 2, (K & 1) != 0, kEps0>(static_cast<const CellRec*>(list), cnt, eps2, L, st);
    else eval_bodies_k<K / 2, (K & 1) != 0, kEps0>(static_cast<const float4*>(list), cnt, eps2, L, st);
  } else if constexpr (K < kMaxK) {
    eval_dispatch<WHAT, kEps0, K + 1>(list, cnt, eps2, L, st, bidx);
  }
}
// The tail particles (Lanes::mB of them): lane l takes list entries l, l + 32, ... and applies each to ALL tail particles in
// scalar arithmetic.  Their accumulators are the halves of the TOP register pairs of the state (the lane table leaves
// those pairs to the tail): unpacked to scalars for the loop, packed again after it.
template <int MB, int WHAT, bool kEps0>
__device__ __forceinline__ void eval_tail_m(const void* list, int cnt, float eps2, const Lanes& L, PassState& st, int lane,
                                            const int* bidx = nullptr) {
  Pos1 p[MB];
  Acc1 a[MB];
#pragma unroll
  for (int j = 0; j < MB; j++) {
    const float4 m0 = __ldg(L.part + L.tail + j);          // warp-uniform address
    p[j].x = m0.x; p[j].y = m0.y; p[j].z = m0.z;
    const Acc2& a2 = st.A[kMaxKP - 1 - (j >> 1)];
    if (j & 1) { a[j].ax = hi(a2.ax); a[j].ay = hi(a2.ay); a[j].az = hi(a2.az); a[j].npot = hi(a2.npot); }
    else { a[j].ax = lo(a2.ax); a[j].ay = lo(a2.ay); a[j].az = lo(a2.az); a[j].npot = lo(a2.npot); }
  }
  if (WHAT == kEvalBodiesSelf) {                      // (see eval_bodies_self_k: tail particle j has tree index L.tail + j)
    for (int e = lane; e < cnt; e += 32) {
      const float4 bb = static_cast<const float4*>(list)[e];
      const int rel = bidx[e] - L.tail;
#pragma unroll
      for (int j = 0; j < MB; j++) pp_interact<kEps0>(p[j], eps2, make_float4(bb.x, bb.y, bb.z, rel == j ? 0.f : bb.w), a[j]);
    }
  } else if (WHAT == kEvalBodies) {
    const float4* b = static_cast<const float4*>(list) + lane;
    const float4* const end = static_cast<const float4*>(list) + cnt;
    for (; b < end; b += 32) {
      const float4 bb = b[0];
#pragma unroll
      for (int j = 0; j < MB; j++) pp_interact<kEps0>(p[j], eps2, bb, a[j]);
    }
  } else {
    const CellRec* r = static_cast<const CellRec*>(list) + lane;
    const CellRec* const end = static_cast<const CellRec*>(list) + cnt;
    for (; r < end; r += 32) {
      const float4 xm = r->xm, q0 = r->q0; const float2 q1 = r->q1;
#pragma unroll
      for (int j = 0; j < MB; j++) {
        if (WHAT == kEvalMono) pp_interact<kEps0>(p[j], eps2, xm, a[j]);
        else pc_interact(p[j], eps2, xm, q0, q1, a[j]);
      }
    }
  }
#pragma unroll
  for (int jj = 0; jj < (MB + 1) / 2; jj++) {
    Acc2& a2 = st.A[kMaxKP - 1 - jj];
    const int j0 = 2 * jj, j1 = (2 * jj + 1 < MB) ? 2 * jj + 1 : 2 * jj;
    const bool two = 2 * jj + 1 < MB;
    // (+ 0 through FADD2: see setup_pass)
    a2.ax = add2(pk(a[j0].ax, two ? a[j1].ax : 0.f), bc(0.f)); a2.ay = add2(pk(a[j0].ay, two ? a[j1].ay : 0.f), bc(0.f));
    a2.az = add2(pk(a[j0].az, two ? a[j1].az : 0.f), bc(0.f)); a2.npot = add2(pk(a[j0].npot, two ? a[j1].npot : 0.f), bc(0.f));
  }
}
template <int WHAT, bool kEps0, int MB = 1>
__device__ __forceinline__ void eval_tail(const void* list, int cnt, float eps2, const Lanes& L, PassState& st, int lane,
                                          const int* bidx = nullptr) {
  if constexpr (kMaxTail >= 1) {
    if (MB == kMaxTail || L.mB == MB) eval_tail_m<MB, WHAT, kEps0>(list, cnt, eps2, L, st, lane, bidx);
    else if constexpr (MB < kMaxTail) eval_tail<WHAT, kEps0, MB + 1>(list, cnt, eps2, L, st, lane, bidx);
  }
}

template <bool kEps0>
__device__ __forceinline__ void eval_cells(const CellRec* rec, int cnt, float eps2, const Lanes& L, PassState& st, bool mono, int lane) {
  if (mono) eval_dispatch<kEvalMono, kEps0>(rec, cnt, eps2, L, st);
  else eval_dispatch<kEvalCells, kEps0>(rec, cnt, eps2, L, st);
  if (L.mB) {                                          // warp-uniform
    if (mono) eval_tail<kEvalMono, kEps0>(rec, cnt, eps2, L, st, lane);
    else eval_tail<kEvalCells, kEps0>(rec, cnt, eps2, L, st, lane);
  }
}

// Opened leaves (List 4): flatten the queued (first, n) ranges into
// body indices, gather the bodies with one coalesced float4 load per lane, evaluate.
// mbar != nullptr (build with TC_BULK_BODIES): the ranges are contiguous runs of 16-byte records, so every lane
// moves its range with ONE cp.async.bulk (1-D TMA copy, no register staging) completing on the warp's mbarrier.
[[maybe_unused]] __device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
template <bool kEps0>
__device__ __forceinline__ void eval_leaves(BodyStage& bs, const int2* leafq, int nq, const float4* __restrict__ part,
                                            float eps2, const Lanes& L, PassState& st, int lane,
                                            unsigned long long* mbar = nullptr, unsigned* phase = nullptr) {
  for (int r0 = 0; r0 < nq; r0 += 32) {
    int f = 0, n = 0;
    if (r0 + lane < nq) { const int2 r = leafq[r0 + lane]; f = r.x; n = r.y; }
    int incl = n;   // inclusive scan of n
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(kFull, incl, d); if (lane >= d) incl += t; }
    const int off = incl - n;
    const int total = __shfl_sync(kFull, incl, 31);
    for (int base = 0; base < total; base += kBodyCap) {
      const int k0 = max(0, base - off), k1 = min(n, base + kBodyCap - off);
      const int cnt = min(kBodyCap, total - base);
      // does this round stage particles of the pass itself, [own_f, own_e)?  (warp-uniform; eps = 0 masks the pair by s^2 = 0)
      const int own_f = L.tail - L.mA, own_e = L.tail + L.mB;
      const bool self_round = !kEps0 && __any_sync(kFull, k1 > k0 && f + k0 < own_e && f + k1 > own_f);
#if TC_BULK_BODIES
      if (mbar) {
        const unsigned bar = smem_u32(mbar);
        // the generic-proxy accesses of the staging area (previous round, or the cell chunk) come before the async writes
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        if (lane == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(cnt * 16) : "memory");
        __syncwarp();
        if (k1 > k0)
          asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                       :: "r"(smem_u32(bs.body + (off + k0 - base))), "l"(part + f + k0), "r"((k1 - k0) * 16), "r"(bar) : "memory");
        unsigned ok;
        do {
          asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                       : "=r"(ok) : "r"(bar), "r"(*phase) : "memory");
        } while (!ok);
        *phase ^= 1u;
        if (self_round) { for (int k = k0; k < k1; k++) bs.bidx[off + k - base] = f + k; __syncwarp(); }
      } else
#endif
      {
        for (int k = k0; k < k1; k++) bs.bidx[off + k - base] = f + k;
        __syncwarp();
        for (int t = lane; t < cnt; t += 32) bs.body[t] = __ldg(part + bs.bidx[t]);
        __syncwarp();
      }
      if (self_round) {
        eval_dispatch<kEvalBodiesSelf, kEps0>(bs.body, cnt, eps2, L, st, bs.bidx);
        if (L.mB) eval_tail<kEvalBodiesSelf, kEps0>(bs.body, cnt, eps2, L, st, lane, bs.bidx);
      } else {
        eval_dispatch<kEvalBodies, kEps0>(bs.body, cnt, eps2, L, st);
        if (L.mB) eval_tail<kEvalBodies, kEps0>(bs.body, cnt, eps2, L, st, lane);
      }
      __syncwarp();
    }
  }
}

// Lane mapping, particles and zeroed accumulators of one pass over particles [first, first + m)
__device__ __forceinline__ void setup_pass(Lanes& L, PassState& st, const float4* __restrict__ part, int first, int m, int lane) {
  const LaneMap lm = c_lanes.map[m];
  L.S = lm.S; L.q = lm.q; L.K = lm.K;
  L.mB = lm.mB; L.mA = m - L.mB; L.tail = first + L.mA; L.part = part;
  m = L.mA;                                              // the mapping covers the particles in front of the tail
  L.s = lane / L.q;
  L.p = lane - L.s * L.q;
  L.active = L.s < L.S;
  // slots beyond m compute on a copy of the pass's first particle; never written back
#pragma unroll
  for (int j = 0; j < kMaxKP; j++) {
    st.A[j].ax = st.A[j].ay = st.A[j].az = st.A[j].npot = 0ull;  // (+0.f, +0.f)
    const int t0 = 2 * j * L.q + L.p, t1 = t0 + L.q;
    const float4 m0 = __ldg(part + first + ((L.active && t0 < m) ? t0 : 0));
    const float4 m1 = __ldg(part + first + ((L.active && t1 < m) ? t1 : 0));
    // (+ 0 through FADD2: the pair is then the result of a real instruction and stays in one aligned
    // register pair; a bare mov.b64 is re-materialised with two MOVs in front of every use)
    st.P[j].x = add2(pk(m0.x, m1.x), bc(0.f)); st.P[j].y = add2(pk(m0.y, m1.y), bc(0.f));
    st.P[j].z = add2(pk(m0.z, m1.z), bc(0.f));
  }
  {  // K odd: the lane's last particle, K - 1, is evaluated with scalar instructions
    const int t = (L.K - 1) * L.q + L.p;
    const float4 m0 = __ldg(part + first + ((L.active && t < m) ? t : 0));
    st.p1.x = m0.x; st.p1.y = m0.y; st.p1.z = m0.z;
    st.a1.ax = st.a1.ay = st.a1.az = st.a1.npot = 0.f;
  }
}

// Where the results of a pass go.  Default: the caller's order (acc [n,3], pot [n], counts [n]).  A SHARD of a
// multi-GPU evaluation writes (ax, ay, az, phi) rows and (n_pc, n_pp) pairs COMPACTLY instead,
// row = the group's offset in this rank's shard + the particle's index in the group: only this rank's particles,
// coalesced 16-byte stores, ready for one all-gather.
struct ShardOut {
  float4* out4 = nullptr;          // [n_slots] or nullptr (not a shard)
  int2* cnt2 = nullptr;            // [n_slots] or nullptr
  const int32_t* off = nullptr;    // [n_groups] by schedule position: first row of the group in its rank's shard
};

// A6: reduce the slices of every particle, write back in the caller's order (or into the shard's compact rows).
// kAdd: add to what is already there (second evaluation kernel of the two-pass variant);
// kSelf: the particles met themselves once in the particle-particle part (remove -m/eps again).
// one particle's result: tree-order index t (row tq of the group), to the caller's order or to the shard's compact rows
template <bool kAdd, bool kSelf>
__device__ __forceinline__ void store_particle(int t, int tq, float ax, float ay, float az, float ph, const float4* __restrict__ part,
                                               const int32_t* __restrict__ orig, float eps2, float* __restrict__ acc,
                                               float* __restrict__ pot, int32_t* __restrict__ out_cnt, int cnt_value,
                                               int32_t* __restrict__ out_cnt2, int cnt2_value, bool self_met,
                                               float4* __restrict__ rows, int2* __restrict__ row_cnt) {
  (void)eps2; (void)self_met;   // (the self pair is excluded where it would occur: eval_bodies_self_k)
  if (!kAdd && rows) {                                                     // shard: compact rows, tree order inside the group
    rows[tq] = make_float4(ax, ay, az, ph);
    if (row_cnt) row_cnt[tq] = make_int2(cnt_value, cnt2_value);
    return;
  }
  const int i = __ldg(orig + t);
  float* a3 = acc + 3 * (size_t)i;
  if (kAdd) { a3[0] += ax; a3[1] += ay; a3[2] += az; if (pot) pot[i] += ph; }
  else { a3[0] = ax; a3[1] = ay; a3[2] = az; if (pot) pot[i] = ph; }
  out_cnt[i] = cnt_value;
  if (out_cnt2) out_cnt2[i] = cnt2_value;
}

template <bool kAdd, bool kSelf>
__device__ __forceinline__ void write_back(const Lanes& L, const PassState& st, const float4* __restrict__ part,
                                           const int32_t* __restrict__ orig, int first, int m, float eps2, int lane,
                                           float* __restrict__ acc, float* __restrict__ pot, int32_t* __restrict__ out_cnt,
                                           int cnt_value, int32_t* __restrict__ out_cnt2 = nullptr, int cnt2_value = 0,
                                           bool self_met = true, float4* __restrict__ rows = nullptr, int2* __restrict__ row_cnt = nullptr) {
  // ---- the particles of the lane mapping: slices reduced with shuffles
#pragma unroll
  for (int j = 0; j < kMaxK; j++) {
    if (j >= L.K) break;                             // warp-uniform
    const Acc2& a2 = st.A[j >> 1];
    float ax, ay, az, ph;
    if (j & 1) { ax = hi(a2.ax); ay = hi(a2.ay); az = hi(a2.az); ph = -hi(a2.npot); }
    else { ax = lo(a2.ax); ay = lo(a2.ay); az = lo(a2.az); ph = -lo(a2.npot); }
    if (!(j & 1) && j == L.K - 1) { ax = st.a1.ax; ay = st.a1.ay; az = st.a1.az; ph = -st.a1.npot; }   // K odd: the single particle
    for (int w = 1; w < L.S; w <<= 1) {
      const float ox = __shfl_down_sync(kFull, ax, w * L.q), oy = __shfl_down_sync(kFull, ay, w * L.q);
      const float oz = __shfl_down_sync(kFull, az, w * L.q), op = __shfl_down_sync(kFull, ph, w * L.q);
      if ((L.s % (2 * w)) == 0 && L.s + w < L.S) { ax += ox; ay += oy; az += oz; ph += op; }
    }
    const int tq = j * L.q + lane;
    if (lane < L.q && tq < L.mA)
      store_particle<kAdd, kSelf>(first + tq, tq, ax, ay, az, ph, part, orig, eps2, acc, pot, out_cnt, cnt_value, out_cnt2, cnt2_value,
                                  self_met, rows, row_cnt);
  }
  // ---- the tail: every lane holds a partial sum of every tail particle (halves of the top register pairs)
#pragma unroll
  for (int j = 0; j < kMaxTail; j++) {
    if (j >= L.mB) break;                            // warp-uniform
    const Acc2& a2 = st.A[kMaxKP - 1 - (j >> 1)];
    float ax, ay, az, ph;
    if (j & 1) { ax = hi(a2.ax); ay = hi(a2.ay); az = hi(a2.az); ph = -hi(a2.npot); }
    else { ax = lo(a2.ax); ay = lo(a2.ay); az = lo(a2.az); ph = -lo(a2.npot); }
#pragma unroll
    for (int w = 16; w >= 1; w >>= 1) {
      ax += __shfl_xor_sync(kFull, ax, w); ay += __shfl_xor_sync(kFull, ay, w);
      az += __shfl_xor_sync(kFull, az, w); ph += __shfl_xor_sync(kFull, ph, w);
    }
    if (lane == 0)
      store_particle<kAdd, kSelf>(L.tail + j, L.mA + j, ax, ay, az, ph, part, orig, eps2, acc, pot, out_cnt, cnt_value, out_cnt2,
                                  cnt2_value, self_met, rows, row_cnt);
  }
  (void)m;
}

// Global interaction lists of the paper-literal two-pass variant (count, scan, write).
struct ListIO {
  unsigned long long *cnt_c, *cnt_l;        // [n_groups]  pass 1: cells / opened-leaf ranges per group
  const unsigned long long *off_c, *off_l;  // [n_groups + 1]  exclusive scans of the counts
  int* cells;                       // cell ids
  int2* leaves;                     // (first_body, n_body)
  int* leaf_bodies;                 // [n_groups] bodies of the opened leaves (n_pp + 1)
};

enum { kFused = 0, kCount = 1, kWrite = 2 };
enum { kFlagWalkOnly = 1, kFlagComRule = 2, kFlagMonopole = 4, kFlagGroupBox = 8 };   // run-time variants of a launch

// kPlain: the launch uses none of the variant readings (R21-R23), so their selects are compiled out
template <int STK, bool kEps0, int MODE = kFused, bool kPlain = false>
__global__ void __launch_bounds__(kWarpsPerCta * 32, TC_MINB)
forces_kernel(const float4* __restrict__ bnd, const float4* __restrict__ xm, const float4* __restrict__ q0,
              const float4* __restrict__ q1, const float4* __restrict__ part, const int32_t* __restrict__ orig,
              const int4* __restrict__ grp, const float4* __restrict__ gbox, int n_groups, float theta, float eps,
              float* __restrict__ acc, float* __restrict__ pot, int32_t* __restrict__ out_npc,
              int32_t* __restrict__ out_npp, DeviceCounters* __restrict__ ctr, uint32_t* __restrict__ spill_all,
              int spill_cap, int flags, ListIO lio, int shard_rank, int shard_count, ShardOut sho) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  WarpSmem<STK>& sm = reinterpret_cast<WarpSmem<STK>*>(smem_raw)[warp];
  uint32_t* spill = spill_all + (size_t)(blockIdx.x * kWarpsPerCta + warp) * (size_t)spill_cap;
  const float eps2 = eps * eps;
  const float th2 = __fmul_rn(theta, theta);
  unsigned long long* mbar = nullptr;
  unsigned bulk_phase = 0;
#if TC_BULK_BODIES
  if (MODE == kFused) {
    mbar = &sm.mbar;
    if (lane == 0) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(mbar)) : "memory");
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
  }
#endif
  const unsigned lt_mask = (1u << lane) - 1u;
  const bool walk_only = flags & kFlagWalkOnly;
  const bool com_rule = !kPlain && (flags & kFlagComRule), mono = !kPlain && (flags & kFlagMonopole);
  const bool group_box = !kPlain && (flags & kFlagGroupBox);

  // root: a leaf root is never tested (O5) — its bodies are the whole leaf list
  const float4 root_b = __ldg(bnd);
  const float4 root_l = __ldg(q1);
  const bool root_leaf = __float_as_int(root_b.w) < 0;
  const int root_a = __float_as_int(root_l.z), root_n = __float_as_int(root_l.w);

  while (true) {
    int g = 0;
    if (lane == 0) g = (int)atomicAdd(&ctr->next_group, 1u);
    g = __shfl_sync(kFull, g, 0);
    // multi-GPU sharding: this launch takes the schedule positions rank, rank + count, ...
    // (neighbours in the cost-ordered schedule cost about the same, so the shards are balanced)
    if (g >= (n_groups - shard_rank + shard_count - 1) / shard_count) break;
    g = g * shard_count + shard_rank;
    const int shard_row = sho.out4 ? __ldg(sho.off + g) : 0;   // first compact row of this group (shards only)
    g = __ldg(&grp[g].w);                    // schedule: costly groups first (tc_build)
    const int4 G = __ldg(grp + g);           // (cell, first_body, n_body, -)
    const float4 gb = __ldg(bnd + G.x);
    const float gbx = gb.x, gby = gb.y, gbz = gb.z, gh = fabsf(gb.w);
    // the group's side of the test: the half side of its cube (R9) or, variant R23, the half extents of its tight box
    float ghx = gh, ghy = gh, ghz = gh;
    if (group_box) { const float4 e = __ldg(gbox + g); ghx = e.x; ghy = e.y; ghz = e.z; }

    // ONE walk per group.  Only a group of more than kPassCap particles (a level-21 leaf of
    // coincident particles, or N_group > kPassCap) is walked once per kPassCap of them.
    for (int pb = 0; pb < G.z; pb += kPassCap) {
      const int m = min(kPassCap, G.z - pb);
      Lanes L;
      PassState ps;
      if (MODE == kFused) setup_pass(L, ps, part, G.y + pb, m, lane);
      unsigned long long woff_c = 0, woff_l = 0;         // MODE kWrite: where this group's lists start
      if (MODE == kWrite) { woff_c = lio.off_c[g]; woff_l = lio.off_l[g]; }

      int ssz = 0, spill_sz = 0, ccnt = 0, lq = 0;
      int n_pc = 0, n_pp = 0, n_open = 0;                // list entries so far; n_open: opened cells (leaves + nodes)
      int n_spills = 0, n_lr = 0;                        // n_lr: opened-leaf ranges so far
      bool overflow = false;
      // Did the pass's particles meet themselves in the particle-particle part?  Always, under the default
      // rule (the boxes of the group and of its ancestors overlap, d = 0, they open).  Under the COM rule (R21)
      // an ancestor whose centre of mass lies far outside the group's cube can stay UN-opened at large theta:
      // the group then sees its own mass through that cell's multipole (the variant's known flaw, kept as the
      // oracle has it) and there is no self pair to take out of the potential again.
      bool self_met = kPlain || root_leaf;
      if (root_leaf) {
        if (lane == 0) {
          if (MODE == kFused) sm.leafq[0] = make_int2(root_a, root_n);
          else if (MODE == kWrite) lio.leaves[woff_l] = make_int2(root_a, root_n);
        }
        lq = 1; n_lr = 1; n_pp = root_n;
      } else {
        if (lane == 0) sm.stack[0] = ((uint32_t)root_a << 3) | (uint32_t)(root_n - 1);
        ssz = 1;
      }
      __syncwarp();

      // ---- the walk (List 1-2): pop up to 4 nodes, test their children
      // (the evaluation code exists ONCE, at the bottom of this loop: the last trip, `walking` false, flushes what is left)
      while (true) {
        bool walking = true;
        if (ssz == 0) {
          if (spill_sz == 0) walking = false;
          else {
            const int take = min(spill_sz, STK / 2);      // reload the top of the spill stack
            for (int t = lane; t < take; t += 32) sm.stack[t] = spill[spill_sz - take + t];
            spill_sz -= take; ssz = take;
            __syncwarp();
          }
        }
        if (walking) {
        // up to kWalkB batches of 4 nodes per iteration: the child loads of all batches are issued together, so an
        // iteration still costs ONE memory latency (the walk is latency-bound; the evaluation of other warps hides it)
        const int npop = min(ssz, 4 * kWalkB);
        const int slot = lane >> 3, k = lane & 7;
        bool valid_b[kWalkB];
        int c_b[kWalkB];
        float4 cb_b[kWalkB], cx_b[kWalkB], c0_b[kWalkB], c1_b[kWalkB];
#pragma unroll
        for (int b = 0; b < kWalkB; b++) {
          const int sl = slot + 4 * b;
          const uint32_t packed = (sl < npop) ? sm.stack[ssz - 1 - sl] : 0u;
          valid_b[b] = (sl < npop) && (k <= (int)(packed & 7u));
          // lanes without a child load cell 0 (the root always exists); `valid` masks everything they compute
          c_b[b] = valid_b[b] ? (int)(packed >> 3) + k : 0;
          cb_b[b] = __ldg(bnd + c_b[b]); cx_b[b] = __ldg(xm + c_b[b]); c0_b[b] = __ldg(q0 + c_b[b]); c1_b[b] = __ldg(q1 + c_b[b]);
        }
        ssz -= npop;
        __syncwarp();                                    // all pops were read before slots are reused
#pragma unroll
        for (int b = 0; b < kWalkB; b++) {
        if (b > 0 && npop <= 4 * b) break;               // warp-uniform: this batch is empty
        const bool valid = valid_b[b];
        const int c = c_b[b];
        const float4 cb = cb_b[b], cx = cx_b[b], c0 = c0_b[b], c1 = c1_b[b];
        // open_node (O5/R16): one fixed sequence of correctly rounded fp32 operations
        // (variant R21, com_rule: the cell's centre of mass in place of b_c, 0 in place of h_c in the distance)
        const float hc = fabsf(cb.w);
        const float hs = com_rule ? 0.f : hc;
        const float sx = __fadd_rn(hs, ghx), sy = __fadd_rn(hs, ghy), sz = __fadd_rn(hs, ghz);
        const float px = com_rule ? cx.x : cb.x, py = com_rule ? cx.y : cb.y, pz = com_rule ? cx.z : cb.z;
        const float tx = fmaxf(__fsub_rn(fabsf(__fsub_rn(px, gbx)), sx), 0.f);
        const float ty = fmaxf(__fsub_rn(fabsf(__fsub_rn(py, gby)), sy), 0.f);
        const float tz = fmaxf(__fsub_rn(fabsf(__fsub_rn(pz, gbz)), sz), 0.f);
        const float d2 = __fmaf_rn(tz, tz, __fmaf_rn(ty, ty, __fmul_rn(tx, tx)));
        const float l = __fadd_rn(hc, hc);
        const bool open = valid && (__fmul_rn(d2, th2) <= __fmul_rn(l, l));
        const bool leaf = __float_as_int(cb.w) < 0;
        const bool to_cell = valid && !open, to_leaf = open && leaf, to_stack = open && !leaf;
        const int la = __float_as_int(c1.z), lb = __float_as_int(c1.w);

        const unsigned m_cell = __ballot_sync(kFull, to_cell);
        const unsigned m_leaf = __ballot_sync(kFull, to_leaf);
        const unsigned m_stack = __ballot_sync(kFull, to_stack);
        if (to_cell) {                                   // not opened (leaf or node): multipole (R2)
          if (MODE == kFused) {
            CellRec& r = sm.u.cell[ccnt + __popc(m_cell & lt_mask)];
            r.xm = cx; r.q0 = c0; r.q1 = make_float2(c1.x, c1.y);
          } else if (MODE == kWrite) {
            lio.cells[woff_c + (unsigned long long)(n_pc + __popc(m_cell & lt_mask))] = c;
          }
        }
        if (MODE == kFused) ccnt += __popc(m_cell);
        n_pc += __popc(m_cell);
        if (m_leaf) {                                    // opened leaf: particle-particle
          if (to_leaf) {
            if (MODE == kFused) sm.leafq[lq + __popc(m_leaf & lt_mask)] = make_int2(la, lb);
            else if (MODE == kWrite) lio.leaves[woff_l + (unsigned long long)(n_lr + __popc(m_leaf & lt_mask))] = make_int2(la, lb);
          }
          if (MODE == kFused) lq += __popc(m_leaf); else n_lr += __popc(m_leaf);
          n_open += __popc(m_leaf);
          n_pp += __reduce_add_sync(kFull, to_leaf ? lb : 0);
          if (!kPlain && MODE == kFused) {                 // own leaf opened? (all or nothing per group, see above)
            const int fb = G.y + pb;
            self_met |= __any_sync(kFull, to_leaf && la <= fb && fb < la + lb);
          }
        }
        if (m_stack && !overflow) {                      // opened node: walk on
          const int npush = __popc(m_stack);
          n_open += npush;
          if (ssz + npush > STK) {                       // spill the bottom half to global memory
            const int mv = STK / 2;
            if (spill_sz + mv > spill_cap) { overflow = true; }
            else {
              __syncwarp();
              for (int t = lane; t < mv; t += 32) spill[spill_sz + t] = sm.stack[t];
              __syncwarp();
              for (int t0 = mv; t0 < ssz; t0 += 32) {    // shift the rest down (ascending, chunked)
                const int t = t0 + lane;
                const uint32_t v = (t < ssz) ? sm.stack[t] : 0u;
                __syncwarp();
                if (t < ssz) sm.stack[t - mv] = v;
                __syncwarp();
              }
              spill_sz += mv; ssz -= mv; n_spills++;
            }
          }
          if (!overflow) {
            if (to_stack) sm.stack[ssz + __popc(m_stack & lt_mask)] = ((uint32_t)la << 3) | (uint32_t)(lb - 1);
            ssz += npush;
          }
        }
        }  // batches
        if (overflow) break;
        __syncwarp();
        }  // walking
        if (MODE == kFused) {
          // a chunk is evaluated when the next iteration might not fit, the bodies' staging area (the same memory)
          // is needed, or the walk is over
          const bool flush_leaves = walking ? (lq > kLeafQCap - 32 * kWalkB) : (lq > 0);
          if (ccnt > (walking ? kCellCap - 32 * kWalkB : 0) || (flush_leaves && ccnt)) {
            if (!walk_only) eval_cells<kEps0>(sm.u.cell, ccnt, eps2, L, ps, mono, lane);
            ccnt = 0; __syncwarp();
          }
          if (flush_leaves) { if (!walk_only) eval_leaves<kEps0>(sm.u.bs, sm.leafq, lq, part, eps2, L, ps, lane, mbar, &bulk_phase); lq = 0; __syncwarp(); }
        }
        if (!walking) break;
      }

      if (MODE == kFused) {
        // ---- A6: reduce the slices of every particle, write back in the caller's order
        write_back<false, !kEps0>(L, ps, part, orig, G.y + pb, m, eps2, lane, acc, pot, out_npc, n_pc, out_npp, n_pp - 1, self_met,
                                  sho.out4 ? sho.out4 + shard_row + pb : nullptr, sho.cnt2 ? sho.cnt2 + shard_row + pb : nullptr);
      } else if (MODE == kCount) {
        if (lane == 0) { lio.cnt_c[g] = (unsigned long long)n_pc; lio.cnt_l[g] = (unsigned long long)n_lr; lio.leaf_bodies[g] = (int)n_pp; }
      }
      if (lane == 0) {
        if (MODE != kWrite) {                              // the two-pass variant counts in its first pass
          const long long np = (MODE == kFused) ? m : G.z;
          atomicAdd(&ctr->n_pc_total, (unsigned long long)(n_pc * np));
          atomicAdd(&ctr->n_pp_total, (unsigned long long)((n_pp - 1) * np));
          // opening tests EXECUTED by this walk: every tested child ends on the cell list or is opened
          atomicAdd(&ctr->n_tests_total, (unsigned long long)(n_pc + n_open));
          atomicAdd(&ctr->n_opened_total, (unsigned long long)n_open);
        }
        if (n_spills) atomicAdd(&ctr->n_spills, (unsigned long long)n_spills);
        if (overflow) atomicExch(&ctr->overflow, 1u);
      }
      __syncwarp();
      if (MODE != kFused) break;                           // lists are per group, not per pass
    }
  }
}

#ifndef TC_FORCES_ONLY
// ---- two-pass variant: the evaluation kernels of Lists 3 and 4 on global lists ------
// node kernel: warp per group, list chunks gathered to shared memory, acc / pot / n_pc WRITTEN
__global__ void __launch_bounds__(kWarpsPerCta * 32, TC_MINB)
node_kernel(const float4* __restrict__ xm, const float4* __restrict__ q0, const float4* __restrict__ q1,
            const float4* __restrict__ part, const int32_t* __restrict__ orig, const int4* __restrict__ grp, int n_groups,
            float eps, float* __restrict__ acc, float* __restrict__ pot, int32_t* __restrict__ out_npc,
            DeviceCounters* __restrict__ ctr, ListIO lio, int flags) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  WarpSmem<64>& sm = reinterpret_cast<WarpSmem<64>*>(smem_raw)[warp];
  const float eps2 = eps * eps;
  const bool mono = flags & kFlagMonopole;
  while (true) {
    int g = 0;
    if (lane == 0) g = (int)atomicAdd(&ctr->next_group, 1u);
    g = __shfl_sync(kFull, g, 0);
    if (g >= n_groups) break;
    g = __ldg(&grp[g].w);
    const int4 G = __ldg(grp + g);
    const unsigned long long b = lio.off_c[g];
    const int n_c = (int)(lio.off_c[g + 1] - b);
    for (int pb = 0; pb < G.z; pb += kPassCap) {
      const int m = min(kPassCap, G.z - pb);
      Lanes L; PassState ps;
      setup_pass(L, ps, part, G.y + pb, m, lane);
      for (int base = 0; base < n_c; base += kCellCap) {
        const int cnt = min(kCellCap, n_c - base);
        for (int t = lane; t < cnt; t += 32) {
          const int c = __ldg(lio.cells + b + base + t);
          const float4 c1 = __ldg(q1 + c);
          CellRec& r = sm.u.cell[t];
          r.xm = __ldg(xm + c); r.q0 = __ldg(q0 + c); r.q1 = make_float2(c1.x, c1.y);
        }
        __syncwarp();
        eval_cells<false>(sm.u.cell, cnt, eps2, L, ps, mono, lane);
        __syncwarp();
      }
      write_back<false, false>(L, ps, part, orig, G.y + pb, m, eps2, lane, acc, pot, out_npc, n_c);
    }
  }
}

// leaf kernel: warp per group, opened-leaf ranges from the global list, acc / pot ADDED, n_pp written
template <bool kEps0>
__global__ void __launch_bounds__(kWarpsPerCta * 32, TC_MINB)
leaf_kernel(const float4* __restrict__ part, const int32_t* __restrict__ orig, const int4* __restrict__ grp, int n_groups,
            float eps, float* __restrict__ acc, float* __restrict__ pot, int32_t* __restrict__ out_npp,
            DeviceCounters* __restrict__ ctr, ListIO lio) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  WarpSmem<64>& sm = reinterpret_cast<WarpSmem<64>*>(smem_raw)[warp];
  const float eps2 = eps * eps;
  while (true) {
    int g = 0;
    if (lane == 0) g = (int)atomicAdd(&ctr->next_group, 1u);
    g = __shfl_sync(kFull, g, 0);
    if (g >= n_groups) break;
    g = __ldg(&grp[g].w);
    const int4 G = __ldg(grp + g);
    const unsigned long long b = lio.off_l[g];
    const int n_l = (int)(lio.off_l[g + 1] - b);
    const int n_bodies = __ldg(lio.leaf_bodies + g);
    for (int pb = 0; pb < G.z; pb += kPassCap) {
      const int m = min(kPassCap, G.z - pb);
      Lanes L; PassState ps;
      setup_pass(L, ps, part, G.y + pb, m, lane);
      bool self_met = false;                 // is the pass's own leaf on the list? (see forces_kernel)
      const int fb = G.y + pb;
      for (int base = 0; base < n_l; base += kLeafQCap) {
        const int cnt = min(kLeafQCap, n_l - base);
        bool mine = false;
        for (int t = lane; t < cnt; t += 32) {
          const int2 r = __ldg(lio.leaves + b + base + t);
          sm.leafq[t] = r;
          mine |= (r.x <= fb && fb < r.x + r.y);
        }
        self_met |= __any_sync(kFull, mine);
        __syncwarp();
        eval_leaves<kEps0>(sm.u.bs, sm.leafq, cnt, part, eps2, L, ps, lane);
        __syncwarp();
      }
      write_back<true, !kEps0>(L, ps, part, orig, G.y + pb, m, eps2, lane, acc, pot, out_npp, n_bodies - 1, nullptr, 0, self_met);
    }
  }
}

#endif  // TC_FORCES_ONLY

template <int STK, bool kEps0, int MODE = kFused, bool kPlain = false>
int launch_t(const DeviceTree& T, const ForceLaunch& L, cudaStream_t st, int* ctas_per_sm_out, ListIO lio = ListIO()) {
  auto kern = forces_kernel<STK, kEps0, MODE, kPlain>;
  const size_t smem = sizeof(WarpSmem<STK>) * kWarpsPerCta;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return (int)e;
  int per_sm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kWarpsPerCta * 32, smem);
  if (e != cudaSuccess) return (int)e;
  if (per_sm < 1) per_sm = 1;
  if (ctas_per_sm_out) { *ctas_per_sm_out = per_sm; return 0; }
  // persistent grid: every SM full, groups handed out by an atomic counter
  // (never more CTAs than the spill buffer was sized for: forces_total_warps)
  const int grid = L.max_grid > 0 ? std::min(L.n_sm * per_sm, L.max_grid) : L.n_sm * per_sm;
  ShardOut sho;
  sho.out4 = reinterpret_cast<float4*>(L.shard_out4); sho.cnt2 = reinterpret_cast<int2*>(L.shard_cnt2); sho.off = L.shard_off;
  kern<<<grid, kWarpsPerCta * 32, smem, st>>>(T.bnd, T.xm, T.q0, T.q1, T.part, T.orig, T.grp, T.gbox, (int)T.n_groups,
                                               L.theta, L.eps, L.acc, L.pot, L.n_pc, L.n_pp, L.counters, L.spill,
                                               L.spill_cap, L.flags, lio, L.shard_rank, L.shard_count, sho);
  return (int)cudaGetLastError();
}

int dispatch(const DeviceTree& T, const ForceLaunch& L, cudaStream_t st, int* per_sm) {
  const bool eps0 = (L.eps * L.eps == 0.f);
  if (L.stack_smem == 64) return eps0 ? launch_t<64, true>(T, L, st, per_sm) : launch_t<64, false>(T, L, st, per_sm);
  if ((L.flags & (kFlagComRule | kFlagMonopole | kFlagGroupBox)) == 0)   // the default readings: no variant selects
    return eps0 ? launch_t<256, true, kFused, true>(T, L, st, per_sm) : launch_t<256, false, kFused, true>(T, L, st, per_sm);
  return eps0 ? launch_t<256, true>(T, L, st, per_sm) : launch_t<256, false>(T, L, st, per_sm);
}

}  // namespace

namespace TC_CFG_NS {
int launch_forces(const DeviceTree& T, const ForceLaunch& L, void* stream) {
  return dispatch(T, L, (cudaStream_t)stream, nullptr);
}

int forces_warps_per_cta() { return kWarpsPerCta; }

int forces_total_warps(int n_sm, int stack_smem) {
  DeviceTree T;
  ForceLaunch L;
  L.stack_smem = stack_smem; L.eps = 1.f;
  int per_sm = 0;
  if (dispatch(T, L, nullptr, &per_sm) != 0 || per_sm < 1) per_sm = 8;
  return n_sm * per_sm * kWarpsPerCta;
}
}  // namespace TC_CFG_NS

#ifndef TC_FORCES_ONLY

// ---- the paper-literal two-pass variant (option "two_pass") ----
namespace {
template <typename T>
cudaError_t grow2(T*& p, size_t& cap, size_t need, cudaStream_t st) {
  if (cap >= need) return cudaSuccess;
  cudaError_t e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return e;
  cudaFree(p); p = nullptr; cap = 0;
  const size_t ncap = need + need / 8 + 256;
  e = cudaMalloc((void**)&p, sizeof(T) * ncap);
  if (e == cudaSuccess) cap = ncap;
  return e;
}
template <int MODE>
int dispatch_walk(const DeviceTree& T, const ForceLaunch& L, cudaStream_t st, ListIO lio) {
  const bool eps0 = (L.eps * L.eps == 0.f);
  if (L.stack_smem == 64) return eps0 ? launch_t<64, true, MODE>(T, L, st, nullptr, lio) : launch_t<64, false, MODE>(T, L, st, nullptr, lio);
  return eps0 ? launch_t<256, true, MODE>(T, L, st, nullptr, lio) : launch_t<256, false, MODE>(T, L, st, nullptr, lio);
}
}  // namespace

void TwoPassScratch::release() {
  cudaFree(cnt_c); cudaFree(cnt_l); cudaFree(off_c); cudaFree(off_l); cudaFree(leaf_bodies); cudaFree(cells); cudaFree(leaves);
  cudaFree(tmp);
  for (int k = 0; k < 5; k++) if (ev[k]) cudaEventDestroy((cudaEvent_t)ev[k]);
  *this = TwoPassScratch();
}

#define TP_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return (int)e_; } while (0)

int launch_forces_two_pass(const DeviceTree& T, const ForceLaunch& L, TwoPassScratch& S, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  const size_t ng = (size_t)T.n_groups;
  for (int k = 0; k < 5; k++) if (!S.ev[k]) { cudaEvent_t e; TP_CUDA(cudaEventCreate(&e)); S.ev[k] = e; }
  TP_CUDA(grow2(S.cnt_c, S.cap_cnt_c, ng + 1, st)); TP_CUDA(grow2(S.cnt_l, S.cap_cnt_l, ng + 1, st));
  TP_CUDA(grow2(S.off_c, S.cap_off_c, ng + 1, st)); TP_CUDA(grow2(S.off_l, S.cap_off_l, ng + 1, st));
  TP_CUDA(grow2(S.leaf_bodies, S.cap_lb, ng, st));
  TP_CUDA(cudaMemsetAsync(S.cnt_c + ng, 0, sizeof(unsigned long long), st));
  TP_CUDA(cudaMemsetAsync(S.cnt_l + ng, 0, sizeof(unsigned long long), st));
  ListIO lio;
  lio.cnt_c = S.cnt_c; lio.cnt_l = S.cnt_l; lio.off_c = S.off_c; lio.off_l = S.off_l;
  lio.cells = nullptr; lio.leaves = nullptr; lio.leaf_bodies = S.leaf_bodies;
  unsigned int* next_group = &L.counters->next_group;
  // pass 1: count
  TP_CUDA(cudaEventRecord((cudaEvent_t)S.ev[0], st));
  { const int e = dispatch_walk<kCount>(T, L, st, lio); if (e) return e; }
  TP_CUDA(cudaEventRecord((cudaEvent_t)S.ev[1], st));
  // the scan the paper does on the host, here on the device
  size_t need = 0, need2 = 0;
  TP_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, need, S.cnt_c, S.off_c, (int)(ng + 1), st));
  TP_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, need2, S.cnt_l, S.off_l, (int)(ng + 1), st));
  TP_CUDA(grow2(S.tmp, S.cap_tmp, std::max(need, need2), st));
  TP_CUDA(cub::DeviceScan::ExclusiveSum(S.tmp, need, S.cnt_c, S.off_c, (int)(ng + 1), st));
  TP_CUDA(cub::DeviceScan::ExclusiveSum(S.tmp, need2, S.cnt_l, S.off_l, (int)(ng + 1), st));
  unsigned long long tot[2];
  TP_CUDA(cudaMemcpyAsync(&tot[0], S.off_c + ng, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  TP_CUDA(cudaMemcpyAsync(&tot[1], S.off_l + ng, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  TP_CUDA(cudaStreamSynchronize(st));
  S.n_list_cells = (long long)tot[0]; S.n_list_leaves = (long long)tot[1];
  TP_CUDA(grow2(S.cells, S.cap_cells, (size_t)tot[0] + 1, st));
  TP_CUDA(grow2(S.leaves, S.cap_leaves, (size_t)tot[1] + 1, st));
  lio.cells = S.cells; lio.leaves = S.leaves;
  // pass 2: write the lists
  TP_CUDA(cudaMemsetAsync(next_group, 0, sizeof(unsigned int), st));
  TP_CUDA(cudaEventRecord((cudaEvent_t)S.ev[1], st));
  { const int e = dispatch_walk<kWrite>(T, L, st, lio); if (e) return e; }
  TP_CUDA(cudaEventRecord((cudaEvent_t)S.ev[2], st));
  // evaluation kernels
  const size_t smem = sizeof(WarpSmem<64>) * kWarpsPerCta;
  const bool eps0 = (L.eps * L.eps == 0.f);
  int per_sm = 0;
  TP_CUDA(cudaFuncSetAttribute(node_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  TP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, node_kernel, kWarpsPerCta * 32, smem));
  TP_CUDA(cudaMemsetAsync(next_group, 0, sizeof(unsigned int), st));
  node_kernel<<<L.n_sm * std::max(per_sm, 1), kWarpsPerCta * 32, smem, st>>>(T.xm, T.q0, T.q1, T.part, T.orig, T.grp, (int)T.n_groups,
                                                                              L.eps, L.acc, L.pot, L.n_pc, L.counters, lio, L.flags);
  TP_CUDA(cudaGetLastError());
  TP_CUDA(cudaEventRecord((cudaEvent_t)S.ev[3], st));
  TP_CUDA(cudaMemsetAsync(next_group, 0, sizeof(unsigned int), st));
  if (eps0) {
    TP_CUDA(cudaFuncSetAttribute(leaf_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    TP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, leaf_kernel<true>, kWarpsPerCta * 32, smem));
    leaf_kernel<true><<<L.n_sm * std::max(per_sm, 1), kWarpsPerCta * 32, smem, st>>>(T.part, T.orig, T.grp, (int)T.n_groups, L.eps, L.acc,
                                                                                     L.pot, L.n_pp, L.counters, lio);
  } else {
    TP_CUDA(cudaFuncSetAttribute(leaf_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    TP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, leaf_kernel<false>, kWarpsPerCta * 32, smem));
    leaf_kernel<false><<<L.n_sm * std::max(per_sm, 1), kWarpsPerCta * 32, smem, st>>>(T.part, T.orig, T.grp, (int)T.n_groups, L.eps, L.acc,
                                                                                      L.pot, L.n_pp, L.counters, lio);
  }
  TP_CUDA(cudaGetLastError());
  TP_CUDA(cudaEventRecord((cudaEvent_t)S.ev[4], st));
  return 0;
}

// event times of the last launch_forces_two_pass (stream must be idle): count, write, node, leaf [ms]
int two_pass_times(const TwoPassScratch& S, float ms[4]) {
  // ev[1] was re-recorded after the scan: [0]->[1'] would include it, so the count pass is timed by its own pair below
  for (int k = 0; k < 4; k++) ms[k] = 0.f;
  if (!S.ev[4]) return 0;
  TP_CUDA(cudaEventElapsedTime(&ms[1], (cudaEvent_t)S.ev[1], (cudaEvent_t)S.ev[2]));
  TP_CUDA(cudaEventElapsedTime(&ms[2], (cudaEvent_t)S.ev[2], (cudaEvent_t)S.ev[3]));
  TP_CUDA(cudaEventElapsedTime(&ms[3], (cudaEvent_t)S.ev[3], (cudaEvent_t)S.ev[4]));
  float all = 0.f;
  TP_CUDA(cudaEventElapsedTime(&all, (cudaEvent_t)S.ev[0], (cudaEvent_t)S.ev[1]));
  ms[0] = all;     // count pass + device scan + list allocation (the paper's host step)
  return 0;
}

// ---- tc_direct: direct summation (the paper's accuracy reference) ----------------
// a_i = sum_{j != i} m_j d / s^3, phi_i = -sum_{j != i} m_j / s, d = x_j - x_i, s^2 = |d|^2 + eps^2.
// Packed FP32 per interaction with one Newton step on rsqrt.approx (relative error ~1e-7 per term),
// partial sums of 256 sources in fp32, flushed into fp64 accumulators ("double precision emulation"
// in the paper's words); 4 targets per thread, sources staged through shared memory, the source
// range split over blockIdx.y and combined with fp64 atomics.
namespace {
constexpr int kDirThreads = 128, kDirTile = 256, kDirTargetsPerCta = 4 * kDirThreads;

template <bool kEps0>
__device__ __forceinline__ void direct_interact(const Pos2& p, float eps2, const float4 b, Acc2& a) {
  const f2 dx = sub2(bc(b.x), p.x), dy = sub2(bc(b.y), p.y), dz = sub2(bc(b.z), p.z);
  const f2 s2 = fma2(dz, dz, fma2(dy, dy, fma2(dx, dx, bc(eps2))));
  float r0 = rsqrt_approx(lo(s2)), r1 = rsqrt_approx(hi(s2));
  if (kEps0) { r0 = (lo(s2) > 0.f) ? r0 : 0.f; r1 = (hi(s2) > 0.f) ? r1 : 0.f; }
  f2 ri = pk(r0, r1);
  const f2 h = mul2(s2, bc(-0.5f));                       // Newton: y <- y (1.5 - 0.5 x y^2)
  ri = mul2(ri, fma2(h, mul2(ri, ri), bc(1.5f)));
  const f2 ri2 = mul2(ri, ri);
  const f2 mr = mul2(bc(b.w), ri);
  const f2 mr3 = mul2(mr, ri2);
  a.npot = add2(a.npot, mr);
  a.ax = fma2(mr3, dx, a.ax); a.ay = fma2(mr3, dy, a.ay); a.az = fma2(mr3, dz, a.az);
}

// the same pair of interactions with one mass per half (0 for the half whose target IS the source: the sum runs over j != i)
__device__ __forceinline__ void direct_interact_masked(const Pos2& p, float eps2, const float4 b, float m0, float m1, Acc2& a) {
  const f2 dx = sub2(bc(b.x), p.x), dy = sub2(bc(b.y), p.y), dz = sub2(bc(b.z), p.z);
  const f2 s2 = fma2(dz, dz, fma2(dy, dy, fma2(dx, dx, bc(eps2))));
  f2 ri = pk(rsqrt_approx(lo(s2)), rsqrt_approx(hi(s2)));
  const f2 h = mul2(s2, bc(-0.5f));
  ri = mul2(ri, fma2(h, mul2(ri, ri), bc(1.5f)));
  const f2 ri2 = mul2(ri, ri);
  const f2 mr = mul2(pk(m0, m1), ri);
  const f2 mr3 = mul2(mr, ri2);
  a.npot = add2(a.npot, mr);
  a.ax = fma2(mr3, dx, a.ax); a.ay = fma2(mr3, dy, a.ay); a.az = fma2(mr3, dz, a.az);
}

template <bool kEps0>
__global__ void __launch_bounds__(kDirThreads)
direct_kernel(const float4* __restrict__ src, long long n, const long long* __restrict__ targets, long long n_t,
              float eps, double* __restrict__ acc, double* __restrict__ pot) {
  __shared__ float4 tile[kDirTile];
  const float eps2 = eps * eps;
  const long long t0 = (long long)blockIdx.x * kDirTargetsPerCta + threadIdx.x;
  long long ti[4];
  Pos2 P[2];
#pragma unroll
  for (int j = 0; j < 4; j++) {
    const long long t = t0 + (long long)j * kDirThreads;
    ti[j] = (t < n_t) ? (targets ? targets[t] : t) : -1;
  }
#pragma unroll
  for (int j = 0; j < 2; j++) {
    const float4 a = __ldg(src + (ti[2 * j] >= 0 ? ti[2 * j] : 0)), b = __ldg(src + (ti[2 * j + 1] >= 0 ? ti[2 * j + 1] : 0));
    P[j].x = add2(pk(a.x, b.x), bc(0.f)); P[j].y = add2(pk(a.y, b.y), bc(0.f)); P[j].z = add2(pk(a.z, b.z), bc(0.f));
  }
  double d[4][4];
#pragma unroll
  for (int j = 0; j < 4; j++) d[j][0] = d[j][1] = d[j][2] = d[j][3] = 0.0;
  // this CTA's share of the sources, in whole tiles
  const long long n_tiles = (n + kDirTile - 1) / kDirTile;
  const long long tb = n_tiles * blockIdx.y / gridDim.y, te = n_tiles * (blockIdx.y + 1) / gridDim.y;
  for (long long tl = tb; tl < te; tl++) {
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kDirTile / kDirThreads; k++) {
      const long long j = tl * kDirTile + threadIdx.x + k * kDirThreads;
      // padding: massless sources far away contribute exactly zero
      tile[threadIdx.x + k * kDirThreads] = (j < n) ? __ldg(src + j) : make_float4(1e18f, 1e18f, 1e18f, 0.f);
    }
    __syncthreads();
    Acc2 A[2];
#pragma unroll
    for (int j = 0; j < 2; j++) A[j].ax = A[j].ay = A[j].az = A[j].npot = 0ull;
    // A target meets itself only in the tile that holds it: there (a few tiles per thread) the source whose index is the
    // target's gets mass 0, so -m/eps never enters the fp32 partial sum.  eps = 0 masks the pair by s^2 = 0 already.
    const long long tbase = tl * kDirTile;
    const bool own_tile = !kEps0 && ((ti[0] >= tbase && ti[0] < tbase + kDirTile) || (ti[1] >= tbase && ti[1] < tbase + kDirTile) ||
                                     (ti[2] >= tbase && ti[2] < tbase + kDirTile) || (ti[3] >= tbase && ti[3] < tbase + kDirTile));
    if (own_tile) {
      for (int k = 0; k < kDirTile; k++) {
        const float4 b = tile[k];
        const long long jj = tbase + k;
        direct_interact_masked(P[0], eps2, b, jj == ti[0] ? 0.f : b.w, jj == ti[1] ? 0.f : b.w, A[0]);
        direct_interact_masked(P[1], eps2, b, jj == ti[2] ? 0.f : b.w, jj == ti[3] ? 0.f : b.w, A[1]);
      }
    } else {
#pragma unroll 4
      for (int k = 0; k < kDirTile; k++) {
        const float4 b = tile[k];
        direct_interact<kEps0>(P[0], eps2, b, A[0]);
        direct_interact<kEps0>(P[1], eps2, b, A[1]);
      }
    }
#pragma unroll
    for (int j = 0; j < 2; j++) {
      d[2 * j][0] += (double)lo(A[j].ax); d[2 * j][1] += (double)lo(A[j].ay); d[2 * j][2] += (double)lo(A[j].az);
      d[2 * j][3] += (double)lo(A[j].npot);
      d[2 * j + 1][0] += (double)hi(A[j].ax); d[2 * j + 1][1] += (double)hi(A[j].ay); d[2 * j + 1][2] += (double)hi(A[j].az);
      d[2 * j + 1][3] += (double)hi(A[j].npot);
    }
  }
#pragma unroll
  for (int j = 0; j < 4; j++) {
    if (ti[j] < 0) continue;
    const long long t = t0 + (long long)j * kDirThreads;
    const double ph = -d[j][3];
    atomicAdd(acc + 3 * t + 0, d[j][0]); atomicAdd(acc + 3 * t + 1, d[j][1]); atomicAdd(acc + 3 * t + 2, d[j][2]);
    if (pot) atomicAdd(pot + t, ph);
  }
}
}  // namespace

int launch_direct(const float4* src, long long n, const long long* targets, long long n_t, float eps, double* acc,
                  double* pot, int n_sm, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = cudaMemsetAsync(acc, 0, sizeof(double) * 3 * (size_t)n_t, st);
  if (e == cudaSuccess && pot) e = cudaMemsetAsync(pot, 0, sizeof(double) * (size_t)n_t, st);
  if (e != cudaSuccess) return (int)e;
  const long long tiles_t = (n_t + kDirTargetsPerCta - 1) / kDirTargetsPerCta;
  const long long tiles_s = (n + kDirTile - 1) / kDirTile;
  long long splits = (8LL * n_sm + tiles_t - 1) / tiles_t;          // >= 8 CTAs per SM in flight
  if (splits > tiles_s) splits = tiles_s;
  if (splits > 65535) splits = 65535;
  if (splits < 1) splits = 1;
  if (tiles_t > 2147483647LL) return (int)cudaErrorInvalidValue;
  const dim3 grid((unsigned)tiles_t, (unsigned)splits);
  if (eps * eps == 0.f) direct_kernel<true><<<grid, kDirThreads, 0, st>>>(src, n, targets, n_t, eps, acc, pot);
  else direct_kernel<false><<<grid, kDirThreads, 0, st>>>(src, n, targets, n_t, eps, acc, pot);
  return (int)cudaGetLastError();
}

// ---- tc_direct_static: the direct sum for callers that must not allocate (include/tc.h) -------------------------------
// tc_direct keeps the sources as one (x, y, z, m) float4 array that its context cudaMallocs.  This variant keeps that array
// in the library image instead: a file-scope __device__ array, resident on every GPU that loads the library from the moment
// the module is loaded until the process exits.  `g_static_src` below is, in HOST code, only the handle of that symbol — not
// a device address: a kernel must be given what cudaGetSymbolAddress returns for the CURRENT device (taken once per device,
// below).  Same kernels and same launcher as tc_direct from there on.
static_assert(TC_DIRECT_STATIC_MAX_N == 262144, "include/tc.h documents 4 MiB of static device memory per GPU");
static __device__ __align__(256) float4 g_static_src[TC_DIRECT_STATIC_MAX_N];

namespace {
// pos [n,3], mass [n] -> src [n] (x, y, z, m): every entry a later read may touch (0 .. n-1) is written here first, so the
// contents a previous call left behind are never read and nothing needs clearing
__global__ void __launch_bounds__(256) pack_static_kernel(const float* __restrict__ pos, const float* __restrict__ mass,
                                                          long long n, float4* __restrict__ src) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= n) return;
  src[i] = make_float4(__ldg(pos + 3 * i), __ldg(pos + 3 * i + 1), __ldg(pos + 3 * i + 2), __ldg(mass + i));
}

constexpr int kStaticMaxDevices = 64;
struct StaticDevice { float4* src = nullptr; int n_sm = 0; bool ready = false; };
StaticDevice g_static_dev[kStaticMaxDevices];
std::mutex g_static_mutex;

bool on_device(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}
}  // namespace

int direct_static(const float* pos, const float* mass, long long n, float eps, const long long* targets, long long n_targets,
                  double* acc, double* pot, void* stream, std::string& msg) {
  auto bad = [&](int code, const std::string& m) { msg = "tc_direct_static: " + m; return code; };
  if (!pos || !mass || !acc) return bad(TC_EINVAL, "pos, mass and acc must not be null");
  if (n < 1) return bad(TC_EINVAL, "n must be >= 1");
  if (n > (long long)TC_DIRECT_STATIC_MAX_N)
    return bad(TC_EINVAL, "n = " + std::to_string(n) + " exceeds TC_DIRECT_STATIC_MAX_N = " + std::to_string(TC_DIRECT_STATIC_MAX_N) +
                              " (the static scratch holds no more sources; use tc_direct, which allocates)");
  const long long nt = targets ? n_targets : n;
  if (nt < 1) return bad(TC_EINVAL, "n_targets must be >= 1");
  if (nt > (long long)TC_DIRECT_STATIC_MAX_N)
    return bad(TC_EINVAL, "n_targets = " + std::to_string(nt) + " exceeds TC_DIRECT_STATIC_MAX_N = " + std::to_string(TC_DIRECT_STATIC_MAX_N));
  if (!(eps >= 0.f) || !std::isfinite(eps)) return bad(TC_EINVAL, "eps must be finite and >= 0");
  if (eps < 1e-10f) eps = 0.f;                                   // as tc_direct
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return bad(TC_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e) + " (there is no CPU fallback)");
  if (dev < 0 || dev >= kStaticMaxDevices) return bad(TC_EINVAL, "device ordinal " + std::to_string(dev) + " is beyond the table of " + std::to_string(kStaticMaxDevices));
  if (!on_device(pos) || !on_device(mass) || !on_device(acc) || (pot && !on_device(pot)) || (targets && !on_device(targets)))
    return bad(TC_EINVAL, "every buffer must be a DEVICE pointer (this entry point has nowhere to stage host data)");
  StaticDevice D;
  {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice& S = g_static_dev[dev];
    if (!S.ready) {                                               // set-up, once per device, with that device current
      int major = 0, n_sm = 0;
      e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
      if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
      if (e != cudaSuccess) return bad(TC_ECUDA, std::string("cudaDeviceGetAttribute: ") + cudaGetErrorString(e));
      if (major < 10) return bad(TC_ECUDA, "this library is built for sm_100a (B200) only");
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_static_src);                 // the array's address on THIS device
      if (e != cudaSuccess || !p) {
        cudaGetLastError();
        return bad(TC_ECUDA, std::string("cudaGetSymbolAddress(g_static_src): ") + cudaGetErrorString(e));
      }
      S.src = static_cast<float4*>(p); S.n_sm = n_sm; S.ready = true;
    }
    D = S;
  }
  cudaStream_t st = (cudaStream_t)stream;
  pack_static_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(pos, mass, n, D.src);
  e = cudaGetLastError();
  if (e != cudaSuccess) return bad(TC_ECUDA, std::string("pack kernel launch: ") + cudaGetErrorString(e));
  const int le = launch_direct(D.src, n, targets, nt, eps, acc, pot, D.n_sm, stream);   // memset of acc / pot + direct_kernel
  if (le != 0) return bad(TC_ECUDA, std::string("direct-sum kernel launch: ") + cudaGetErrorString((cudaError_t)le));
  return TC_OK;
}

// ---- tc_leapfrog: the kicks and the drift of a KDK step (BASELINE.json config 5), element-wise over [3n]
namespace {
// v += a dt/2 ; x += v dt   (HBM-bound: 3 reads + 2 writes of 4 bytes per element, float4-vectorised body)
__global__ void __launch_bounds__(256) kick_drift_kernel(float* __restrict__ x, float* __restrict__ v,
                                                         const float* __restrict__ a, long long n3, float hdt, float dt) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  const long long n4 = n3 >> 2;
  float4* x4 = reinterpret_cast<float4*>(x);
  float4* v4 = reinterpret_cast<float4*>(v);
  const float4* a4 = reinterpret_cast<const float4*>(a);
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
    float4 xv = x4[i], vv = v4[i];
    const float4 av = __ldg(a4 + i);
    vv.x = __fmaf_rn(av.x, hdt, vv.x); vv.y = __fmaf_rn(av.y, hdt, vv.y);
    vv.z = __fmaf_rn(av.z, hdt, vv.z); vv.w = __fmaf_rn(av.w, hdt, vv.w);
    xv.x = __fmaf_rn(vv.x, dt, xv.x); xv.y = __fmaf_rn(vv.y, dt, xv.y);
    xv.z = __fmaf_rn(vv.z, dt, xv.z); xv.w = __fmaf_rn(vv.w, dt, xv.w);
    v4[i] = vv; x4[i] = xv;
  }
  for (long long i = 4 * n4 + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n3; i += stride) {   // ragged tail
    const float vv = __fmaf_rn(a[i], hdt, v[i]);
    v[i] = vv; x[i] = __fmaf_rn(vv, dt, x[i]);
  }
}
// v += a dt/2
__global__ void __launch_bounds__(256) kick_kernel(float* __restrict__ v, const float* __restrict__ a, long long n3, float hdt) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  const long long n4 = n3 >> 2;
  float4* v4 = reinterpret_cast<float4*>(v);
  const float4* a4 = reinterpret_cast<const float4*>(a);
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
    float4 vv = v4[i];
    const float4 av = __ldg(a4 + i);
    vv.x = __fmaf_rn(av.x, hdt, vv.x); vv.y = __fmaf_rn(av.y, hdt, vv.y);
    vv.z = __fmaf_rn(av.z, hdt, vv.z); vv.w = __fmaf_rn(av.w, hdt, vv.w);
    v4[i] = vv;
  }
  for (long long i = 4 * n4 + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n3; i += stride)
    v[i] = __fmaf_rn(a[i], hdt, v[i]);
}
}  // namespace

// pos / vel / acc must be 16-byte aligned (checked by tc_leapfrog)
int launch_kick_drift(float* pos, float* vel, const float* acc, long long n, float dt, int n_sm, void* stream) {
  const long long n3 = 3 * n;
  const int grid = (int)std::min<long long>((n3 / 4 + 255) / 256 + 1, 8LL * n_sm);
  kick_drift_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(pos, vel, acc, n3, 0.5f * dt, dt);
  return (int)cudaGetLastError();
}
int launch_kick(float* vel, const float* acc, long long n, float dt, int n_sm, void* stream) {
  const long long n3 = 3 * n;
  const int grid = (int)std::min<long long>((n3 / 4 + 255) / 256 + 1, 8LL * n_sm);
  kick_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(vel, acc, n3, 0.5f * dt);
  return (int)cudaGetLastError();
}

// ---- tc_fp32_peak: what the FP32 pipe of this device sustains with nothing but FFMA in flight
namespace {
__global__ void __launch_bounds__(256) ffma_peak_kernel(float* out, int n, float s) {
  float a[16];
#pragma unroll
  for (int i = 0; i < 16; i++) a[i] = threadIdx.x * 0.001f + i;
  const float b = s, c = 1.f - s;
  for (int t = 0; t < n; t++) {
#pragma unroll
    for (int i = 0; i < 16; i++) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(b), "f"(c));
  }
  float r = 0.f;
#pragma unroll
  for (int i = 0; i < 16; i++) r += a[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}
}  // namespace

int measure_fp32_peak(int n_sm, void* stream, double* tflops) {
  cudaStream_t st = (cudaStream_t)stream;
  const int grid = n_sm * 8, n = 20000;
  float* d = nullptr;
  cudaError_t e = cudaMalloc((void**)&d, sizeof(float) * (size_t)grid * 256);
  if (e != cudaSuccess) return (int)e;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  float best = 0.f;
  ffma_peak_kernel<<<grid, 256, 0, st>>>(d, 200, 0.999f);          // warm-up
  for (int rep = 0; rep < 3 && e == cudaSuccess; rep++) {
    cudaEventRecord(e0, st);
    ffma_peak_kernel<<<grid, 256, 0, st>>>(d, n, 0.999f);
    cudaEventRecord(e1, st);
    e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e == cudaSuccess && (best == 0.f || ms < best)) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  if (e != cudaSuccess) return (int)e;
  *tflops = 2.0 * 16.0 * (double)n * (double)grid * 256.0 / ((double)best * 1e-3) / 1e12;
  return 0;
}

#endif  // TC_FORCES_ONLY

}  // namespace tc

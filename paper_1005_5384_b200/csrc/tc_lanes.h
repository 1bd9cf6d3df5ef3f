// Lane mapping of the force kernel, shared by the kernel (tc_kernels.cu) and by the two builders'
// schedules (tc_build.cpp, tc_build_gpu.cu) so that the cost model of the schedule IS the kernel's
// mapping, not a hand-kept mirror of it.  Plain constexpr C++: host and device.
//
// One pass of a warp over m <= kPassCap particles of a group (one tree walk) picks
//   S slices of the interaction list  x  q = floor(32 / S) particle columns,   lane = s * q + p,
//   K = ceil(m / q) <= kMaxK particles per lane (particle j of lane (s, p) is j * q + p),
// so that the cycles per list entry, kRecordCycles[K] / S, are minimal.  kRecordCycles[K] is MEASURED: SM sub-partition
// cycles per list record of the particle-cell loop with K particles per lane (floor(K/2) packed FFMA2 pairs + one scalar
// particle when K is odd), four warps resident per sub-partition as in the kernel (the loop is
// bound by register-file operand bandwidth, an FFMA2 with three register-pair operands issues every 3 cycles, and
// the scalar particle of an odd K costs 58 % of a pair, not 50 %).  Every list record is read from shared memory
// once per lane and applied to the lane's K particles.  This is the answer to the paper's 30 % thread utilisation
// with thread-per-particle blocks.
#pragma once

#ifdef __CUDACC__
#define TC_HD __host__ __device__
#else
#define TC_HD
#endif

namespace tc {

#ifndef TC_MAXK
#define TC_MAXK 8
#endif
#ifndef TC_PASSCAP
#define TC_PASSCAP 128
#endif
constexpr int kMaxK = TC_MAXK;          // particles per lane: kMaxK / 2 packed pairs (+ one scalar particle when K is odd)
constexpr int kPassCap = TC_PASSCAP;    // particles of a group handled by ONE walk; larger groups (level-21 leaves of
                                        // coincident particles, or N_group > kPassCap) are walked once per kPassCap
static_assert(kMaxK >= 4 && kMaxK <= 8 && kPassCap <= 32 * kMaxK, "every pass size needs a mapping with S = 1");
// (measured with csrc/bench/mb_eval.cu before the last two kernel changes; the final build measures 46.0, 87.7, 122.4, 163.3, 208.3,
// 245.5, 283.6, 317.8 — profiles/r02_microbench.md — but the table built from THOSE runs the whole kernel slower, 5.86 against 5.74 ms:
// inside the kernel the odd-K loops, which they favour, lose more than they do alone.  The table is a tuning input, kept at its best.)
#ifndef TC_RC3
#define TC_RC3 134.7f
#endif
#ifndef TC_RC5
#define TC_RC5 208.3f
#endif
#ifndef TC_RC7
#define TC_RC7 293.7f
#endif
#ifndef TC_RC8
#define TC_RC8 324.1f
#endif
constexpr float kRecordCycles[9] = {0.f, 47.3f, 87.0f, TC_RC3, 160.6f, TC_RC5, 240.8f, TC_RC7, TC_RC8};

// TAIL: the lane mapping wastes lane-slots whenever m is not S*q*K-shaped (37 particles in 40 slots on 30 lanes).  So up
// to kMaxTail particles of the pass, its LAST mB ones, can be taken out of the mapping and evaluated differently: every
// lane is its own slice (S = 32, q = 1) and applies ITS records to all mB tail particles in scalar arithmetic; the
// mapping then covers the m - mB particles in front (32 + 5 instead of 37: 100 % and 94 % of the lanes busy).  The tail's
// accumulators live in the halves of the top register pairs of the mapping's state, which is why a tail of mB particles
// leaves the mapping 4 - ceil(mB/2) pairs: floor(K/2) + ceil(mB/2) <= kMaxK/2.
#ifndef TC_MAXTAIL
#define TC_MAXTAIL 4
#endif
constexpr int kMaxTail = TC_MAXTAIL;
static_assert(kMaxTail >= 0 && kMaxTail <= 4, "the tail lives in the top two register pairs");
#ifndef TC_TAIL_OVER
#define TC_TAIL_OVER 1.0f
#endif
#ifndef TC_TAIL_MIN_M
#define TC_TAIL_MIN_M 24
#endif
constexpr int kTailMinM = TC_TAIL_MIN_M;      // no tail below this pass size: small groups' chunks are short and the tail's own loop
                                              // set-up per chunk costs more than the slots it saves (N_group = 16: 8.65 -> 8.99 ms with tails)
constexpr float kTailCycles = 47.3f / 32.f;   // cycles per list entry and tail particle: the K = 1 loop at S = 32
constexpr float kTailOverhead = TC_TAIL_OVER; // per list entry: the tail's own loop set-up per chunk (positions, unpack / repack);
                                              // measured: tail off 5.777 ms, on 5.746 (overhead 0.3) / 5.738 (1.0) at config 3

struct LaneMap {
  unsigned char S, q, K, mB;   // mB: particles of the tail (the mapping covers m - mB)
};

// The table is a TEMPLATE over the tail limit: libtc_b200.so holds translation units with different limits (the sparse kernel
// build has none, the dense build and the builders' cost model use 4), and one class name with two different inline
// constructors would break the one-definition rule.  LaneTableT<0> and LaneTableT<4> are simply different types.
template <int MaxTail>
struct LaneTableT {
  static_assert(MaxTail >= 0 && MaxTail <= 4, "the tail lives in the top two register pairs");
  LaneMap map[kPassCap + 1];
  int cost8[kPassCap + 1];    // cycles per list entry of a pass over m particles, in units of 1/8 cycle
  constexpr LaneTableT() : map{}, cost8{} {
    map[0] = LaneMap{1, 32, 1, 0};
    cost8[0] = 0;
    for (int m = 1; m <= kPassCap; m++) {
      int bs = 0, bq = 0, bk = 0, bb = 0;
      float best = 1e30f;
      for (int mb = 0; mb <= (m >= kTailMinM ? MaxTail : 0) && mb < m; mb++) {
        const float tail = mb ? kTailCycles * (float)mb + kTailOverhead : 0.f;
        for (int s = 1; s <= 32; s++) {
          const int q = 32 / s;
          const int k = (m - mb + q - 1) / q;
          if (k > kMaxK || k / 2 + (mb + 1) / 2 > kMaxK / 2) continue;
          const float c = kRecordCycles[k] / (float)s + tail;
          if (c < best) { best = c; bs = s; bq = q; bk = k; bb = mb; }
        }
      }
      map[m] = LaneMap{(unsigned char)bs, (unsigned char)bq, (unsigned char)bk, (unsigned char)bb};
      cost8[m] = (int)(best * 8.f + 0.5f);
    }
  }
  // every pass size has a mapping, no tail is longer than the limit the kernel of this translation unit was compiled for
  // (a longer one would leave the last particles of a pass unevaluated, silently), and mapping + tail cover the pass
  constexpr bool consistent() const {
    for (int m = 1; m <= kPassCap; m++) {
      const LaneMap& l = map[m];
      if (l.mB > MaxTail || l.S < 1 || l.q != 32 / l.S || l.K < 1 || l.K > kMaxK) return false;
      if ((int)l.q * l.K < m - l.mB || l.K / 2 + (l.mB + 1) / 2 > kMaxK / 2) return false;
    }
    return true;
  }
};
using LaneTable = LaneTableT<kMaxTail>;   // the table of THIS translation unit
static_assert(LaneTable().consistent(), "lane table: a mapping exceeds this build's tail limit or does not cover its pass");

// Cost class of a whole group of `cnt` particles for the schedule (costly groups run first): cycles per
// list entry in 1/8 cycles, integer so that the host and the device builder agree bit for bit; <= kMaxCostClass.
// `shift` coarsens the classes (schedule_class_shift below): inside a class the groups stay in Morton order.
constexpr int kMaxCostClass = 1000000;
template <int MaxTail>
TC_HD constexpr int group_cost_class(const LaneTableT<MaxTail>& t, long long cnt, int shift) {
  const long long c = ((cnt / kPassCap) * (long long)t.cost8[kPassCap] + (long long)t.cost8[cnt % kPassCap]) >> shift;
  return c > kMaxCostClass ? kMaxCostClass : (int)c;
}
// Costly-first order only matters for the tail of the launch: with few groups per warp (config 3: 35 603 groups on 2 368
// persistent warps) the exact order is worth 5 % (5.78 against 6.10 ms in pure Morton order).  With hundreds of groups per
// warp the tail is nothing and PURE MORTON order keeps the warps in flight on neighbouring groups, which is what the L2
// sees when the tree no longer fits in it (N = 2^24: 0.6 GB of tree, profiles/r02_walk_literal_config5.md).
#ifndef TC_MORTON_MIN_GROUPS
#define TC_MORTON_MIN_GROUPS 400000
#endif
TC_HD constexpr int schedule_class_shift(long long n_groups) { return n_groups >= TC_MORTON_MIN_GROUPS ? 30 : 0; }

}  // namespace tc

// Host octree builder of the B200 tree-code (step A0 of DESIGN.md).
//
// The paper keeps tree construction and multipole moments on the host
// (PAPER.md:17,41); so does this library.  Unlike the paper's sequential builder
// this one is a Morton-key radix sort followed by a level-by-level
// (breadth-first) split of sorted key ranges, OpenMP-parallel inside each level,
// and a bottom-up parallel-axis accumulation of the fp64 moments.  Cells come out
// in breadth-first order with the children of a node contiguous, which is what the
// walk kernel wants: the 8 child tests of a node are 8 adjacent float4 loads.
//
// Readings: O1 root cube + integer grid, O2 leaf iff count <=
// N_leaf or level 21, children = non-empty octants in order 4bx+2by+bz, O3 tight
// bbox -> boundary cube, mass, COM, traceless quadrupole, O4 groups.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <memory>
#include <new>

#ifdef _OPENMP
#include <omp.h>
#endif

#include "tc_internal.h"
#include "tc_lanes.h"

namespace tc {
namespace {

inline uint64_t spread21(uint64_t v) {  // bit i -> bit 3i
  v &= 0x1fffffull;
  v = (v | (v << 32)) & 0x1f00000000ffffull;
  v = (v | (v << 16)) & 0x1f0000ff0000ffull;
  v = (v | (v << 8)) & 0x100f00f00f00f00full;
  v = (v | (v << 4)) & 0x10c30c30c30c30c3ull;
  v = (v | (v << 2)) & 0x1249249249249249ull;
  return v;
}

// Sort element: the top 3 BITS bits of the Morton key (the first BITS tree levels) above the particle index,
// in ONE 64-bit word (half the memory traffic of a (key, idx) pair in every pass of the sort, and the arrays
// of 2^20 particles stay in the cache).  The full keys are kept beside it, in the caller's order, for the rare
// cells that are split below level BITS.
struct SortPlan {
  int bits;        // tree levels covered by the sorted prefix (3 bits each)
  int low;         // 63 - 3 bits: key bits below the sorted prefix
  int idxb;        // 64 - 3 bits: index bits of an element
  uint64_t imask;  // (1 << idxb) - 1
};
inline SortPlan sort_plan(int64_t n) {
  // a prefix of 11 levels is enough up to a few million particles; deeper trees want a longer one (fewer cells
  // finished by the comparison sort: 33 vs 40 ms at N = 2^24), as far as the index still fits beside it
  const int bits = (n > (int64_t(1) << 22) && n <= (int64_t(1) << 25)) ? 13 : 11;   // 13 levels leave 25 index bits
  SortPlan P;
  P.bits = bits; P.low = 63 - 3 * bits; P.idxb = 64 - 3 * bits; P.imask = (uint64_t(1) << P.idxb) - 1;
  return P;
}

// O1: integer grid coordinates and 63-bit Morton keys of all particles; returns the OR of all keys.
// One body, two instantiations: baseline x86-64, and AVX2 + BMI2 (vectorised floor / min / max, bit
// interleave by PDEP), chosen at run time — the arithmetic is the same correctly rounded fp64 sequence.
#define TC_KEYS_BODY(SPREAD)                                                                        \
  uint64_t key_or = 0;                                                                              \
  _Pragma("omp parallel for schedule(static) reduction(| : key_or)")                                \
  for (int64_t i = 0; i < n; i++) {                                                                 \
    uint64_t g[3];                                                                                  \
    for (int k = 0; k < 3; k++) {                                                                   \
      double v = std::floor(((double)pos[4 * i + k] - org[k]) * scale);                             \
      v = std::min(std::max(v, 0.0), gmax);                                                         \
      g[k] = (uint64_t)v;                                                                           \
    }                                                                                               \
    /* octant o = 4 bx + 2 by + bz at every level  ->  x is the most significant of each triple */  \
    const uint64_t key = (SPREAD(g[0]) << 2) | (SPREAD(g[1]) << 1) | SPREAD(g[2]);                  \
    fullkey[i] = key; elem[i] = ((key >> low) << idxb) | (uint64_t)i;                               \
    key_or |= key;                                                                                  \
  }                                                                                                 \
  return key_or;

uint64_t compute_keys_base(const float* pos /* (x,y,z,m) per particle */, int64_t n, const double* org, double scale, double gmax, uint64_t* fullkey,
                           uint64_t* elem, int low, int idxb) {
  TC_KEYS_BODY(spread21)
}
#if defined(__x86_64__) && defined(__GNUC__)
#define TC_PDEP21(x) __builtin_ia32_pdep_di((x), 0x1249249249249249ull)
#pragma GCC push_options
#pragma GCC target("avx2,bmi2")
uint64_t compute_keys_v3(const float* pos, int64_t n, const double* org, double scale, double gmax, uint64_t* fullkey,
                         uint64_t* elem, int low, int idxb) {
  TC_KEYS_BODY(TC_PDEP21)
}
#pragma GCC pop_options
#endif
uint64_t compute_keys(const float* pos, int64_t n, const double* org, double scale, double gmax, uint64_t* fullkey,
                      uint64_t* elem, int low, int idxb) {
#if defined(__x86_64__) && defined(__GNUC__)
  if (__builtin_cpu_supports("avx2") && __builtin_cpu_supports("bmi2")) return compute_keys_v3(pos, n, org, scale, gmax, fullkey, elem, low, idxb);
#endif
  return compute_keys_base(pos, n, org, scale, gmax, fullkey, elem, low, idxb);
}

// Sort of the elements by Morton key, stable (equal keys keep ascending index).  NP LSD radix passes
// order them by the 3 BITS-bit key prefix they carry (BITS tree levels); a run of equal prefixes only needs its low
// key bits ordered when it is longer than `n_leaf` (it is then split below level BITS), which is rare — those
// runs are finished with std::stable_sort on the full keys.  Shorter runs end up inside one leaf, where the
// order of the members is immaterial (it stays the caller's order).  (Measured with (key, idx) pairs: 11 bits
// 2.5 vs 4.2 ms at N = 2^20, 13 bits 33 vs 40 ms at 2^24.)
// Returns the buffer that holds the sorted array (`a` or `tmp`: no copy back after an odd number of passes).
template <int BITS, int NP>
uint64_t* radix_sort_t(uint64_t* a, uint64_t* tmp, int64_t n, uint64_t key_or, int n_leaf, const uint64_t* fullkey) {
  // the 3 BITS prefix bits are sorted in NP passes; the first (3 BITS) % NP passes take one bit more
  constexpr int WB = (3 * BITS) / NP, WREM = (3 * BITS) % NP;
  constexpr int R = 1 << (WB + (WREM ? 1 : 0)), LOW = 63 - 3 * BITS, IDXB = 64 - 3 * BITS;
  constexpr uint64_t IMASK = (uint64_t(1) << IDXB) - 1;
  const auto by_full_key = [fullkey](uint64_t x, uint64_t y) { return fullkey[x & IMASK] < fullkey[y & IMASK]; };
  if (n < 8192) {   // small inputs: the histograms would cost more than the sort
    std::stable_sort(a, a + n, by_full_key);
    return a;
  }
  int nthreads = 1;
#ifdef _OPENMP
  nthreads = omp_get_max_threads();
#endif
  if (n < (1 << 16)) nthreads = 1;
  std::vector<int64_t> hist((size_t)nthreads * R);
  uint64_t* src = a;
  uint64_t* dst = tmp;
  int done = 0;                                                       // prefix bits already sorted
  for (int pass = 0; pass < NP; pass++) {
    const int w = WB + (pass < WREM ? 1 : 0);
    const uint64_t dmask = (uint64_t(1) << w) - 1;
    const int shift = IDXB + done;
    done += w;
    if (((key_or >> (shift - IDXB + LOW)) & dmask) == 0) continue;    // digit is zero in every key
    std::fill(hist.begin(), hist.end(), 0);
#pragma omp parallel num_threads(nthreads)
    {
#ifdef _OPENMP
      const int t = omp_get_thread_num();
#else
      const int t = 0;
#endif
      const int64_t lo = n * t / nthreads, hi = n * (t + 1) / nthreads;
      int64_t* h = &hist[(size_t)t * R];
      for (int64_t i = lo; i < hi; i++) h[(src[i] >> shift) & dmask]++;
#pragma omp barrier
#pragma omp single
      {
        int64_t run = 0;
        for (int d = 0; d < R; d++)
          for (int tt = 0; tt < nthreads; tt++) {
            const int64_t c = hist[(size_t)tt * R + d];
            hist[(size_t)tt * R + d] = run;
            run += c;
          }
      }
      for (int64_t i = lo; i < hi; i++) dst[h[(src[i] >> shift) & dmask]++] = src[i];
    }
    std::swap(src, dst);
  }
  a = src;
  // finish the long runs (parallel over run starts; runs are disjoint)
#pragma omp parallel for schedule(dynamic, 65536)
  for (int64_t i = 0; i < n; i++) {
    const uint64_t pre = a[i] >> IDXB;
    if (i > 0 && (a[i - 1] >> IDXB) == pre) continue;      // not a run start
    int64_t j = i + 1;
    while (j < n && j - i <= n_leaf && (a[j] >> IDXB) == pre) j++;
    if (j - i <= n_leaf) continue;
    while (j < n && (a[j] >> IDXB) == pre) j++;
    std::stable_sort(a + i, a + j, by_full_key);
  }
  return a;
}
uint64_t* radix_sort(const SortPlan& P, uint64_t* a, uint64_t* tmp, int64_t n, uint64_t key_or, int n_leaf, const uint64_t* fullkey) {
  // passes: 4 x 8-9 bits for the 33-bit prefix (256-512 write streams per thread stay in L1: 1.8 vs 2.1 ms at N = 2^20,
  // 5 passes 2.6 ms); the longer prefixes of large N are memory-bound per pass, so 3 passes (23 vs 31 ms at 2^24)
  switch (P.bits) {
    case 13: return radix_sort_t<13, 3>(a, tmp, n, key_or, n_leaf, fullkey);
    default: return radix_sort_t<11, 4>(a, tmp, n, key_or, n_leaf, fullkey);
  }
}

struct CellProp {   // fp64 moments, fp32-exact bounding box
  float bmin[3], bmax[3];
  double M, X[3], Q[6];  // Q: xx,yy,zz,xy,xz,yz about X
};

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

void* HostScratch::get(int k, size_t bytes) {
  if (cap[k] < bytes) {
    std::free(buf[k]); buf[k] = nullptr; cap[k] = 0;
    const size_t want = bytes + bytes / 8 + 64;
    buf[k] = std::malloc(want);
    if (buf[k]) cap[k] = want;
  }
  return buf[k];
}
HostScratch::~HostScratch() { for (void* p : buf) std::free(p); }

int build_host_tree(const float4* xyzm, int64_t n, int n_leaf, int n_group,
                    HostTree& T, PackedAlloc alloc, void* alloc_user, std::string& msg, const float* bbox6) {
  if (n < 1 || n_leaf < 1 || n_group < 1) { msg = "build: n, n_leaf, n_group must be >= 1"; return TC_EINVAL; }
  T.n = n; T.n_leaf = n_leaf; T.n_group = n_group;
  const bool timing = std::getenv("TC_BUILD_TIMING") != nullptr;
  double t_prev = omp_get_wtime();
  auto lap = [&](const char* what) { if (timing) { const double t = omp_get_wtime(); std::fprintf(stderr, "[tc_build] %-10s %8.3f ms\n", what, (t - t_prev) * 1e3); t_prev = t; } };

  // ---- O1: root cube and integer grid ("a cube containing all particles")
  double lo[3], hi[3];
  for (int k = 0; k < 3; k++) { lo[k] = std::numeric_limits<double>::infinity(); hi[k] = -lo[k]; }
  if (bbox6) {
    for (int k = 0; k < 3; k++) { lo[k] = (double)bbox6[k]; hi[k] = (double)bbox6[3 + k]; }
  } else {
    double l0 = lo[0], l1 = lo[1], l2 = lo[2], h0 = hi[0], h1 = hi[1], h2 = hi[2];
#pragma omp parallel for schedule(static) reduction(min : l0, l1, l2) reduction(max : h0, h1, h2)
    for (int64_t i = 0; i < n; i++) {
      const double x = (double)xyzm[i].x, y = (double)xyzm[i].y, z = (double)xyzm[i].z;
      l0 = std::min(l0, x); h0 = std::max(h0, x);
      l1 = std::min(l1, y); h1 = std::max(h1, y);
      l2 = std::min(l2, z); h2 = std::max(h2, z);
    }
    lo[0] = l0; lo[1] = l1; lo[2] = l2; hi[0] = h0; hi[1] = h1; hi[2] = h2;
  }
  lap("bbox");
  double ext = 0.0;
  for (int k = 0; k < 3; k++) ext = std::max(ext, hi[k] - lo[k]);
  double side = ext * (1.0 + std::ldexp(1.0, -20));
  if (side == 0.0) side = 1.0;
  double org[3];
  for (int k = 0; k < 3; k++) org[k] = (lo[k] + hi[k]) / 2.0 - side / 2.0;
  const double scale = std::ldexp(1.0, 21) / side;
  const double gmax = std::ldexp(1.0, 21) - 1.0;

  // key buffers: plain arrays (no zero fill; every element is written below)
  // (from the context's grow-only scratch: a rebuild touches no fresh pages)
  const SortPlan SP = sort_plan(n);
  uint64_t* const fullkey = static_cast<uint64_t*>(T.scratch.get(0, sizeof(uint64_t) * (size_t)n));   // caller's order
  uint64_t* keys = static_cast<uint64_t*>(T.scratch.get(1, sizeof(uint64_t) * 2 * (size_t)n));        // elements, and their twin
  if (!fullkey || !keys) { msg = "build: out of host memory"; return TC_ENOMEM; }
  const uint64_t key_or = compute_keys(reinterpret_cast<const float*>(xyzm), n, org, scale, gmax, fullkey, keys, SP.low, SP.idxb);
  lap("keys");
  keys = radix_sort(SP, keys, keys + n, n, key_or, n_leaf, fullkey);
  lap("sort");

  // ---- O2: breadth-first split of sorted key ranges
  // cell arrays (struct of vectors), breadth-first, children contiguous
  std::vector<int32_t>&c_begin = T.scratch.c_begin, &c_count = T.scratch.c_count, &c_first_child = T.scratch.c_first_child,
                      &c_nchild = T.scratch.c_nchild;
  // their SIZE is a high-water mark that survives between builds (a rebuild of the same problem fills nothing in again);
  // the cells of this build are [0, lvl_e), and every one of them is written below
  const auto grow_cells = [&](size_t need) {
    if (c_begin.size() >= need) return;
    const size_t to = std::max(need, c_begin.size() + c_begin.size() / 2);
    c_begin.resize(to); c_count.resize(to); c_first_child.resize(to); c_nchild.resize(to);
  };
  grow_cells(1);
  std::vector<int64_t> level_start;  // first cell id of every level (+ end sentinel)
  c_begin[0] = 0; c_count[0] = (int32_t)n; c_first_child[0] = -1; c_nchild[0] = 0;
  level_start.push_back(0);
  int64_t lvl_b = 0, lvl_e = 1;
  int level = 0;
  std::vector<int32_t>& nch = T.scratch.nch;
  while (true) {
    level_start.push_back(lvl_e);
    if (level == kMaxLevel) break;
    const int shift = 3 * (kMaxLevel - 1 - level);
    // the octant digit of this level: inside the element's prefix for the first `bits` levels, from the full key below
    const bool in_prefix = level < SP.bits;
    const int pshift = SP.idxb + 3 * (SP.bits - 1 - level);
    const uint64_t imask = SP.imask;
    const auto octant = [=](uint64_t q) -> uint64_t { return in_prefix ? (q >> pshift) & 7 : (fullkey[q & imask] >> shift) & 7; };
    const int64_t nl = lvl_e - lvl_b;
    nch.assign((size_t)nl + 1, 0);
    // pass 1: the non-empty octants of every node of this level; their starts are kept for pass 2
    std::vector<int32_t>& bounds = T.scratch.bounds;
    if (bounds.size() < (size_t)nl * 9) bounds.resize((size_t)nl * 9);
    int32_t* const bnds = bounds.data();
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t c = lvl_b; c < lvl_e; c++) {
      if (c_count[c] <= n_leaf) continue;  // leaf (R4: <=)
      const uint64_t* kb = keys + c_begin[c];
      const uint64_t* ke = kb + c_count[c];
      int32_t* bd = bnds + 9 * (size_t)(c - lvl_b);
      int cnt = 0;
      const uint64_t* p = kb;
      while (p < ke) {
        const uint64_t o = octant(*p);
        bd[cnt++] = (int32_t)(p - keys);
        // first key of this cell with octant > o
        p = std::partition_point(p, ke, [&](uint64_t q) { return octant(q) <= o; });
      }
      bd[cnt] = (int32_t)(ke - keys);
      nch[(size_t)(c - lvl_b)] = cnt;
    }
    int64_t total = 0;
    for (int64_t i = 0; i < nl; i++) { const int32_t v = nch[i]; nch[i] = (int32_t)total; total += v; }
    nch[nl] = (int32_t)total;
    if (total == 0) break;
    if (lvl_e + total > (int64_t)0x0fffffff) { msg = "build: more than 2^28 cells"; return TC_EINVAL; }
    const int64_t new_e = lvl_e + total;
    grow_cells((size_t)new_e);
    // pass 2: create the children
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t c = lvl_b; c < lvl_e; c++) {
      const int32_t k = nch[(size_t)(c - lvl_b) + 1] - nch[(size_t)(c - lvl_b)];
      if (k == 0) { c_first_child[c] = -1; c_nchild[c] = 0; continue; }   // leaf
      const int64_t first = lvl_e + nch[(size_t)(c - lvl_b)];
      c_first_child[c] = (int32_t)first; c_nchild[c] = k;
      const int32_t* bd = bnds + 9 * (size_t)(c - lvl_b);
      for (int j = 0; j < k; j++) { c_begin[first + j] = bd[j]; c_count[first + j] = bd[j + 1] - bd[j]; }
    }
    lvl_b = lvl_e; lvl_e = new_e; level++;
  }
  // the last level was not expanded: all of its cells are leaves
  for (int64_t c = lvl_b; c < lvl_e; c++) { c_first_child[c] = -1; c_nchild[c] = 0; }
  const int64_t nc = lvl_e;
  T.n_cells = nc;
  T.depth = (int32_t)level_start.size() - 2;
  const int n_levels = (int)level_start.size() - 1;

  lap("split");
  // ---- O4: groups = maximal cells with count <= N_group, or leaves, Morton order
  std::vector<int32_t>& groups = T.scratch.groups;
  groups.clear();
  {
    std::vector<int32_t> st;
    st.push_back(0);
    while (!st.empty()) {
      const int32_t c = st.back(); st.pop_back();
      if (c_count[c] <= n_group || c_nchild[c] == 0) { groups.push_back(c); continue; }
      for (int j = c_nchild[c] - 1; j >= 0; j--) st.push_back(c_first_child[c] + j);
    }
  }
  T.n_groups = (int64_t)groups.size();

  // ---- pack: SoA float4 arrays in one buffer (layout in tc_internal.h)
  PackedLayout& Y = T.lay;
  size_t off = 0;
  Y.off_bnd = off;  off = align256(off + sizeof(float4) * (size_t)nc);
  Y.off_xm = off;   off = align256(off + sizeof(float4) * (size_t)nc);
  Y.off_q0 = off;   off = align256(off + sizeof(float4) * (size_t)nc);
  Y.off_q1 = off;   off = align256(off + sizeof(float4) * (size_t)nc);
  Y.off_part = off; off = align256(off + sizeof(float4) * (size_t)n);
  Y.off_orig = off; off = align256(off + sizeof(int32_t) * (size_t)n);
  Y.off_grp = off;  off = align256(off + sizeof(int4) * groups.size());
  Y.off_gbox = off; off = align256(off + sizeof(float4) * groups.size());
  Y.bytes = off;
  char* base = (char*)alloc(alloc_user, Y.bytes);
  if (!base) { msg = "build: cannot allocate the packed tree buffer"; return TC_ENOMEM; }
  float4* bnd = (float4*)(base + Y.off_bnd);
  float4* xm = (float4*)(base + Y.off_xm);
  float4* q0 = (float4*)(base + Y.off_q0);
  float4* q1 = (float4*)(base + Y.off_q1);
  float4* part = (float4*)(base + Y.off_part);
  int32_t* orig = (int32_t*)(base + Y.off_orig);
  int4* grp = (int4*)(base + Y.off_grp);
  float4* gbox = (float4*)(base + Y.off_gbox);
  lap("groups");
  // particles in tree (Morton) order, gathered ONCE straight into the packed buffer: the moments below and the
  // kernels read them sequentially
#pragma omp parallel for schedule(static)
  for (int64_t t = 0; t < n; t++) {
    const int64_t i = (int64_t)(keys[t] & SP.imask);
    part[t] = xyzm[i];                       // one aligned 16-byte read per particle
    orig[t] = (int32_t)i;
  }
  lap("gather");
  // ---- O3: cell properties, fp64, bottom-up.  Leaves: direct sums
  // over members.  Nodes: union of the children's boxes, parallel-axis shift of the
  // children's moments to the node's centre of mass.
  CellProp* prop = static_cast<CellProp*>(T.scratch.get(2, sizeof(CellProp) * (size_t)nc));   // every entry is written below
  if (!prop) { msg = "build: out of host memory"; return TC_ENOMEM; }
  int64_t n_leaves = 0;
  for (int L = n_levels - 1; L >= 0; L--) {
    const int64_t b = level_start[L], e = level_start[L + 1];
#pragma omp parallel for schedule(dynamic, 128) reduction(+ : n_leaves)
    for (int64_t c = b; c < e; c++) {
      CellProp& P = prop[c];
      double M = 0.0, S[3] = {0, 0, 0};
      if (c_nchild[c] == 0) {
        n_leaves++;
        float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
        const int64_t pb = c_begin[c], pe = pb + c_count[c];
        for (int64_t t = pb; t < pe; t++) {
          const float4 b = part[t];
          const float xyz[3] = {b.x, b.y, b.z};
          const double m = (double)b.w;
          for (int k = 0; k < 3; k++) {
            const float v = xyz[k];
            mn[k] = std::min(mn[k], v); mx[k] = std::max(mx[k], v);
            S[k] += m * (double)v;
          }
          M += m;
        }
        for (int k = 0; k < 3; k++) { P.bmin[k] = mn[k]; P.bmax[k] = mx[k]; }
        P.M = M;
        for (int k = 0; k < 3; k++)  // massless cell (R19): centre of the boundary cube
          P.X[k] = (M > 0.0) ? S[k] / M : ((double)mn[k] + (double)mx[k]) / 2.0;
        double Q[6] = {0, 0, 0, 0, 0, 0};
        for (int64_t t = pb; t < pe; t++) {
          const float4 b = part[t];
          const double m = (double)b.w;
          const double yx = (double)b.x - P.X[0], yy = (double)b.y - P.X[1], yz = (double)b.z - P.X[2];
          const double y2 = yx * yx + yy * yy + yz * yz;
          Q[0] += m * (3.0 * yx * yx - y2); Q[1] += m * (3.0 * yy * yy - y2); Q[2] += m * (3.0 * yz * yz - y2);
          Q[3] += m * (3.0 * yx * yy); Q[4] += m * (3.0 * yx * yz); Q[5] += m * (3.0 * yy * yz);
        }
        for (int k = 0; k < 6; k++) P.Q[k] = Q[k];
      } else {
        const int64_t f = c_first_child[c], l = f + c_nchild[c];
        for (int k = 0; k < 3; k++) { P.bmin[k] = INFINITY; P.bmax[k] = -INFINITY; }
        for (int64_t ch = f; ch < l; ch++) {
          const CellProp& C = prop[ch];
          for (int k = 0; k < 3; k++) {
            P.bmin[k] = std::min(P.bmin[k], C.bmin[k]); P.bmax[k] = std::max(P.bmax[k], C.bmax[k]);
            S[k] += C.M * C.X[k];
          }
          M += C.M;
        }
        P.M = M;
        for (int k = 0; k < 3; k++)
          P.X[k] = (M > 0.0) ? S[k] / M : ((double)P.bmin[k] + (double)P.bmax[k]) / 2.0;
        double Q[6] = {0, 0, 0, 0, 0, 0};
        for (int64_t ch = f; ch < l; ch++) {
          const CellProp& C = prop[ch];
          const double dx = C.X[0] - P.X[0], dy = C.X[1] - P.X[1], dz = C.X[2] - P.X[2];
          const double d2 = dx * dx + dy * dy + dz * dz;
          Q[0] += C.Q[0] + C.M * (3.0 * dx * dx - d2); Q[1] += C.Q[1] + C.M * (3.0 * dy * dy - d2);
          Q[2] += C.Q[2] + C.M * (3.0 * dz * dz - d2);
          Q[3] += C.Q[3] + C.M * (3.0 * dx * dy); Q[4] += C.Q[4] + C.M * (3.0 * dx * dz);
          Q[5] += C.Q[5] + C.M * (3.0 * dy * dz);
        }
        for (int k = 0; k < 6; k++) P.Q[k] = Q[k];
      }
    }
  }
  T.n_leaves = n_leaves;

  lap("moments");
  try { T.link.resize((size_t)nc * 4); T.q6.resize((size_t)nc * 6); } catch (...) { msg = "build: out of host memory"; return TC_ENOMEM; }

#pragma omp parallel for schedule(static)
  for (int64_t c = 0; c < nc; c++) {
    const CellProp& P = prop[c];
    // boundary cube (Fig. 1): same centre as the tight box, side = its largest side.
    // FP32 form (R20): centre rounded to nearest, half side = reach of the tight box
    // from that rounded centre, rounded towards +inf, so the fp32 cube contains the box and the
    // opening test gives d = 0 exactly for every cell inside the group (R14).
    float b[3];
    double reach = 0.0;
    for (int k = 0; k < 3; k++) {
      const double lo = (double)P.bmin[k], hi = (double)P.bmax[k];
      b[k] = (float)(0.5 * (lo + hi));
      reach = std::fmax(reach, std::fmax(hi - (double)b[k], (double)b[k] - lo));
    }
    float h = (float)reach;
    if ((double)h < reach) h = std::nextafter(h, HUGE_VALF);
    const bool leaf = c_nchild[c] == 0;
    bnd[c] = make_float4(b[0], b[1], b[2], leaf ? -h : h);  // sign bit of h <=> leaf (-0.0f if h == 0)
    xm[c] = make_float4((float)P.X[0], (float)P.X[1], (float)P.X[2], (float)P.M);
    // the device arrays carry -Q: the packed-FP32 evaluation then needs no run-time negation (tc_kernels.cu)
    q0[c] = make_float4(-(float)P.Q[0], -(float)P.Q[1], -(float)P.Q[2], -(float)P.Q[3]);
    int32_t la, lb;
    if (leaf) { la = c_begin[c]; lb = c_count[c]; } else { la = c_first_child[c]; lb = c_nchild[c]; }
    float fa, fb;
    std::memcpy(&fa, &la, 4); std::memcpy(&fb, &lb, 4);
    q1[c] = make_float4(-(float)P.Q[4], -(float)P.Q[5], fa, fb);
    T.link[4 * c + 0] = leaf ? -1 : c_first_child[c];
    T.link[4 * c + 1] = c_nchild[c];
    T.link[4 * c + 2] = c_begin[c];
    T.link[4 * c + 3] = c_count[c];
    for (int k = 0; k < 6; k++) T.q6[6 * c + k] = (float)P.Q[k];
  }
  lap("pack");
  // Schedule (grp[i].w = i-th group to run): the persistent kernel hands groups out through an
  // atomic counter, so costly groups go first and the tail of the launch is made of cheap ones.
  // Cost model = issue slots per list entry of the kernel's lane mapping: tc_lanes.h, the table the kernel
  // itself reads.  Stable: Morton order inside a cost class keeps neighbouring groups together.
  {
    static constexpr LaneTable lanes = LaneTable();
    const int shift = schedule_class_shift((long long)groups.size());
    // counting sort by cost class, descending; stable, so Morton order survives inside a class
    const size_t ng = groups.size();
    std::vector<int32_t> cls(ng);
    int32_t cmax = 0;
#pragma omp parallel for schedule(static) reduction(max : cmax)
    for (size_t g = 0; g < ng; g++) {
      const int64_t cnt = c_count[groups[g]];
      cls[g] = group_cost_class(lanes, cnt, shift);
      cmax = std::max(cmax, cls[g]);
    }
    std::vector<int32_t> start((size_t)cmax + 2, 0);
    for (size_t g = 0; g < ng; g++) start[(size_t)(cmax - cls[g]) + 1]++;
    for (size_t k = 1; k < start.size(); k++) start[k] += start[k - 1];
    std::vector<int32_t> order(ng);
    for (size_t g = 0; g < ng; g++) order[(size_t)start[(size_t)(cmax - cls[g])]++] = (int32_t)g;
#pragma omp parallel for schedule(static)
    for (size_t g = 0; g < ng; g++) {
      const int32_t c = groups[g];
      grp[g] = make_int4(c, c_begin[c], c_count[c], order[g]);
      // variant R23: half extents of the tight box about the fp32 centre of the boundary cube, per axis,
      // rounded towards +inf (the R20 construction axis by axis; their maximum is the cube's half side)
      float e[3];
      for (int k = 0; k < 3; k++) {
        const double lo = (double)prop[c].bmin[k], hi = (double)prop[c].bmax[k];
        const float bk = (float)(0.5 * (lo + hi));
        const double reach = std::fmax(hi - (double)bk, (double)bk - lo);
        e[k] = (float)reach;
        if ((double)e[k] < reach) e[k] = std::nextafter(e[k], HUGE_VALF);
      }
      gbox[g] = make_float4(e[0], e[1], e[2], 0.f);
    }
  }
  lap("schedule");
  return TC_OK;
}

}  // namespace tc

// ============================================================================
//  ORACLE — TEST INFRASTRUCTURE ONLY.  NOT PART OF THE PRODUCT PATH.
//
//  A plain, slow, fp64 CPU restatement of the force calculation of
//  arXiv 1005.5384 (Gaburov, Bedorf, Portegies Zwart, ICCS 2010), written from
//  the paper under the readings O1-O6 / R1-R18 of
//  SURVEY.md §8(c) (restated in DESIGN.md §3).  Only tests/, __graft_entry__.smoke()
//  and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
//  It shares no code, header, table or helper with paper_1005_5384_b200/csrc/.
//
//  Everything is fp64 on the fp32 inputs widened to fp64, compiled with
//  -ffp-contract=off.  The only fp32 arithmetic is the optional "shadow" of
//  the opening test (R16): the paper's device code works in FP32
//  (PAPER.md:145,185), so where floating point decides an integer (open / do
//  not open) the decision can be taken in that precision by BOTH sides; the
//  fp64 decision is always computed beside it and disagreements ("borderline
//  opening flips") are counted per group.
//
//  Pins (tests/test_oracle_*.py, -m "not gpu"):
//    tree        : brute-force cell enumeration from the definition; invariants
//    moments     : parallel-axis merge of children; tracelessness; COM in bbox
//    quadrupole  : closed form, two masses at +-s (tests/golden/quadrupole_two_mass.txt)
//    softened quadrupole (R11, sigma^2 = r^2 + eps^2 in the s^-5 and s^-7 terms too): hand-evaluated values at
//                  eps = 0.375, 0.5 and 0.1 with Q != 0, on and off axis
//                  (tests/golden/quadrupole_two_mass_softened.txt), and a = -grad(phi) of the same cell term by
//                  central differences at eps = 0, 0.1, 0.5
//    walk        : coverage invariant; theta = 0; brute force over all (group, cell) pairs
//    evaluation  : N = 2 closed form; theta = 0 == direct sum; theta -> 0 convergence;
//                  momentum invariant; Plummer analytic field
//    direct sum  : N = 2, N = 3 closed forms; sum m a = 0
//    variants    : R21 (opening test on the cell's centre of mass) and R22 (monopole-only cells), both off
//                  by default: lists re-derived from the recursive definition, theta = 0, own cells open
//                  in fp32, monopole closed form, error orders (tests/test_oracle_variants.py);
//                  R23 (the group enters the opening test as its tight box): hand-computed threshold of an
//                  elongated group (tests/golden/group_box_threshold.txt), interval-gap brute force
//  "parity unpinned": the opening RULE itself (R1) — the paper never prints
//  its formula (PAPER.md:79 calls open_node, never defined) — and every value
//  that lives only in Figs. 4-8.
// ============================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int MAXLEV = 21;  // R7: 21 levels, 63-bit key space

struct OCell {
  int level;
  int parent;
  int child[8];       // cell id per octant o = 4 bx + 2 by + bz, -1 = empty (R6)
  int n_child;        // number of non-empty octants; 0 <=> leaf
  int64_t begin, count;  // members are perm[begin .. begin+count)
  double bmin[3], bmax[3];  // tight bounding box (Fig. 1)
  double b[3], h;           // boundary cube: centre, half side (Fig. 1)
  double M, X[3];           // mass, centre of mass
  double Q[6];              // traceless quadrupole about X: xx,yy,zz,xy,xz,yz (R10)
  float b32[3], h32;        // fp32-rounded boundary (what an FP32 device stores)
  float e32[3];             // R23: fp32 half extents of the tight box about b32, per axis, rounded up
};

struct Oracle {
  int64_t n = 0;
  int n_leaf = 0, n_group = 0;
  // variants (R21, R22): 0 = the default readings
  int open_rule = 0;   // 0: cube-to-cube distance (R1); 1: group cube to the cell's centre of mass (R21)
  int quadrupole = 1;  // 1: monopole + quadrupole (R10); 0: monopole only (R22)
  int group_box = 0;   // 0: the group is its boundary cube (R9); 1: its tight box, per-axis half extents (R23)
  std::vector<double> x, y, z, m;  // inputs widened to fp64
  std::vector<int32_t> gx, gy, gz; // O1 integer grid coordinates
  double org[3], side;
  std::vector<int64_t> perm;       // Morton-ordered particle indices (result of the recursion)
  std::vector<OCell> cells;
  std::vector<int> groups;         // cell ids, Morton order (O4)
  int depth = 0;
  int64_t n_leaves = 0;
};

// ---- O1: root cube and integer grid ("a cube containing all particles"; R8)
void root_cube(Oracle& T) {
  double lo[3], hi[3];
  for (int k = 0; k < 3; k++) { lo[k] = std::numeric_limits<double>::infinity(); hi[k] = -lo[k]; }
  for (int64_t i = 0; i < T.n; i++) {
    const double p[3] = {T.x[i], T.y[i], T.z[i]};
    for (int k = 0; k < 3; k++) { lo[k] = std::min(lo[k], p[k]); hi[k] = std::max(hi[k], p[k]); }
  }
  double ext = 0.0;
  for (int k = 0; k < 3; k++) ext = std::max(ext, hi[k] - lo[k]);
  double side = ext * (1.0 + std::ldexp(1.0, -20));
  if (side == 0.0) side = 1.0;
  T.side = side;
  for (int k = 0; k < 3; k++) {
    const double c = (lo[k] + hi[k]) / 2.0;
    T.org[k] = c - side / 2.0;
  }
  const double scale = std::ldexp(1.0, 21) / side;
  const double gmax = std::ldexp(1.0, 21) - 1.0;
  T.gx.resize(T.n); T.gy.resize(T.n); T.gz.resize(T.n);
  for (int64_t i = 0; i < T.n; i++) {
    const double p[3] = {T.x[i], T.y[i], T.z[i]};
    int32_t g[3];
    for (int k = 0; k < 3; k++) {
      double v = std::floor((p[k] - T.org[k]) * scale);
      v = std::min(std::max(v, 0.0), gmax);
      g[k] = (int32_t)v;
    }
    T.gx[i] = g[0]; T.gy[i] = g[1]; T.gz[i] = g[2];
  }
}

// ---- O3: cell properties by direct sums over the members (R10)
void cell_properties(Oracle& T, OCell& c) {
  for (int k = 0; k < 3; k++) { c.bmin[k] = std::numeric_limits<double>::infinity(); c.bmax[k] = -c.bmin[k]; }
  double M = 0.0, S[3] = {0, 0, 0};
  for (int64_t t = c.begin; t < c.begin + c.count; t++) {
    const int64_t i = T.perm[t];
    const double p[3] = {T.x[i], T.y[i], T.z[i]};
    for (int k = 0; k < 3; k++) {
      c.bmin[k] = std::min(c.bmin[k], p[k]);
      c.bmax[k] = std::max(c.bmax[k], p[k]);
      S[k] += T.m[i] * p[k];
    }
    M += T.m[i];
  }
  double ext = 0.0;
  for (int k = 0; k < 3; k++) {
    c.b[k] = (c.bmin[k] + c.bmax[k]) / 2.0;
    ext = std::max(ext, c.bmax[k] - c.bmin[k]);
  }
  c.h = ext / 2.0;
  c.M = M;
  for (int k = 0; k < 3; k++) c.X[k] = (M > 0.0) ? S[k] / M : c.b[k];  // massless cell: reading R19
  double Q[6] = {0, 0, 0, 0, 0, 0};
  for (int64_t t = c.begin; t < c.begin + c.count; t++) {
    const int64_t i = T.perm[t];
    const double yx = T.x[i] - c.X[0], yy = T.y[i] - c.X[1], yz = T.z[i] - c.X[2];
    const double y2 = yx * yx + yy * yy + yz * yz;
    Q[0] += T.m[i] * (3.0 * yx * yx - y2);
    Q[1] += T.m[i] * (3.0 * yy * yy - y2);
    Q[2] += T.m[i] * (3.0 * yz * yz - y2);
    Q[3] += T.m[i] * (3.0 * yx * yy);
    Q[4] += T.m[i] * (3.0 * yx * yz);
    Q[5] += T.m[i] * (3.0 * yy * yz);
  }
  for (int k = 0; k < 6; k++) c.Q[k] = Q[k];
  // R20: the FP32 representation of the boundary must still CONTAIN the tight
  // box, otherwise rounding of b or h can push a particle on a face of its own group's box
  // outside the group's cube and R14 (the own leaf opens, d = 0) is lost in FP32.
  // b32 = fp32(b); h32 = the largest distance from b32 to a face of the tight box, rounded UP.
  for (int k = 0; k < 3; k++) c.b32[k] = (float)c.b[k];
  double far = 0.0;
  for (int k = 0; k < 3; k++) {
    far = std::max(far, c.bmax[k] - (double)c.b32[k]);
    far = std::max(far, (double)c.b32[k] - c.bmin[k]);
  }
  float hf = (float)far;
  if ((double)hf < far) hf = std::nextafterf(hf, std::numeric_limits<float>::infinity());
  c.h32 = hf;
  // R23: the same containment argument per axis (the tight box seen from the rounded centre)
  for (int k = 0; k < 3; k++) {
    const double reach = std::max(c.bmax[k] - (double)c.b32[k], (double)c.b32[k] - c.bmin[k]);
    float ef = (float)reach;
    if ((double)ef < reach) ef = std::nextafterf(ef, std::numeric_limits<float>::infinity());
    c.e32[k] = ef;
  }
}

// ---- O2: recursive cubic subdivision (R4, R6, R7)
int build_cell(Oracle& T, int64_t begin, int64_t count, int level, int parent, std::vector<int64_t>& tmp) {
  const int id = (int)T.cells.size();
  T.cells.emplace_back();
  {
    OCell& c = T.cells[id];
    c.level = level; c.parent = parent; c.begin = begin; c.count = count; c.n_child = 0;
    for (int o = 0; o < 8; o++) c.child[o] = -1;
  }
  T.depth = std::max(T.depth, level);
  const bool leaf = (count <= T.n_leaf) || (level == MAXLEV);
  if (leaf) { T.n_leaves++; cell_properties(T, T.cells[id]); return id; }
  // split on bit (20 - level) of each grid coordinate: the child's level is level+1
  const int bit = MAXLEV - 1 - level;
  int64_t cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  auto octant = [&](int64_t i) {
    return 4 * ((T.gx[i] >> bit) & 1) + 2 * ((T.gy[i] >> bit) & 1) + ((T.gz[i] >> bit) & 1);
  };
  for (int64_t t = begin; t < begin + count; t++) cnt[octant(T.perm[t])]++;
  int64_t off[8], run = 0;
  for (int o = 0; o < 8; o++) { off[o] = run; run += cnt[o]; }
  {
    int64_t pos[8];
    for (int o = 0; o < 8; o++) pos[o] = off[o];
    for (int64_t t = begin; t < begin + count; t++) { const int64_t i = T.perm[t]; tmp[pos[octant(i)]++] = i; }
    for (int64_t t = 0; t < count; t++) T.perm[begin + t] = tmp[t];
  }
  for (int o = 0; o < 8; o++) {
    if (cnt[o] == 0) continue;
    const int ch = build_cell(T, begin + off[o], cnt[o], level + 1, id, tmp);
    T.cells[id].child[o] = ch;
    T.cells[id].n_child++;
  }
  cell_properties(T, T.cells[id]);
  return id;
}

// ---- O4: groups = maximal cells with count <= N_group, or leaves (R5)
void find_groups(Oracle& T, int c) {
  const OCell& C = T.cells[c];
  if (C.count <= T.n_group || C.n_child == 0) { T.groups.push_back(c); return; }
  for (int o = 0; o < 8; o++) if (C.child[o] >= 0) find_groups(T, C.child[o]);
}

// ---- O5: the opening test (List 2 PAPER.md:73-91 `open_node`; R1, R9, R14)
//  fp64: d_k = max(0, |b_c,k - b_g,k| - h_c - h_g), open iff d^2 theta^2 <= (2 h_c)^2
//  rule 1 (R21): the cell is represented by its centre of mass: d_k = max(0, |X_c,k - b_g,k| - h_g)
inline bool open64(const OCell& c, const OCell& g, double theta, double* margin, int rule, int gbox) {
  double d2 = 0.0;
  for (int k = 0; k < 3; k++) {
    // the group's side of the test: half side of its boundary cube (R9), or, variant R23,
    // the half extent of its tight box along this axis
    const double hg = gbox ? (g.bmax[k] - g.bmin[k]) / 2.0 : g.h;
    const double d = rule ? std::max(0.0, std::fabs(c.X[k] - g.b[k]) - hg)
                          : std::max(0.0, std::fabs(c.b[k] - g.b[k]) - c.h - hg);
    d2 += d * d;
  }
  const double l = 2.0 * c.h;
  if (margin) *margin = (l > 0.0) ? std::fabs(std::sqrt(d2) * theta - l) / l : std::numeric_limits<double>::infinity();
  return d2 * theta * theta <= l * l;
}
//  fp32 shadow (R16): the same test on the fp32-rounded boundaries in one fixed
//  sequence of correctly rounded fp32 operations:
//     s = h_c + h_g;  t_k = max(|b_c,k - b_g,k| - s, 0)
//     d2 = fma(t_z,t_z, fma(t_y,t_y, t_x*t_x));  l = h_c + h_c
//     open iff d2 * (theta*theta) <= l * l
//  rule 1: the same sequence with the fp32 centre of mass in place of b_c and 0 in place of h_c
//  gbox (R23): s_k = h_c + e_g,k per axis in place of s
inline bool open32(const OCell& c, const OCell& g, float theta, int rule, int gbox) {
  float t[3];
  for (int k = 0; k < 3; k++) {
    const float s = (rule ? 0.0f : c.h32) + (gbox ? g.e32[k] : g.h32);
    const float u = (rule ? (float)c.X[k] : c.b32[k]) - g.b32[k];
    const float v = std::fabs(u) - s;
    t[k] = std::fmax(v, 0.0f);
  }
  float d2 = t[0] * t[0];
  d2 = std::fmaf(t[1], t[1], d2);
  d2 = std::fmaf(t[2], t[2], d2);
  const float th2 = theta * theta;
  const float l = c.h32 + c.h32;
  const float lhs = d2 * th2;
  const float rhs = l * l;
  return lhs <= rhs;
}

struct WalkOut {
  std::vector<int> cell_list, leaf_list;
  double min_margin = std::numeric_limits<double>::infinity();
  int64_t n_flips = 0;   // tests where the fp32 shadow and the fp64 decision differ
  int64_t n_tests = 0;
};

// mode 0: decide in fp64; mode 1: decide with the fp32 shadow
void walk_group(const Oracle& T, int gcell, double theta, int mode, WalkOut& W) {
  W.cell_list.clear(); W.leaf_list.clear();
  W.min_margin = std::numeric_limits<double>::infinity(); W.n_flips = 0; W.n_tests = 0;
  const OCell& G = T.cells[gcell];
  if (T.cells[0].n_child == 0) { W.leaf_list.push_back(0); return; }  // root is a leaf
  std::vector<int> stack;
  stack.push_back(0);
  while (!stack.empty()) {
    const int node = stack.back(); stack.pop_back();
    const OCell& P = T.cells[node];
    for (int o = 0; o < 8; o++) {
      const int ch = P.child[o];
      if (ch < 0) continue;
      const OCell& C = T.cells[ch];
      double margin;
      const bool o64 = open64(C, G, theta, &margin, T.open_rule, T.group_box);
      const bool o32 = open32(C, G, (float)theta, T.open_rule, T.group_box);
      W.n_tests++;
      W.min_margin = std::min(W.min_margin, margin);
      if (o64 != o32) W.n_flips++;
      const bool open = mode ? o32 : o64;
      if (open) {
        if (C.n_child != 0) stack.push_back(ch);       // opened node: walk on
        else W.leaf_list.push_back(ch);                // opened leaf: particle-particle
      } else {
        W.cell_list.push_back(ch);                     // not opened (leaf or node): multipole (R2)
      }
    }
  }
}

// ---- O6: evaluation (List 3/4 PAPER.md:105-135; R10, R11, R12, R13)
void eval_group(const Oracle& T, int gcell, const WalkOut& W, double eps,
                double* acc, double* pot, int64_t* npc, int64_t* npp) {
  const OCell& G = T.cells[gcell];
  const double eps2 = eps * eps;
  int64_t nbody = 0;
  for (int l : W.leaf_list) nbody += T.cells[l].count;
  for (int64_t t = G.begin; t < G.begin + G.count; t++) {
    const int64_t i = T.perm[t];
    double ax = 0, ay = 0, az = 0, ph = 0;
    for (int cidx : W.cell_list) {   // particle-cell: monopole + quadrupole
      const OCell& C = T.cells[cidx];
      const double rx = T.x[i] - C.X[0], ry = T.y[i] - C.X[1], rz = T.z[i] - C.X[2];
      const double s2 = rx * rx + ry * ry + rz * rz + eps2;
      const double s = std::sqrt(s2);
      const double s3 = s2 * s, s5 = s3 * s2, s7 = s5 * s2;
      if (!T.quadrupole) {             // R22: monopole only
        ax += -C.M * rx / s3; ay += -C.M * ry / s3; az += -C.M * rz / s3;
        ph += -C.M / s;
        continue;
      }
      const double Qrx = C.Q[0] * rx + C.Q[3] * ry + C.Q[4] * rz;
      const double Qry = C.Q[3] * rx + C.Q[1] * ry + C.Q[5] * rz;
      const double Qrz = C.Q[4] * rx + C.Q[5] * ry + C.Q[2] * rz;
      const double rQr = rx * Qrx + ry * Qry + rz * Qrz;
      ax += -C.M * rx / s3 + Qrx / s5 - 2.5 * rQr * rx / s7;
      ay += -C.M * ry / s3 + Qry / s5 - 2.5 * rQr * ry / s7;
      az += -C.M * rz / s3 + Qrz / s5 - 2.5 * rQr * rz / s7;
      ph += -C.M / s - 0.5 * rQr / s5;
    }
    for (int l : W.leaf_list) {      // particle-particle, self excluded
      const OCell& L = T.cells[l];
      for (int64_t u = L.begin; u < L.begin + L.count; u++) {
        const int64_t j = T.perm[u];
        if (j == i) continue;
        const double rx = T.x[i] - T.x[j], ry = T.y[i] - T.y[j], rz = T.z[i] - T.z[j];
        const double r2 = rx * rx + ry * ry + rz * rz;
        const double s2 = r2 + eps2;
        if (s2 == 0.0) continue;     // eps = 0 and coincident: contributes nothing (O6)
        const double s = std::sqrt(s2);
        const double s3 = s2 * s;
        ax += -T.m[j] * rx / s3; ay += -T.m[j] * ry / s3; az += -T.m[j] * rz / s3;
        ph += -T.m[j] / s;
      }
    }
    if (acc) { acc[3 * i + 0] = ax; acc[3 * i + 1] = ay; acc[3 * i + 2] = az; }
    if (pot) pot[i] = ph;
    if (npc) npc[i] = (int64_t)W.cell_list.size();
    if (npp) npp[i] = nbody - 1;
  }
}

}  // namespace

extern "C" {

void* orc_create(int64_t n, const float* pos, const float* mass, int n_leaf, int n_group) {
  if (n < 1 || n_leaf < 1 || n_group < 1) return nullptr;
  Oracle* T = new Oracle();
  T->n = n; T->n_leaf = n_leaf; T->n_group = n_group;
  T->x.resize(n); T->y.resize(n); T->z.resize(n); T->m.resize(n);
  for (int64_t i = 0; i < n; i++) {
    T->x[i] = (double)pos[3 * i]; T->y[i] = (double)pos[3 * i + 1]; T->z[i] = (double)pos[3 * i + 2];
    T->m[i] = (double)mass[i];
  }
  root_cube(*T);
  T->perm.resize(n);
  for (int64_t i = 0; i < n; i++) T->perm[i] = i;
  std::vector<int64_t> tmp(n);
  build_cell(*T, 0, n, 0, -1, tmp);
  find_groups(*T, 0);
  return T;
}

void orc_destroy(void* h) { delete (Oracle*)h; }

// variants (R21, R22); 0 / 1 = the default readings
void orc_set_variant(void* h, int open_rule, int quadrupole) {
  Oracle* T = (Oracle*)h;
  T->open_rule = open_rule ? 1 : 0; T->quadrupole = quadrupole ? 1 : 0;
}

// variant R23: 1 = the group enters the opening test as its tight box
void orc_set_group_box(void* h, int group_box) { ((Oracle*)h)->group_box = group_box ? 1 : 0; }

int64_t orc_n_cells(void* h) { return (int64_t)((Oracle*)h)->cells.size(); }
int64_t orc_n_leaves(void* h) { return ((Oracle*)h)->n_leaves; }
int64_t orc_n_groups(void* h) { return (int64_t)((Oracle*)h)->groups.size(); }
int orc_depth(void* h) { return ((Oracle*)h)->depth; }

void orc_get_root(void* h, double* org, double* side) {
  Oracle* T = (Oracle*)h;
  for (int k = 0; k < 3; k++) org[k] = T->org[k];
  *side = T->side;
}
void orc_get_grid(void* h, int32_t* g) {
  Oracle* T = (Oracle*)h;
  for (int64_t i = 0; i < T->n; i++) { g[3 * i] = T->gx[i]; g[3 * i + 1] = T->gy[i]; g[3 * i + 2] = T->gz[i]; }
}
void orc_get_perm(void* h, int64_t* perm) {
  Oracle* T = (Oracle*)h;
  std::memcpy(perm, T->perm.data(), sizeof(int64_t) * T->n);
}
void orc_get_groups(void* h, int32_t* g) {
  Oracle* T = (Oracle*)h;
  for (size_t i = 0; i < T->groups.size(); i++) g[i] = T->groups[i];
}
// every array may be NULL
void orc_get_cells(void* h, int32_t* level, int32_t* parent, int32_t* child8, int32_t* n_child,
                   int64_t* begin, int64_t* count, double* bmin, double* bmax, double* b, double* hh,
                   double* M, double* X, double* Q) {
  Oracle* T = (Oracle*)h;
  for (size_t c = 0; c < T->cells.size(); c++) {
    const OCell& C = T->cells[c];
    if (level) level[c] = C.level;
    if (parent) parent[c] = C.parent;
    if (child8) for (int o = 0; o < 8; o++) child8[8 * c + o] = C.child[o];
    if (n_child) n_child[c] = C.n_child;
    if (begin) begin[c] = C.begin;
    if (count) count[c] = C.count;
    for (int k = 0; k < 3; k++) {
      if (bmin) bmin[3 * c + k] = C.bmin[k];
      if (bmax) bmax[3 * c + k] = C.bmax[k];
      if (b) b[3 * c + k] = C.b[k];
      if (X) X[3 * c + k] = C.X[k];
    }
    if (hh) hh[c] = C.h;
    if (M) M[c] = C.M;
    if (Q) for (int k = 0; k < 6; k++) Q[6 * c + k] = C.Q[k];
  }
}

// fp32 boundaries used by the shadow test (R20): b32 [n_cells,3], h32 [n_cells]
void orc_get_bnd32(void* h, float* b32, float* h32) {
  Oracle* T = (Oracle*)h;
  for (size_t c = 0; c < T->cells.size(); c++) {
    for (int k = 0; k < 3; k++) b32[3 * c + k] = T->cells[c].b32[k];
    h32[c] = T->cells[c].h32;
  }
}

// R23: fp32 half extents of every cell's tight box about its fp32 centre: e32 [n_cells,3]
void orc_get_ext32(void* h, float* e32) {
  Oracle* T = (Oracle*)h;
  for (size_t c = 0; c < T->cells.size(); c++)
    for (int k = 0; k < 3; k++) e32[3 * c + k] = T->cells[c].e32[k];
}

// Walk one group (index into the group list).  Returns 0, or -1 if a list does not fit.
int orc_walk(void* h, int64_t group, double theta, int mode,
             int32_t* cell_list, int64_t cap_c, int32_t* leaf_list, int64_t cap_l,
             int64_t* n_c, int64_t* n_l, double* min_margin, int64_t* n_flips, int64_t* n_tests) {
  Oracle* T = (Oracle*)h;
  WalkOut W;
  walk_group(*T, T->groups[group], theta, mode, W);
  *n_c = (int64_t)W.cell_list.size(); *n_l = (int64_t)W.leaf_list.size();
  if (min_margin) *min_margin = W.min_margin;
  if (n_flips) *n_flips = W.n_flips;
  if (n_tests) *n_tests = W.n_tests;
  if (*n_c > cap_c || *n_l > cap_l) return -1;
  std::copy(W.cell_list.begin(), W.cell_list.end(), cell_list);
  std::copy(W.leaf_list.begin(), W.leaf_list.end(), leaf_list);
  return 0;
}

// Forces on the particles of the selected groups (sel == NULL: all groups).
// acc [n,3], pot [n], npc [n], npp [n] are indexed by the caller's particle
// index; entries of particles outside the selection are left untouched.
// Per-group outputs (indexed by position in `sel`, or by group if sel == NULL):
// g_min_margin, g_flips, g_tests (each may be NULL).  Returns the number of
// interactions evaluated (sum over particles of n_pc + n_pp).
int64_t orc_forces(void* h, double theta, double eps, int mode,
                   int64_t n_sel, const int64_t* sel,
                   double* acc, double* pot, int64_t* npc, int64_t* npp,
                   double* g_min_margin, int64_t* g_flips, int64_t* g_tests) {
  Oracle* T = (Oracle*)h;
  const int64_t ng = sel ? n_sel : (int64_t)T->groups.size();
  int64_t total = 0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : total)
  for (int64_t s = 0; s < ng; s++) {
    const int64_t g = sel ? sel[s] : s;
    const int gcell = T->groups[g];
    WalkOut W;
    walk_group(*T, gcell, theta, mode, W);
    eval_group(*T, gcell, W, eps, acc, pot, npc, npp);
    int64_t nbody = 0;
    for (int l : W.leaf_list) nbody += T->cells[l].count;
    total += T->cells[gcell].count * ((int64_t)W.cell_list.size() + nbody - 1);
    if (g_min_margin) g_min_margin[s] = W.min_margin;
    if (g_flips) g_flips[s] = W.n_flips;
    if (g_tests) g_tests[s] = W.n_tests;
  }
  return total;
}

// fp64 direct summation (the paper's accuracy reference):
// a_i = sum_{j != i} -m_j r_ij / (r_ij^2 + eps^2)^{3/2},  phi_i = sum_{j != i} -m_j / (r_ij^2 + eps^2)^{1/2}
// targets == NULL: all particles; acc [n_t,3], pot [n_t] indexed by target position.
void orc_direct(int64_t n, const float* pos, const float* mass, double eps,
                int64_t n_t, const int64_t* targets, double* acc, double* pot) {
  const double eps2 = eps * eps;
  const int64_t nt = targets ? n_t : n;
#pragma omp parallel for schedule(static)
  for (int64_t t = 0; t < nt; t++) {
    const int64_t i = targets ? targets[t] : t;
    const double xi = pos[3 * i], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
    double ax = 0, ay = 0, az = 0, ph = 0;
    for (int64_t j = 0; j < n; j++) {
      if (j == i) continue;
      const double rx = xi - (double)pos[3 * j], ry = yi - (double)pos[3 * j + 1], rz = zi - (double)pos[3 * j + 2];
      const double s2 = rx * rx + ry * ry + rz * rz + eps2;
      if (s2 == 0.0) continue;
      const double s = std::sqrt(s2);
      const double w = (double)mass[j] / (s2 * s);
      ax -= w * rx; ay -= w * ry; az -= w * rz;
      ph -= (double)mass[j] / s;
    }
    if (acc) { acc[3 * t] = ax; acc[3 * t + 1] = ay; acc[3 * t + 2] = az; }
    if (pot) pot[t] = ph;
  }
}

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"

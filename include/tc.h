/* ============================================================================
 *  tc.h — C ABI of the B200-native tree-code force calculation
 *  (hot path of arXiv 1005.5384, Gaburov, Bedorf & Portegies Zwart, ICCS 2010).
 *
 *  What the library computes (citations are /root/reference/PAPER.md lines):
 *    - host: octree by recursive cubic subdivision down to N_leaf,
 *      tight bounding boxes -> boundary cubes (Fig. 1), mass, centre
 *      of mass and quadrupole moments per cell, groups,
 *      packed into SoA float4 arrays and moved in ONE bulk copy;
 *    - device (sm_100a): per group, the non-recursive stack walk with the opening
 *      test on cell boundaries (Sec. 2.2, List 2) fused with the
 *      evaluation of the interaction lists as particle-cell (monopole + quadrupole)
 *      and particle-particle softened gravity (Sec. 2.3, Lists 3-4).
 *  The exact formulae (the paper only cites them) are the readings O1-O6 / R1-R18
 *  listed in DESIGN.md section 3.
 *
 *  Conventions: G = 1; every function is thread-compatible per context (one
 *  thread at a time per tc_ctx); no function throws or aborts; all int-returning
 *  functions return TC_OK (0) or a negative TC_E* code and keep a message that
 *  tc_last_error() returns.  There is NO CPU fallback: without a CUDA device
 *  tc_create() returns NULL and tc_forces() cannot be reached.
 * ========================================================================== */
#ifndef TC_H_
#define TC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tc_ctx tc_ctx;

enum {
  TC_OK = 0,
  TC_EINVAL = -1,    /* bad argument (null, out of range, non-finite)            */
  TC_ESTATE = -2,    /* call order: no particles / no tree / host-only context   */
  TC_ECUDA = -3,     /* a CUDA runtime call or kernel failed; see tc_last_error  */
  TC_ENOMEM = -4,    /* host or device allocation failed                         */
  TC_EOVERFLOW = -5  /* a device-side walk stack exceeded its spill capacity     */
};

/* tc_create_ex flags */
#define TC_FLAG_HOST_ONLY 1u /* no device: set_particles/build/get_tree work (host
                                builder tests); tc_forces returns TC_ESTATE.      */

/* Tree / timing statistics, filled by tc_get_stats.  Times follow the paper's
 * split T_host / T_GPU plus the copy.                        */
typedef struct tc_stats {
  int64_t n;              /* particles                                            */
  int64_t n_cells;        /* cells in the tree (nodes + leaves, root included)    */
  int64_t n_leaves;
  int64_t n_groups;
  int32_t depth;          /* deepest level (root = 0)                             */
  int32_t n_leaf;         /* N_leaf of the last tc_build                          */
  int32_t n_group;        /* N_group of the last tc_build                         */
  int32_t reserved;
  int64_t n_pc_total;     /* sum over particles of particle-cell interactions of
                             the last tc_forces                                   */
  int64_t n_pp_total;     /* same, particle-particle (self excluded)              */
  int64_t n_tests_total;  /* opening tests EXECUTED by the last tc_forces: one walk per group; only a group of more
                             than 128 particles (N_group > 128, or a level-21 leaf of coincident particles) is walked once per 128 */
  int64_t n_spills;       /* walk-stack spills to global memory (last tc_forces)  */
  double t_host_ms;       /* last tc_build: host tree + moments + pack            */
  double t_copy_ms;       /* last tc_build: bulk host->device copy (wall)         */
  double t_gpu_ms;        /* last tc_forces: device time of the force kernel(s),
                             CUDA events on the context's stream                  */
  int64_t tree_bytes;     /* bytes of the single bulk H2D copy of tc_build        */
  /* option "two_pass" only (0 otherwise): the paper's kernels timed one by one   */
  double t_walk_count_ms; /* walk pass 1 (count) + scan of the list sizes + list allocation         */
  double t_walk_write_ms; /* walk pass 2 (write the lists to global memory)                         */
  double t_node_ms;       /* body-node evaluation kernel (List 3)                                   */
  double t_leaf_ms;       /* body-leaf evaluation kernel (List 4)                                   */
  int64_t list_bytes;     /* bytes of the global interaction lists                                  */
  int64_t n_opened_total; /* of n_tests_total: tests that OPENED the cell (nodes walked on + leaves sent to the particle-particle
                             list); the others put the cell on a group's cell list.  The paper's walk metric
                             counts 16 bytes per test + 16 per opened cell.                 */
} tc_stats;

/* Select the current CUDA device, create the context and its stream.
 * Returns NULL on failure (no device, out of memory).  Multiple contexts are
 * allowed; there is no global state.                                            */
tc_ctx* tc_create(void);
tc_ctx* tc_create_ex(uint32_t flags);

/* Free everything owned by the context.  NULL is a no-op.                       */
void tc_destroy(tc_ctx* ctx);

/* Particles (the host owns allocation and transfers).
 *   pos  : n x 3 fp32, row-major (x,y,z)        mass : n fp32
 * HOST or DEVICE pointers (resolved with cudaPointerGetAttributes).  The data is
 * COPIED; the caller may free or overwrite it on return.  Invalidates the tree.
 * Errors: TC_EINVAL (null, n < 1, n > 2^31-1, non-finite position, negative or
 * non-finite mass).                                                             */
int tc_set_particles(tc_ctx* ctx, const float* pos, const float* mass, int64_t n);

/* Host octree: root cube, recursive 8-way split until a cell
 * holds <= n_leaf particles (or level 21), tight bounding boxes, boundary cubes,
 * fp64 moments rounded to fp32, groups (N_group from tc_set_option, default 128),
 * SoA float4 packing, one bulk host->device copy.
 * Errors: TC_ESTATE (no particles), TC_EINVAL (n_leaf < 1), TC_ENOMEM, TC_ECUDA. */
int tc_build(tc_ctx* ctx, int n_leaf);

/* The hot path: for every group walk the tree with opening
 * angle theta, evaluate particle-cell (monopole+quadrupole) and particle-particle
 * Plummer-softened interactions, write accelerations and potentials.
 *   acc : n x 3 fp32 (ax,ay,az), pot : n fp32 or NULL — CALLER-ALLOCATED, host or
 *   device, in the CALLER's particle order.
 * Host pointers: synchronous on return.  Device pointers: stream-ordered on the
 * context's stream (tc_set_stream); errors of the kernel surface at tc_sync().
 * eps < 1e-10 is taken as eps = 0 (coincident pairs then contribute nothing): m / eps^3 of the self pair must stay
 * finite in fp32; theta > 1e18 (theta^2 overflows fp32) is refused.  The sums run over j != i: the pair (i, i) is excluded
 * by index where it would occur (the rounds that stage the group's own particles), so no -m_i/eps term enters phi_i.
 * Errors: TC_ESTATE (tree not built / host-only / shard_count > 1: use tc_forces_shard), TC_EINVAL
 * (theta < 0, theta > 1e18, eps < 0, non-finite, acc NULL), TC_ECUDA, TC_EOVERFLOW.                 */
int tc_forces(tc_ctx* ctx, float theta, float eps, float* acc, float* pot);

/* Options (double-valued).  Keys:
 *   "n_group"     N_group >= 1; takes effect at the next tc_build
 *   "device_build" 0 (default: host build, as in the paper) or 1: tc_build runs the same
 *                 construction on the GPU (tc_build_gpu.cu) and writes the packed tree in device memory —
 *                 no bulk H2D; t_host_ms of tc_stats is then the wall time of the device build, t_copy_ms 0.
 *                 Cells, boundary cubes, groups and counts are identical to the host build's.
 *   "open_rule"   0 (default: minimum distance between the group's and the cell's boundary cubes, R1)
 *                 or 1: distance from the group's cube to the cell's centre of mass (variant R21): about 45 %
 *                 fewer interactions and about twice the error at equal theta.
 *   "group_box"   0 (default: the group enters the opening test as its boundary cube, R9) or 1: as its
 *                 TIGHT box with per-axis half extents (variant R23): d_k = max(0, |b_c,k - b_g,k| - h_c - e_g,k);
 *                 still conservative, about 1 % fewer interactions.  Combines with "open_rule".
 *   "quadrupole"  1 (default: monopole + quadrupole) or 0: monopole-only cells (variant R22, the expansion of
 *                 the Hamada et al. code the paper compares with).
 *   "kernel_config" launch configuration of the fused kernel: 0 (default) = chosen by the mean number of particles per
 *                 group, 1 = sparse (16 warps per SM, for small groups), 2 = dense (12 warps per SM with larger
 *                 shared-memory chunks and more registers, for large groups).  Same arithmetic, same lists: results differ
 *                 by summation order only (the chunk boundaries move).  1 and 2 are honoured with either "stack_smem";
 *                 0 picks the sparse build whenever "stack_smem" is 64.  Ignored while "two_pass" is 1 (that pipeline's
 *                 kernels exist in one configuration).
 *   "shard_count", "shard_rank"   ONE force evaluation over k GPUs (tc_forces_shard below): this context is
 *                 rank shard_rank of shard_count.  Default 1 / 0.
 *   "two_pass"    0 (default: the fused kernel) or 1: the paper-literal pipeline —
 *                 walk-count kernel, scan of the list sizes, walk-write kernel (lists in global memory),
 *                 body-node kernel, body-leaf kernel; same lists, same counts, same results up to
 *                 summation order; an A/B against the fused design, timed per kernel in tc_stats.
 *   "walk_only"   measurement aid of bench.py, documented in include/tc_bench.h
 *   "stack_smem"  walk-stack entries kept in shared memory per warp before
 *                 spilling to global memory: 256 (default) or 64 (test of the
 *                 spill path)
 * Unknown key or bad value -> TC_EINVAL.                                        */
int tc_set_option(tc_ctx* ctx, const char* key, double value);

/* Per-particle interaction counts of the last tc_forces, caller's order:
 * n_pc = |cell list of the particle's group|, n_pp = bodies of the opened leaves
 * minus the particle itself.  HOST pointers, n int32 each; either may be NULL.
 * Synchronises the context's stream.                                            */
int tc_get_counts(tc_ctx* ctx, int32_t* n_pc, int32_t* n_pp);

int tc_get_stats(tc_ctx* ctx, tc_stats* out);

/* Use the caller's CUDA stream (a cudaStream_t passed as void*; NULL = the
 * context's own stream).  The context never destroys a caller's stream.
 * The own stream is created cudaStreamNonBlocking: it is NOT ordered with the
 * legacy default stream.  The raw handle of the legacy default stream is 0 = NULL,
 * so to queue the context's work on it pass cudaStreamLegacy ((cudaStream_t)0x1),
 * or cudaStreamPerThread for the per-thread default stream.                      */
int tc_set_stream(tc_ctx* ctx, void* cuda_stream);

/* Block until all work queued by this context has finished; returns TC_ECUDA /
 * TC_EOVERFLOW if the last stream-ordered tc_forces failed.                      */
int tc_sync(tc_ctx* ctx);

/* Message of the last error of this context ("" if none).  Owned by the context.
 * ctx == NULL returns the message of the last failed tc_create or tc_direct_static
 * on the calling thread.                                                          */
const char* tc_last_error(const tc_ctx* ctx);

/* Inspection of the packed host tree of the last tc_build (tests of the host
 * builder; no device needed).  Every pointer is a HOST array or NULL:
 *   perm      [n]          original index of the i-th particle in tree (Morton) order
 *   cell_bnd  [n_cells,4]  boundary cube (bx,by,bz,h), h >= 0            (Fig. 1)
 *   cell_xm   [n_cells,4]  centre of mass and mass (X,Y,Z,M)
 *   cell_q    [n_cells,6]  traceless quadrupole xx,yy,zz,xy,xz,yz
 *   cell_link [n_cells,4]  first_child, n_child (0 = leaf), first_body, n_body
 *   groups    [n_groups]   cell id of every group, Morton order
 * Sizes come from tc_get_stats.                                                 */
int tc_get_tree(tc_ctx* ctx, int32_t* perm, float* cell_bnd, float* cell_xm, float* cell_q,
                int32_t* cell_link, int32_t* groups);

/* `steps` kick-drift-kick leapfrog steps entirely on the device (BASELINE.json config 5;
 * the paper leaves time integration to the host).  Per step, in fp32:
 *     v += a dt/2 ;  x += v dt ;  tc_set_particles(x, mass) ; tc_build(n_leaf) ; a = tc_forces(theta, eps) ;  v += a dt/2
 *   pos, vel, acc [n,3], mass, pot [n] (pot may be NULL): DEVICE arrays owned by the caller, pos / vel / acc / pot
 *   16-byte aligned; pos, vel, acc, pot are updated in place and hold x, v, a(x), phi(x) of the last step on return.
 *   have_acc != 0: acc already holds a(pos) (e.g. from a previous call) and the initial force evaluation is
 *   skipped; with have_acc == 0 (or steps == 0) the forces at the start are evaluated first.
 * The tree is rebuilt every step by the context's builder (option "device_build": nothing leaves the device;
 * default host build: positions go to the host and the packed tree comes back each step, as in the paper).
 * Stream-ordered like tc_forces with device pointers: call tc_sync before reading the arrays elsewhere.
 * tc_get_stats / tc_get_counts then describe the LAST force evaluation.
 * Errors: TC_EINVAL (null / host pointer / misaligned / n < 1 / steps < 0 / non-finite dt, theta, eps; a particle
 * that left the finite range is reported by the tc_set_particles of that step), TC_ESTATE (host-only context). */
int tc_leapfrog(tc_ctx* ctx, float* pos, float* vel, const float* mass, int64_t n, float dt, int steps, int n_leaf,
                float theta, float eps, float* acc, float* pot, int have_acc);

/* Half extents of every group's TIGHT box about the centre of its boundary cube (variant R23, option
 * "group_box"), fp32, rounded up so that the box contains every particle of the group:
 *   half_ext [n_groups,3]  HOST array, groups in Morton order (as `groups` of tc_get_tree).
 * TC_ESTATE without a built tree, TC_EINVAL for NULL.                                                     */
int tc_get_group_boxes(tc_ctx* ctx, float* half_ext);

/* Direct summation over ALL particles of the last tc_set_particles — the paper's accuracy reference
 * (forces "by direct summation ... with double precision emulation"):
 *   a_i = sum_{j != i} m_j (x_j - x_i) / s^3,  phi_i = -sum_{j != i} m_j / s,  s^2 = |x_j - x_i|^2 + eps^2
 * for the n_targets particles listed in `targets` (HOST int64 indices in the caller's order; NULL = all
 * n particles, n_targets ignored).  Interactions are evaluated in packed FP32 with a Newton-refined
 * rsqrt, partial sums of 256 sources are accumulated in fp64.  No tree is needed (tc_build not required).
 *   acc : n_targets x 3 fp64, pot : n_targets fp64 or NULL — CALLER-ALLOCATED, host or device (both the
 *   same kind); host pointers: synchronous on return; device pointers: stream-ordered.
 * eps == 0: coincident pairs contribute nothing.
 * Errors: TC_ESTATE (no particles / host-only), TC_EINVAL (null acc, bad eps, target out of range),
 * TC_ENOMEM, TC_ECUDA.                                                                              */
int tc_direct(tc_ctx* ctx, float eps, const int64_t* targets, int64_t n_targets, double* acc, double* pot);

/* ---- Direct summation WITHOUT any allocation -----------------------------------------------------------------
 * For whom: code that is not allowed to obtain device memory at the moment it needs forces.  Examples: a plugin
 * running inside a host application whose memory pool owns the whole GPU and hands out fixed buffers (a cudaMalloc
 * from a guest library would fail or fragment the pool); a real-time or in-situ analysis step that may not take
 * the driver's allocation lock, which can stall for milliseconds and synchronises the device on cudaFree; a
 * process that has already filled the 180 GB with its own data.  Every other entry point of this library creates a
 * context (tc_create) and grows device buffers on demand; this one does neither.
 *
 * What it computes: exactly tc_direct (same kernels, same arithmetic):
 *   a_i = sum_{j != i} m_j (x_j - x_i) / s^3,  phi_i = -sum_{j != i} m_j / s,  s^2 = |x_j - x_i|^2 + eps^2
 * over the n particles given in THIS call, for the targets listed.
 *   pos [n,3] fp32, mass [n] fp32                INPUTS, device, caller's order, not modified
 *   targets [n_targets] int64 or NULL            device; NULL = all n particles (n_targets ignored).  Indices must lie
 *                                                in [0, n): they are NOT checked (checking would need a read-back);
 *                                                a negative index leaves its output row at zero
 *   acc [n_targets,3] fp64, pot [n_targets] fp64 or NULL     OUTPUTS, device, owned by the caller; zeroed, then written
 *   cuda_stream                                  a cudaStream_t as void*; NULL = the legacy default stream.  All work is
 *                                                queued on it and the call returns without synchronising: order your
 *                                                reads of acc / pot after it on the same stream (or synchronise it).
 * Inputs are not validated beyond the sizes (a NaN position gives NaN results).
 *
 * Where the working memory comes from: the kernel reads its sources as one packed (x, y, z, m) array.  Here that
 * array is a fixed block of TC_DIRECT_STATIC_MAX_N x 16 bytes = 4 MiB inside the library image; EVERY GPU that loads
 * libtc_b200.so holds these 4 MiB from the first use of the library on that GPU until the process exits, whether
 * or not this function is ever called.  n and n_targets beyond TC_DIRECT_STATIC_MAX_N are refused with TC_EINVAL
 * and a message naming the limit (use tc_direct then).  The function itself calls no cudaMalloc, cudaFree, or any
 * library routine that allocates device memory.
 *
 * First call on each device: it looks up the block's address on the current device (cudaGetSymbolAddress) and the
 * SM count, once, under a lock; later calls only launch.  Make that first call during set-up, outside any CUDA
 * stream capture (the look-up is not a stream operation and may initialise the module).
 *
 * Sharing: there is ONE block per GPU, shared by every caller in the process, and it keeps what the last call put
 * there.  Nothing in it has to start at zero (each call rewrites entries 0 .. n-1 before reading them and reads no
 * others), so consecutive calls on one stream are independent.  Two calls that can run on the GPU at the same time
 * — different streams, or different host threads with their own streams — overwrite each other's sources: that is
 * a data race with wrong results and no error.  Serialise them (one stream, or an event between them).
 *
 * Errors: TC_EINVAL (null pos / mass / acc, n or n_targets < 1 or above the limit, eps negative or non-finite,
 * a host pointer), TC_ECUDA (no device, not sm_100, symbol look-up or launch failed).  The message is returned by
 * tc_last_error(NULL) on the calling thread.                                                                       */
#define TC_DIRECT_STATIC_MAX_N 262144
int tc_direct_static(const float* pos, const float* mass, int64_t n, float eps, const int64_t* targets,
                     int64_t n_targets, double* acc, double* pot, void* cuda_stream);

/* ---- ONE force evaluation over k GPUs ------------------------------------
 * Groups are independent given the read-only tree (one walk per group, nothing is exchanged between
 * groups), so the path shards without any collective inside the walk or the evaluation.  One context per GPU, each
 * with the SAME particles, options and tree, and options "shard_count" = k, "shard_rank" = r.  Rank r evaluates the
 * groups at positions r, r + k, ... of the cost-ordered schedule (neighbours in the schedule cost the same: balanced)
 * and writes ONLY its own particles, compactly: one row (ax, ay, az, phi) per particle, its groups in schedule order,
 * particles in tree order inside a group.  The caller all-gathers the rows of all ranks (16 bytes per particle in
 * total — the one exchange of the path; NCCL all-gather) and tc_shard_scatter puts them in the caller's particle order.
 *
 * tc_shard_size:    *n_slots = rows every rank contributes = max over ranks of the particles a rank evaluates
 *                   (the same number on every rank; rows beyond a rank's own count are never written).
 * tc_forces_shard:  A1-A6 for this rank's groups.  out4 [n_slots,4] fp32 and cnt2 [n_slots,2] int32 ((n_pc, n_pp) per
 *                   row) or NULL: DEVICE buffers of the caller, stream-ordered.  theta, eps as tc_forces.  The totals
 *                   in tc_stats are those of the shard; tc_get_counts is not valid after a shard (TC_ESTATE).
 * tc_shard_scatter: gathered4 [k, n_slots, 4] (rank-major, as an all-gather delivers it) and gathered_cnt2
 *                   [k, n_slots, 2] or NULL -> acc [n,3], pot [n] or NULL, n_pc / n_pp [n] or NULL in the CALLER's
 *                   particle order.  All DEVICE buffers, stream-ordered.  With k = 1 the pair
 *                   tc_forces_shard + tc_shard_scatter gives bit for bit the result of tc_forces; for k > 1 too:
 *                   every particle is computed by exactly one rank with the arithmetic of the single-GPU launch.
 * Errors: TC_ESTATE (no tree / host-only), TC_EINVAL (null or host pointer, shard_rank >= shard_count, two_pass),
 * TC_ENOMEM, TC_ECUDA, TC_EOVERFLOW.                                                                              */
int tc_shard_size(tc_ctx* ctx, int64_t* n_slots);
int tc_forces_shard(tc_ctx* ctx, float theta, float eps, float* out4, int32_t* cnt2);
int tc_shard_scatter(tc_ctx* ctx, const float* gathered4, const int32_t* gathered_cnt2, float* acc, float* pot,
                     int32_t* n_pc, int32_t* n_pp);

#ifdef __cplusplus
}
#endif
#endif /* TC_H_ */

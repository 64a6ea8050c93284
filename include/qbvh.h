/* qbvh.h — C-ABI of libqbvh.so: quantized-BVH Verlet neighbor lists on NVIDIA B200 (sm_100a).
 *
 * Method: Howard et al., "Quantized bounding volume hierarchies for neighbor search in molecular
 * simulations on graphics processing units", arXiv:1901.08088.  Citations are lines of
 * /root/reference/PAPER.md ("PAPER.md:<line>") plus the section / equation / algorithm they fall in.
 *
 * The library solves the problem stated in PAPER.md:31 (§1): "determine the subset of particles
 * within a distance r_c of a given particle ... saved to construct a Verlet (neighbor) list", under
 * periodic boundaries with lattice-vector images, fp32 particle data
 * (PAPER.md:154, 176).  Every step runs in CUDA kernels; there is no CPU fallback.
 *
 * Conventions
 *   - All functions return int (or int64 where noted): >= 0 success, < 0 one of QBVH_ERR_*.
 *     No exceptions, no aborts, no printing.
 *   - "DEVICE" pointers are CUDA device pointers valid on the current device; "HOST" pointers are
 *     ordinary host memory.  The library never allocates device memory: the caller supplies one
 *     workspace (qbvh_set_workspace) that holds the tree and all scratch.
 *   - One process-global context: the last built tree.  qbvh_neighbors may be called any number of
 *     times per build (different r_list, larger capacity on retry).  Not thread-safe.
 *   - All work is enqueued on the stream given to qbvh_set_stream (default: stream 0).
 *     qbvh_build is fully asynchronous.  qbvh_neighbors synchronises that stream once, to read
 *     back 8 bytes (max count, error flags).
 *   - Determinism: the same inputs give a bit-identical node array and identical rows as sets;
 *     the order of entries within a row is unspecified (sorted build => deterministic).
 */
#ifndef QBVH_H
#define QBVH_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define QBVH_OK 0
#define QBVH_ERR_INVALID_ARG (-1)      /* NULL pointer, N < 0, N >= 2^30, max_neigh < 0, bad box, bad option      */
#define QBVH_ERR_NOT_BUILT (-2)        /* qbvh_neighbors / export before a successful qbvh_build                   */
#define QBVH_ERR_WORKSPACE (-3)        /* workspace missing, misaligned (256 B) or smaller than qbvh_workspace_bytes */
#define QBVH_ERR_CUTOFF_TOO_LARGE (-4) /* some padded r_ij >= L_d/2: a pair could be seen through two images       */
#define QBVH_ERR_TYPE_RANGE (-5)       /* a type id outside [0, T) was seen by the build (reported by qbvh_neighbors) */
#define QBVH_ERR_CUDA (-6)             /* a CUDA runtime call failed; text via qbvh_error_string(QBVH_ERR_CUDA)    */
#define QBVH_ERR_INTERNAL (-7)         /* an internal bound was violated (the traversal's work list); the
                                          lists of that call are invalid.  Never seen; reported instead of corrupting. */
#define QBVH_ERR_NOALLOC_LIMIT (-8)    /* qbvh_morton_keys_noalloc: N is larger than QBVH_NOALLOC_MAX_N, the size its built-in
                                          scratch array was compiled for; use the workspace path (qbvh_build) instead   */

#define QBVH_MAX_TYPES 4 /* type id lives in bits 30-31 of the 32-bit sort key above the 30-bit Morton code */

/* ---- set-up -------------------------------------------------------------------------------- */

/* Stream for all subsequent work.  cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream). */
int qbvh_set_stream(void *cuda_stream);

/* Number of particle types T in [1, QBVH_MAX_TYPES] for subsequent builds (default 1).  One BVH per type,
 * queried across types with per-pair cutoffs (reading R14 in DESIGN.md). */
int qbvh_set_num_types(int32_t T);

/* Bytes of DEVICE workspace needed for N particles and T types (tree + scratch), a multiple of 256. */
int64_t qbvh_workspace_bytes(int64_t N, int32_t T);

/* Caller-owned DEVICE workspace, 256-byte aligned; must stay valid until the next qbvh_set_workspace and its
 * CONTENTS must not be modified by the caller between qbvh_build calls: rebuilding on the same workspace with the
 * same N does not clear the tree builder's meeting slots, it tells stale ones apart by a per-build tag (DESIGN.md
 * §3.6), so foreign data written there could be mistaken for a sibling.  Call qbvh_set_workspace again (same
 * pointer is fine) after using the memory for anything else: that clears the slots at the next build.
 * Invalidates the current tree.  qbvh_set_workspace(NULL, 0) detaches the library from the memory. */
int qbvh_set_workspace(void *dev_ptr, int64_t bytes);

/* Options (all take effect at the next qbvh_build unless noted). */
#define QBVH_OPT_LEAF_COLLAPSE 1 /* k in [1,32]: the build may collapse a subtree of <= k consecutive Z-order particles
                                    into one range leaf, whose particles the traversal distance-checks directly
                                    ("subtree collapse"); which subtrees: qbvh_set_collapse_hint.
                                    k = 1 is exactly the paper's one-particle-per-leaf tree. Default 32.           */
#define QBVH_OPT_STATS 2         /* 0/1: qbvh_neighbors runs the instrumented traversal and fills qbvh_get_stats
                                    (takes effect immediately; slower — never use when timing). Default 0.
                                    The census writes a row per particle, so qbvh_neighbors_range refuses to run
                                    with it (QBVH_ERR_INVALID_ARG); under qbvh_neighbors_f64 its `neighbors` field
                                    counts by the widened fp32 cutoff (r + 8 ulp32(M)), not by the fp64 predicate.  */
#define QBVH_OPT_VARIANT 3       /* which traversal kernel qbvh_neighbors launches: 0 = Algorithm 1 as written, one
                                    thread per particle; 1 (default) = one warp per query group.
                                    Both produce identical lists.                                                 */
#define QBVH_OPT_DEBUG_BUILD_TAG 4 /* testing only: v in [1, 2^18): the next qbvh_build on this workspace uses meeting-
                                    slot tag v (forward jumps only) — lets a test reach the 18-bit wrap.           */
#define QBVH_OPT_DEBUG_SCAN_SPIN 5  /* testing only: SM clock cycles a block of the build's 128-tile cell scan (cell grid
                                    level 6, or level 5 with >= 3 types) waits for the other blocks before it sums the
                                    counters in front of its tile itself (default 2^18, about 130 us; 0: never wait).
                                    Either way the result is the same; the bound only matters on a device too busy to
                                    hold all 128 blocks at once, where an unbounded wait could hang.               */
#define QBVH_OPT_GROUP_MAX 6        /* v in [1,32], default 32: the largest query group (particles one warp of the production
                                    traversal searches for together) the next build emits.  Smaller groups have
                                    tighter search boxes (fewer candidates per member) but fill fewer lanes of their warp.
                                    The lists do not depend on it.                                                 */
#define QBVH_OPT_CELL_LEVEL 7       /* 0 (default): the build picks its Morton-cell grid (2^level cells per axis over the BOX)
                                    from N alone, which assumes the particles fill the box; 2..6: use this level — for a
                                    droplet or slab that occupies a small part of the box a finer grid keeps the cells small
                                    (profiles/r03_configs.md).  Lowered if T * 8^level would exceed 2^18.  The tree and the
                                    lists do not depend on it.                                                     */
int qbvh_set_option(int32_t key, int32_t value);

/* Hint for the build-side subtree collapse ("collapse subtrees according to an appropriate heuristic",
 * PAPER.md:230): r_hint[b] = the query radius tree b (particle type b) will be searched with, e.g. max_a r_list[a][b].
 *   r_hint HOST  n <= QBVH_MAX_TYPES floats; n = 0 or r_hint[b] <= 0: no hint for that tree.
 * With a hint, two sibling range leaves are merged into one range leaf (of at most QBVH_OPT_LEAF_COLLAPSE particles)
 * only if that lowers the expected cost of a query — an integer surface-area-like model on the quantized boxes
 * swollen by the radius.  Without one, every subtree of at most QBVH_OPT_LEAF_COLLAPSE particles
 * collapses.  Collapsed subtrees' descendants are never written.  Takes effect at the next qbvh_build. */
int qbvh_set_collapse_hint(const float *r_hint, int32_t n);
int qbvh_get_option(int32_t key);

/* ---- the hot path --------------------------------------------------------------------------- */

/* Build the quantized linear BVH(s).  PAPER.md:61-67 (§2.1: Morton codes in the box divided into 2^10-1 bins
 * per axis, sort along the Z-order curve, Karras hierarchy, bounding boxes fit by walking up from the leaves),
 * PAPER.md:69,75 (left child + rope per node for stackless traversal), PAPER.md:89 (§2.2: bounds snapped
 * outward onto 2^10-1 bins per axis of the ROOT-node box, 3 x 10 bits per bound word, 16-byte node).
 *   pos   DEVICE  N x 3 fp32 row-major xyz; expected wrapped into [lo_d, lo_d + L_d).  Not referenced after
 *                 the call's kernels have run (the tree keeps its own Z-ordered copy in the workspace).
 *   type  DEVICE  N int32 in [0, T), or NULL => all particles type 0.
 *   N     0 <= N < 2^30.  N = 0 is a valid (empty) build.
 *   box   HOST    6 floats {lo_x, lo_y, lo_z, L_x, L_y, L_z}: orthorhombic cell, periodic in x, y, z; L_d > 0 finite.
 * Positions outside the box never corrupt the tree (Morton bins clamp, boxes are fit to actual coordinates)
 * but periodic images are then wrong. */
int qbvh_build(const float *pos, const int32_t *type, int64_t N, const float *box);

/* Traverse the tree(s) once per particle (Algorithm 1: bitset of the 27 periodic images whose
 * search sphere overlaps the root, stackless left/rope walk, sphere-AABB test of eq. 2 PAPER.md:144-146 on the
 * decompressed box) and emit the exact Verlet list: a leaf hit is kept iff the canonical fp32 minimum-image
 * predicate d2 <= r_ij^2 holds and j != i.
 *   r_list_ij HOST    T x T fp32 row-major, symmetric; r_ij <= 0 => that pair of types is skipped.
 *   nlist     DEVICE  N x max_neigh int32 row-major; row i = neighbors of ORIGINAL particle i as ORIGINAL
 *                     indices, in unspecified order; entries at positions >= n_neigh[i] are unspecified.
 *   n_neigh   DEVICE  N int32; the true number of neighbors of particle i (may exceed max_neigh).
 *   max_neigh row capacity, >= 0.
 * Returns M = max_i n_neigh[i] (>= 0).  M <= max_neigh: all rows complete.  M > max_neigh: OVERFLOW — rows with
 * n_neigh[i] > max_neigh hold max_neigh true neighbors; re-allocate with capacity >= M and call again. */
int qbvh_neighbors(const float *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh);

/* The same call in two halves, for callers that keep the stream busy (an MD step enqueues its force kernels behind
 * the list) and for timing the device work without a host round trip inside it:
 *   qbvh_neighbors_enqueue  checks its arguments, enqueues the traversal on the stream and returns QBVH_OK (or < 0)
 *                           without waiting; arguments as for qbvh_neighbors (nlist, n_neigh stay in use until the
 *                           result has been taken);
 *   qbvh_neighbors_result   synchronises the stream and returns what qbvh_neighbors would have returned for the last
 *                           enqueue (M >= 0, or QBVH_ERR_TYPE_RANGE / QBVH_ERR_INTERNAL / QBVH_ERR_CUDA);
 *                           QBVH_ERR_NOT_BUILT if nothing was enqueued since the last result, or if another
 *                           neighbor call (or a build) came in between: those overwrite the result words.
 * qbvh_neighbors is exactly enqueue followed by result. */
int qbvh_neighbors_enqueue(const float *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh);
int qbvh_neighbors_result(void);
/* The enqueue halves of qbvh_neighbors_f64 and qbvh_neighbors_range (declared below; same arguments, same
 * qbvh_neighbors_result afterwards). */
int qbvh_neighbors_f64_enqueue(const double *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh);
int qbvh_neighbors_range_enqueue(const float *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh, int64_t first, int64_t count);

/* Query sharding ("straightforwardly generalized to execute on multiple GPUs"): the
 * same traversal for the particles at sorted (Z-order) positions [first, first + count) only.  Row k of nlist and
 * n_neigh[k] belong to the particle at sorted position first + k, whose original index is QBVH_EXPORT_PERM[first + k];
 * entries are ORIGINAL indices as always.  nlist: DEVICE count x max_neigh; n_neigh: DEVICE count.  Returns the
 * maximum count over the range.  Needs QBVH_OPT_VARIANT = 1 and QBVH_OPT_STATS = 0 (else QBVH_ERR_INVALID_ARG).  Every GPU of a sharded run holds all positions (one all-gather), builds the same
 * tree and calls this for its own slice (paper_1901_08088_b200/sharded.py). */
int qbvh_neighbors_range(const float *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh, int64_t first, int64_t count);

/* ---- double-precision particle data -----------------------------
 * The tree stays what it is — fp32 frames, 10-bit quantized boxes, 16-byte nodes, built from the positions rounded to
 * fp32 — "the sphere radius is padded to account for uncertainty from loss of precision when the particle data is
 * double precision", and the exact leaf test is the fp64 minimum-image predicate:
 *   D_d = p_j[d] - p_i[d], wrapped once by L_d;  d2 = fma(Dz,Dz, fma(Dy,Dy, Dx Dx));  neighbor <=> d2 <= r_ij^2  (fp64)
 * A pair is first judged in fp32 on the rounded positions with the cutoff widened / narrowed by 8 ulp32(M)
 * (M = max_d(|lo_d| + 2 L_d)); only pairs inside that band (about one in two thousand) are decided in fp64.
 *   pos   DEVICE  N x 3 fp64 row-major, wrapped into [lo_d, lo_d + L_d).   box  HOST 6 doubles {lo_xyz, L_xyz}.
 *   r_list_ij HOST T x T fp64.   nlist / n_neigh / max_neigh / return value: as for qbvh_neighbors.
 * qbvh_neighbors_f64 requires the last build to be qbvh_build_f64 (and qbvh_neighbors a qbvh_build): otherwise
 * QBVH_ERR_INVALID_ARG.  QBVH_OPT_VARIANT must be 1. */
int qbvh_build_f64(const double *pos, const int32_t *type, int64_t N, const double *box);
int qbvh_neighbors_f64(const double *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh);

/* The paper's own operating mode ("the object in the leaf node is processed as a neighbor" without a
 * distance check, positions are not loaded; the benchmarks only count): Algorithm 1 as printed, one
 * thread per particle in Z-order, accepting every particle whose (collapsed) leaf box overlaps the padded search
 * sphere in some image.  With QBVH_OPT_LEAF_COLLAPSE = 1 at build time this is exactly the paper's kernel.
 *   r_list_ij HOST    T x T fp32 as for qbvh_neighbors.
 *   n_overlap DEVICE  N int32; for ORIGINAL particle i the number of accepted particles j != i (true neighbors plus
 *                     the false positives of the quantized leaf boxes).
 * Returns max_i n_overlap[i] (>= 0), or < 0. */
int qbvh_count_overlaps(const float *r_list_ij, int32_t *n_overlap);

/* ---- the same two calls with HOST buffers (end-to-end path: copies are part of the call) ------------------ */

/* Bytes of DEVICE staging the *_host calls need for N particles with row capacity max_neigh. */
int64_t qbvh_staging_bytes(int64_t N, int32_t max_neigh);
int qbvh_set_staging(void *dev_ptr, int64_t bytes);
/* pos, type: HOST (pinned memory makes the copies asynchronous).  Otherwise as qbvh_build. */
int qbvh_build_host(const float *pos, const int32_t *type, int64_t N, const float *box);
/* nlist, n_neigh: HOST (N x max_neigh and N int32).  n_neigh is copied back whole.  Of row i the first
 * min(n_neigh[i], max_neigh) entries are valid afterwards, as for qbvh_neighbors; what lies beyond them is
 * unspecified (either untouched or overwritten):
 *   - nlist in pinned (page-locked, device-mapped) memory, 16-byte aligned, max_neigh % 4 == 0: the rows are written
 *     by the SMs straight into the host buffer, the valid entries of each row rounded up to 16 bytes;
 *   - otherwise (pageable memory, odd capacities): the copy engine moves the first min(M, max_neigh) columns of
 *     every row (M = the return value).
 * Otherwise as qbvh_neighbors. */
int qbvh_neighbors_host(const float *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh);
/* Bytes the last qbvh_neighbors_host call copied from the device. */
int64_t qbvh_last_d2h_bytes(void);

/* ---- for callers that cannot allocate device memory ------------------------------------------------------------
 * Every call above needs a workspace the caller got from cudaMalloc (or from an allocator built on it).  Some callers
 * have no such source: a plugin or callback that runs inside another GPU program and is only handed that program's
 * buffers; code under a framework whose memory pool already owns all of the HBM, where a plain cudaMalloc fails; a
 * latency-critical loop where cudaMalloc / cudaFree are banned because they synchronise the device.  For them, ONE
 * entry point that allocates nothing, anywhere: step a1 of the path — the Morton keys of all particles (PAPER.md:61,
 * §2.1: box divided into 2^10-1 bins per axis, bits interleaved along the Z-order curve) and the root box of each
 * type's tree with its quantization step (§2.2) — e.g. to re-order particle arrays along the Z-curve or
 * to quantize against the same frame as the tree.  Its working memory (one 96-byte record per block of 1024 particles,
 * for the two-stage min/max reduction) is a fixed array compiled into the library: 393,472 bytes of device memory on
 * every GPU that loads libqbvh.so, held until the process exits.  Hence:
 *   - N <= QBVH_NOALLOC_MAX_N, otherwise QBVH_ERR_NOALLOC_LIMIT and nothing is enqueued;
 *   - all calls (from any thread, on any stream) share that one array per GPU and the call starts by clearing the part
 *     of it that must be zero: two calls whose device work can overlap — different streams without an ordering
 *     between them — race on it and give wrong frames.  Calls on one stream, or ordered by events, are fine;
 *   - the first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device
 *     current, which may also make the runtime load the module): make that first call outside any stream capture.
 * The call uses none of the library's global state (no workspace, no qbvh_set_stream, no tree) and leaves it alone.
 * It calls no cudaMalloc, cudaFree, cudaHostAlloc or other allocating routine; it enqueues one memset of 256 bytes and
 * one kernel on `cuda_stream` and returns without waiting.
 *   pos     DEVICE  N x 3 fp32 row-major, as for qbvh_build.      type  DEVICE N int32 in [0, T), or NULL (all type 0).
 *   box     HOST    6 floats {lo_xyz, L_xyz}, as for qbvh_build.   T     number of types, 1..QBVH_MAX_TYPES.
 *   keys    DEVICE  N uint32 out: type << 30 | 30-bit Morton code of particle i — the multiset of
 *                   QBVH_EXPORT_KEYS_SORTED, in input order.  An out-of-range type is keyed as type 0 (as qbvh_build).
 *   frames  DEVICE  4 x 12 floats out: per type {lo_xyz, hi_xyz, delta_xyz, 0, 0, 0}, bitwise what QBVH_EXPORT_FRAMES
 *                   shows after qbvh_build on the same input; all zero for a type without particles.
 *   status  DEVICE  1 int32 out: bit 0 set iff some type id was outside [0, T).
 *   cuda_stream     a cudaStream_t (NULL: the default stream).
 * Returns QBVH_OK, QBVH_ERR_INVALID_ARG, QBVH_ERR_NOALLOC_LIMIT or QBVH_ERR_CUDA.  N = 0 is valid (frames all zero). */
#define QBVH_NOALLOC_MAX_N 4194304 /* 2^22 particles = 4096 block records */
int qbvh_morton_keys_noalloc(const float *pos, const int32_t *type, int64_t N, const float *box, int32_t T,
                             uint32_t *keys, float *frames, int32_t *status, void *cuda_stream);

/* ---- inspection ----------------------------------------------------------------------------- */

/* The padded pruning radius the traversal uses in every sphere/box overlap test (never in the pair predicate):
 *   r_pad = up( up(r (1 + 2^-20)) + 8 ulp32(M) ),  M = max_d(|lo_d| + 2 L_d)      (reading R11)
 * "the sphere radius is padded to account for uncertainty from loss of precision" — here for the
 * fp32 roundings of x_i + v_j, y - x' and the squared sum, so that no true pair is pruned.
 * Pure host arithmetic, needs no device.  box: HOST 6 floats as for qbvh_build.  Returns < 0 on bad arguments. */
float qbvh_padded_radius(float r, const float *box);
/* Its square rounded UP to fp32: the right-hand side d2 <= R2 of the sphere/box test of eq. 2 as the
 * traversal kernels receive it (rounding it any other way could prune a box the padded sphere touches).  Host only. */
float qbvh_padded_radius_sq(float r, const float *box);

typedef struct qbvh_stats {
    uint64_t node_tests;    /* sphere-AABB tests of Algorithm 1 line 12 (root tests of line 4 excluded)           */
    uint64_t leaf_overlaps; /* tests that hit a leaf (one-particle or collapsed range)                             */
    uint64_t dist_checks;   /* exact pair-predicate evaluations                                                    */
    uint64_t neighbors;     /* accepted pairs (= sum of n_neigh)                                                   */
    uint64_t images;        /* set bits of the image bitset, Algorithm 1 line 4, summed over particles and trees   */
    /* the five above: census of Algorithm 1 walked once per PARTICLE (the paper's kernel).
       the six below: the production kernel, which walks the tree once per query GROUP. */
    uint64_t groups;            /* query groups traversed                                                          */
    uint64_t group_node_tests;  /* box-box tests of tree nodes against a group's search volume                     */
    uint64_t group_leaf_hits;   /* (collapsed) leaves that passed it                                               */
    uint64_t group_candidates;  /* particles of those leaves within reach of the group box                         */
    uint64_t group_dist_checks; /* exact pair-predicate evaluations (candidates x group members)                   */
    uint64_t group_walk_steps;  /* warp steps of the walk (up to 32 node tests each)                               */
} qbvh_stats;
/* Counters of the last qbvh_neighbors call made with QBVH_OPT_STATS = 1. */
int qbvh_get_stats(qbvh_stats *out);

/* Debug export of build products (for parity tests of steps a1..a6).  Copies min(bytes, available) bytes into
 * `dst` after synchronising the stream; returns the number of bytes available, or < 0.  dst: HOST memory; for the
 * array products (KEYS_SORTED, PERM, NODES, PARENT, FRAMES, SORTED_POS) DEVICE memory works as well (a sharded run
 * keeps the Z-order permutation on the GPU that way). */
#define QBVH_EXPORT_KEYS_SORTED 1 /* uint32 [N]: type << 30 | 30-bit Morton code, ascending                       */
#define QBVH_EXPORT_PERM 2        /* uint32 [N]: original index of the particle at sorted position k              */
#define QBVH_EXPORT_NODES 3       /* int32 [2N-1][4] = {lo, hi, left, rope}; internal node i at i (Karras
                                     numbering), leaf of sorted position k at N-1+k; left >= 0: left child,
                                     left < 0: a (range) leaf, ~first sorted position, the range ends where the
                                     rope's target starts; rope = -1: END.  Only nodes reachable
                                     from the roots are written: descendants of a range leaf do not exist.       */
#define QBVH_EXPORT_PARENT 4      /* int32 [2N-1]: parent node, -1 for roots and unused slots                     */
#define QBVH_EXPORT_FRAMES 5      /* float [4][12]: {lo_xyz, hi_xyz, delta_xyz, 0,0,0} quantization frame per type */
#define QBVH_EXPORT_SEGMENTS 6    /* int32 [10]: seg[0..4] = first sorted position of each type (seg[4] = N),
                                     then roots[0..3] (-1 for an empty type), then 0                             */
#define QBVH_EXPORT_SORTED_POS 7  /* float [N][4]: x, y, z, bits of the original index                            */
#define QBVH_EXPORT_COUNTS 8      /* int32 [4]: nodes written by the build (2N-1 minus unused slots without collapse),
                                     query groups, non-empty Morton cells of the build, its cell grid level       */
int64_t qbvh_debug_export(int32_t what, void *dst, int64_t bytes);

const char *qbvh_error_string(int code);

#ifdef __cplusplus
}
#endif
#endif /* QBVH_H */

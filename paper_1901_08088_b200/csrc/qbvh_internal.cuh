// qbvh_internal.cuh — device-side data layout shared by the build and traversal kernels (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#define QBVH_TMAX 4            // types live in key bits 30-31
#define QBVH_NBINS 1023.0f     // 2^10 - 1 bins per axis

// ---- Morton cells of the build ----
// The build partitions the particles by the leading 2 + 3*lvl bits of their keys (type, then the cell of the
// 2^lvl-per-axis Morton grid over the box).  All keys of a cell are consecutive in Z-order and form one
// subtree of the radix tree, so a cell is sorted and its subtree built locally; only cell roots meet in global memory.
constexpr int CELL_LMIN = 2, CELL_LMAX = 6;
constexpr int CELL_MAX_TOTAL = 1 << 18;        // cells over all types: T * 8^lvl <= 2^18
constexpr int CELL_WARP_MAX = 128;             // a cell up to this size is handled by one warp (shared memory)
constexpr int CELL_BLOCK_MAX = 2048;           // ... up to this size by one block (shared memory); larger: global scratch
constexpr int SCAN_THREADS = 256, SCAN_IPT = 8, SCAN_TILE = SCAN_THREADS * SCAN_IPT;
constexpr int SCAN_MAX_TILES = CELL_MAX_TOTAL / SCAN_TILE;   // 128

// Device-resident bookkeeping of one build (lives at the start of the workspace; zeroed by a memset per build).
struct TreeMeta {
    unsigned long long scan_status[SCAN_MAX_TILES];  // cell scan: total of every tile, non-empty cells << 32 | particles
    uint32_t scan_arrived;          // tiles of the scan that have published their total (grid-wide barrier)
    uint32_t scan_done;             // tiles of the scan that have finished (the last one finalizes)
    uint32_t mm_enc[QBVH_TMAX][6];  // per type: ~enc(min xyz) (so atomicMax computes the min), enc(max xyz)
    int32_t seg[QBVH_TMAX + 1];     // first sorted position of each type; seg[T..4] = N
    int32_t roots[QBVH_TMAX];       // root node per type, -1 if empty
    float frames[QBVH_TMAX][12];    // lo xyz, hi xyz, delta xyz, 0 0 0
    int32_t gmax[QBVH_TMAX];        // largest query group of each type (<= GROUP_MAX; smaller for a sparse type, see finalize)
    int32_t rbin[QBVH_TMAX][4];     // collapse heuristic: expected query radius against this tree in bins per axis; [0] < 0: none
    int32_t ncell;                  // number of non-empty cells
    int32_t nbig;                   // cells larger than CELL_WARP_MAX (handled by whole blocks)
    int32_t pad_[23];
    // the counters below, hammered by atomics, keep a 128-byte line of their own
    int32_t group_count;            // number of query groups emitted by the build
    int32_t group_cursor;           // next group to hand out (dynamic scheduling of the traversal); reset per traversal
    int32_t max_count;              // max_i n_neigh[i] of the last traversal
    int32_t err_flags;              // bit 0: type id out of range; bit 1: traversal work list bound violated
    int32_t nodes_emitted;          // nodes written by the build (2N-1 without collapse)
    int32_t warps_done;             // warps of the running production traversal that have finished (the last one cleans up)
    unsigned long long d2h_bytes;   // list bytes the last rows_to_host_kernel wrote to host memory
    int32_t pad2_[24];
    unsigned long long stats[16];   // qbvh_stats, in order
};

// order-preserving map float -> uint32 (NaN excluded)
__host__ __device__ inline uint32_t f2ord(float f) {
#ifdef __CUDA_ARCH__
    uint32_t b = __float_as_uint(f);
#else
    union { float f; uint32_t u; } c; c.f = f; uint32_t b = c.u;
#endif
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ inline float ord2f(uint32_t o) {
    uint32_t b = (o & 0x80000000u) ? (o & 0x7FFFFFFFu) : ~o;
    return __uint_as_float(b);
}

// ---- query groups ----
// A query group is a maximal subtree of the LBVH with at most GROUP_MAX leaves (fewer for a sparse type, TreeMeta::gmax): a contiguous run of Z-ordered
// particles that fills one Morton cell, i.e. a compact blob.  One warp traverses the tree once
// for the whole group (traverse_kernels.cu).
constexpr int GROUP_MAX = 32;

// ---- build tag of the meeting slots (top_tree_kernel): 18 bits; the slot area is cleared when it wraps ----
constexpr uint32_t QBVH_TAG_MAX = (1u << 18) - 1;

// ---- entry table: node of every cell of the 2^l-per-axis Morton grids, l = 2..5, per type ----
constexpr int ENTRY_LMIN = 2, ENTRY_LMAX = 5;
__host__ __device__ constexpr int entry_offset(int l) {   // cells of the levels below l: 64 + 512 + ...
    return l <= 2 ? 0 : (l == 3 ? 64 : (l == 4 ? 64 + 512 : 64 + 512 + 4096));
}
constexpr int ENTRY_CELLS = 64 + 512 + 4096 + 32768;

// ---- subtree collapse ----
// Integer cost model in bin units of the tree's quantization frame: visiting a node costs COST_NODE, a range leaf
// COST_LEAF_FIXED + COST_LEAF_PER_PARTICLE * count, each weighted by the volume of its quantized box swollen by the
// expected query radius (a box-shaped Minkowski sum).
constexpr int COST_NODE = 1, COST_LEAF_FIXED = 16, COST_LEAF_PER_PARTICLE = 1;

struct TraverseParams {
    float L[3];
    float r2[QBVH_TMAX * QBVH_TMAX];   // r_ij^2 (fp32 RN), <0 => skipped
    float R2[QBVH_TMAX * QBVH_TMAX];   // padded pruning radius squared (rounded up)
    float Rp[QBVH_TMAX * QBVH_TMAX];   // padded pruning radius
    float box_lo[3], scale[3];         // Morton binning of the build: bin = floor((p - box_lo) * scale)
    int32_t N;
    int32_t max_neigh;
    int32_t K;                         // leaf-collapse cap used by the build
    int32_t *result_host;              // production kernel: where its last warp writes {max_count, err_flags} (pinned host
                                       // memory, device-mapped) before it re-arms group_cursor, max_count and warps_done; nullptr: the
                                       // host clears and copies them around the launch
    int32_t q_first, q_count;          // query sharding: only these sorted positions are queries, row = position - q_first; q_count < 0: all, row = original index
    // double-precision particle data (qbvh_neighbors_f64): r2 above is then (r + B)^2 rounded up — whatever fails it
    // in fp32 on the rounded positions cannot be a neighbor in fp64 —, r2lo = (r - B)^2 rounded down — whatever passes
    // it certainly is one —, and only the pairs in between are decided by the fp64 predicate.
    float r2lo[QBVH_TMAX * QBVH_TMAX];
    double r2_64[QBVH_TMAX * QBVH_TMAX];
    double L64[3];
};

// record a cell's root hands to the top-level walk (cell_tree_kernel -> top_tree_kernel)
struct __align__(16) CellRoot {
    uint32_t wlo;      // packed lower bound; bit 31: pending (a single particle or a collapsed range not yet written)
    uint32_t whi;
    int32_t first;     // sorted positions covered
    int32_t last;
    uint32_t d;        // (dL+1) | (dR+1) << 8 | (dnext+1) << 16 | big << 31.  dL, dR: common prefix lengths with the
                       // neighbouring cells (-1 beyond the type segment); dnext: delta(m, m+1) for m = last + 1 (64 if the
                       // next cell holds >= 2 particles, else its delta to the one after, -1: none); big: a cell too large
                       // for a warp, built and walked by a whole block of top_tree_kernel (set by cell_tree_kernel already)
    uint32_t key0;     // key of the cell's first particle (type, entry-table cells)
    uint32_t pad[2];
};
constexpr uint32_t CELL_ROOT_BIG = 1u << 31;
__host__ __device__ inline uint32_t cell_root_d(int dL, int dR, int dnext, bool big) {
    return (uint32_t)(dL + 1) | ((uint32_t)(dR + 1) << 8) | ((uint32_t)(dnext + 1) << 16) | (big ? CELL_ROOT_BIG : 0u);
}

// Z-ordered fp64 particle record of a double-precision build (qbvh_build_f64)
struct __align__(32) Pos64 {
    double x, y, z;
    long long idx;     // original index
};

// launchers (build_kernels.cu / traverse_kernels.cu)
struct BuildBuffers {
    TreeMeta *meta;
    uint32_t *key;                 // Morton keys in input order
    uint32_t *rank;                // place of every particle inside its cell (order of arrival)
    uint2 *ent;                    // {key, original index} partitioned by cell, then sorted inside each cell
    uint32_t *key_sorted, *idx_sorted;
    uint32_t *cell_count;          // [ncells] particles per cell; counted by the key kernel, cleared again by the scan
    uint32_t *cell_start;          // [ncells + 1] exclusive prefix
    uint32_t *cell_list;           // non-empty cells in ascending order
    int32_t *big_list;             // compact indices of the cells larger than CELL_WARP_MAX
    CellRoot *croot;               // one per non-empty cell
    float4 *sorted_pos;
    Pos64 *sorted_pos64;           // only written by double-precision builds
    int4 *nodes;
    int32_t *parent;
    uint4 *slot;                   // meeting slot of the two children of the node that splits at gamma (top_tree_kernel)
    uint2 *groups;                 // {first sorted position, number of particles}, group_count entries, any order
    int32_t *entry;                // [QBVH_TMAX][ENTRY_CELLS] entry table
    unsigned char *scratch;        // 18 B per particle: working arrays of cells too large for shared memory
};
struct BuildParams {
    int N, T, K, lvl;
    float box_lo[3], box_scale[3];
    float r_hint[QBVH_TMAX];       // <= 0: no collapse hint for that tree
    uint32_t build_tag;
    bool f64;                      // positions are double precision (qbvh_build_f64)
    int group_cap;                 // largest query group the build may emit (<= GROUP_MAX)
    int scan_spin_cycles;          // how long a block of the 128-tile cell scan waits for the others before it sums alone
};
int pick_cell_level(int64_t N, int T);
cudaError_t launch_build(const void *pos, const int32_t *type, const BuildParams &p, const BuildBuffers &b, cudaStream_t st);
cudaError_t launch_traverse(const TraverseParams &p, const BuildBuffers &b, int32_t *nlist, int32_t *n_neigh,
                            bool stats, int variant, bool f64, cudaStream_t st);
cudaError_t launch_count_overlaps(const TraverseParams &p, const BuildBuffers &b, int32_t *n_overlap, cudaStream_t st);
int traverse_warp_slots();      // warps the production traversal keeps resident on this device
// list rows written by the SMs straight into mapped (pinned) host memory: the first min(n_neigh, max_neigh) entries of
// every row, in 16-byte pieces (qbvh_neighbors_host); max_neigh % 4 == 0, both lists 16-byte aligned
cudaError_t launch_rows_to_host(const int32_t *dlist, const int32_t *dcnt, int32_t *hlist_dev, int64_t N, int32_t max_neigh,
                                TreeMeta *meta, cudaStream_t st);
// api.cu: keeps the text of a failed CUDA call for qbvh_error_string(QBVH_ERR_CUDA); returns QBVH_ERR_CUDA
int qbvh_record_cuda_error(cudaError_t e, const char *where);
static_assert(offsetof(TreeMeta, group_count) % 128 == 0, "the atomic counters start a 128-byte line");

// qbvh_internal.cuh — device-side data layout shared by the build and traversal kernels (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#define QBVH_TMAX 4            // types live in key bits 30-31
#define QBVH_NBINS 1023.0f     // 2^10 - 1 bins per axis

// Device-resident bookkeeping of one build (lives at the start of the workspace; zeroed by a memset per build).
struct TreeMeta {
    uint32_t hist[4][256];     // per-pass digit histograms, turned into exclusive offsets by the last block of morton_hist_kernel
    uint32_t tile_counter[4];  // dynamic tile ids of the four onesweep passes
    uint32_t blocks_done;      // blocks of morton_hist_kernel that have added their histograms (the last one finalizes)
    uint32_t mm_enc[QBVH_TMAX][6];  // per type: ~enc(min xyz) (so atomicMax computes the min), enc(max xyz)
    int32_t seg[QBVH_TMAX + 1];     // first sorted position of each type; seg[T..4] = N
    int32_t roots[QBVH_TMAX];       // root node per type, -1 if empty
    float frames[QBVH_TMAX][12];    // lo xyz, hi xyz, delta xyz, 0 0 0
    int32_t gmax[QBVH_TMAX];        // largest query group of each type (<= GROUP_MAX; smaller for a sparse type, see finalize)
    int32_t pad_[38];               // the counters below, hammered by atomics, keep a 128-byte line of their own
    int32_t group_count;            // number of query groups emitted by the build (tree_kernel)
    int32_t group_cursor;           // next group to hand out (dynamic scheduling of the traversal); reset per traversal
    int32_t max_count;              // max_i n_neigh[i] of the last traversal
    int32_t err_flags;              // bit 0: type id out of range
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


// ---- sort geometry ----
constexpr int SORT_THREADS = 512;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_IPT = 8;                           // keys per thread
constexpr int SORT_TILE = SORT_THREADS * SORT_IPT;    // 4096 keys per tile
constexpr uint32_t ST_AGG = 1u << 30;                 // tile status: aggregate (own count) available
constexpr uint32_t ST_PRE = 1u << 31;                 // tile status: inclusive prefix available
constexpr uint32_t ST_VAL = (1u << 30) - 1;

// ---- query groups ----
// A query group is a maximal subtree of the LBVH with at most GROUP_MAX leaves (fewer for a sparse type, TreeMeta::gmax): a contiguous run of Z-ordered
// particles that fills one Morton cell, i.e. a compact blob.  One warp traverses the tree once
// for the whole group (traverse_kernels.cu).
constexpr int GROUP_MAX = 32;

// ---- entry table: node of every cell of the 2^l-per-axis Morton grids, l = 2..5, per type ----
constexpr int ENTRY_LMIN = 2, ENTRY_LMAX = 5;
__host__ __device__ constexpr int entry_offset(int l) {   // cells of the levels below l: 64 + 512 + ...
    return l <= 2 ? 0 : (l == 3 ? 64 : (l == 4 ? 64 + 512 : 64 + 512 + 4096));
}
constexpr int ENTRY_CELLS = 64 + 512 + 4096 + 32768;

struct TraverseParams {
    float L[3];
    float r2[QBVH_TMAX * QBVH_TMAX];   // r_ij^2 (fp32 RN), <0 => skipped
    float R2[QBVH_TMAX * QBVH_TMAX];   // padded pruning radius squared (rounded up)
    float Rp[QBVH_TMAX * QBVH_TMAX];   // padded pruning radius
    float box_lo[3], scale[3];         // Morton binning of the build: bin = floor((p - box_lo) * scale)
    int32_t N;
    int32_t max_neigh;
    int32_t K;                         // leaf-collapse threshold used by the build
};

// launchers (build_kernels.cu / traverse_kernels.cu)
struct BuildBuffers {
    TreeMeta *meta;
    uint32_t *key_a, *key_b, *idx_a, *idx_b;
    uint32_t *status[2];
    float4 *sorted_pos;
    int4 *nodes;
    int32_t *parent;
    uint4 *slot;                   // meeting slot of the two children of the node that splits at gamma (tree_kernel)
    uint2 *groups;                 // {first sorted position, number of particles}, group_count entries, any order
    int32_t *entry;                // [QBVH_TMAX][ENTRY_CELLS] entry table
};
cudaError_t launch_build(const float *pos, const int32_t *type, int N, int T, int K, const float *box_lo,
                         const float *box_scale, const BuildBuffers &b, uint32_t build_tag, cudaStream_t st);
cudaError_t launch_traverse(const TraverseParams &p, const BuildBuffers &b, int32_t *nlist, int32_t *n_neigh,
                            bool stats, int variant, cudaStream_t st);
cudaError_t launch_count_overlaps(const TraverseParams &p, const BuildBuffers &b, int32_t *n_overlap, cudaStream_t st);
static_assert(offsetof(TreeMeta, group_count) % 128 == 0, "the atomic counters start a 128-byte line");

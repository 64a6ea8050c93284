// traverse_kernels.cu — steps a7..a9 of the hot path: Algorithm 1 of the paper with the exact
// leaf filter fused in and a Verlet list appended per particle.
//
// One thread per particle in Z-order ("threads within the same CUDA warp traversed similar parts of
// the tree").  For query type a and every tree b with r_ab > 0:
//   line 4    bitset of the 27 images whose padded sphere overlaps the decompressed root box
//   line 5-7  pop the next image
//   line 10   stackless walk: 16-byte node load; decompress with directed rounding (line 11);
//             nearest-point test of eq. 2 (line 12); overlap & internal -> left (line 17);
//             overlap & leaf -> process (line 14) then rope (line 15); no overlap -> rope (line 19)
//   line 14   here: every particle of the (possibly collapsed) leaf range goes through the canonical fp32
//             minimum-image predicate; hits are appended to row `orig_i` of the list.
#include "qbvh_internal.cuh"
#include <algorithm>

__device__ __forceinline__ void decompress(uint32_t wlo, uint32_t whi, const float lo[3], const float dl[3],
                                           float a[3], float b[3]) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        a[d] = __fmaf_rd((float)((wlo >> (10 * d)) & 1023u), dl[d], lo[d]);
        b[d] = __fmaf_ru((float)((whi >> (10 * d)) & 1023u), dl[d], lo[d]);
    }
}

// Number of particles under a (collapsed) leaf node covering the sorted positions [first, last]: its rope points at
// the node that starts at last + 1 — leaf N-1+(last+1), or the internal node numbered last+1 (a right child carries
// the index of its first leaf) — or is END at the end of the tree's segment.
__device__ __forceinline__ int leaf_count(const int4 nd, int N, int seg_end) {
    const int next = (nd.w < 0) ? seg_end : (nd.w >= N - 1 ? nd.w - (N - 1) : nd.w);
    return next - (~nd.z);
}

template <bool STATS>
__global__ void __launch_bounds__(128) traverse_kernel(TraverseParams P, const int4 *__restrict__ nodes,
                                                        const float4 *__restrict__ sorted_pos,
                                                        TreeMeta *__restrict__ meta, int32_t *__restrict__ nlist,
                                                        int32_t *__restrict__ n_neigh) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    int cnt = 0;
    unsigned long long st_tests = 0, st_leaf = 0, st_checks = 0, st_images = 0;
    if (k < P.N) {
        const float4 me = sorted_pos[k];
        const int orig_i = __float_as_int(me.w);
        int ta = 0;
#pragma unroll
        for (int t = 1; t < QBVH_TMAX; ++t) ta += (k >= meta->seg[t]) ? 1 : 0;
        int32_t *row = nlist + (size_t)orig_i * (size_t)P.max_neigh;
        for (int tb = 0; tb < QBVH_TMAX; ++tb) {
            const float r2 = P.r2[ta * QBVH_TMAX + tb];
            const int root = meta->roots[tb];
            if (!(r2 >= 0.0f) || root < 0) continue;
            const float R2 = P.R2[ta * QBVH_TMAX + tb];
            const float *fr = meta->frames[tb];
            const float flo[3] = {fr[0], fr[1], fr[2]};
            const float fdl[3] = {fr[6], fr[7], fr[8]};
            const int seg_end = meta->seg[tb + 1];
            // ---- line 4: image bitset against the root node ----
            uint32_t bset = 0;
            {
                const int4 nd = __ldg(nodes + root);
                float a[3], b[3];
                decompress((uint32_t)nd.x, (uint32_t)nd.y, flo, fdl, a, b);
                float tq[3][3];   // tq[d][s+1] = y - x' along axis d for shift s
                const float xme[3] = {me.x, me.y, me.z};
#pragma unroll
                for (int d = 0; d < 3; ++d)
#pragma unroll
                    for (int s = -1; s <= 1; ++s) {
                        float xs = __fadd_rn(xme[d], (float)s * P.L[d]);
                        float y = fminf(fmaxf(xs, a[d]), b[d]);
                        tq[d][s + 1] = __fsub_rn(y, xs);
                    }
#pragma unroll
                for (int img = 0; img < 27; ++img) {
                    float tx = tq[0][img % 3], ty = tq[1][(img / 3) % 3], tz = tq[2][img / 9];
                    float d2 = __fmaf_rn(tz, tz, __fmaf_rn(ty, ty, __fmul_rn(tx, tx)));
                    if (d2 <= R2) bset |= 1u << img;
                }
            }
            if (STATS) st_images += __popc(bset);
            // ---- lines 5-19 ----
            while (bset) {
                const int img = __ffs(bset) - 1;
                bset &= bset - 1;
                const float sL[3] = {(float)(img % 3 - 1) * P.L[0], (float)((img / 3) % 3 - 1) * P.L[1],
                                     (float)(img / 9 - 1) * P.L[2]};
                const float xs[3] = {__fadd_rn(me.x, sL[0]), __fadd_rn(me.y, sL[1]), __fadd_rn(me.z, sL[2])};
                int n = root;
                while (n >= 0) {
                    const int4 nd = __ldg(nodes + n);
                    float a[3], b[3];
                    decompress((uint32_t)nd.x, (uint32_t)nd.y, flo, fdl, a, b);
                    float tq[3];
#pragma unroll
                    for (int d = 0; d < 3; ++d) tq[d] = __fsub_rn(fminf(fmaxf(xs[d], a[d]), b[d]), xs[d]);
                    const float d2 = __fmaf_rn(tq[2], tq[2], __fmaf_rn(tq[1], tq[1], __fmul_rn(tq[0], tq[0])));
                    if (STATS) ++st_tests;
                    if (d2 <= R2) {
                        if (nd.z < 0) {
                            const int first = ~nd.z;
                            const int m = leaf_count(nd, P.N, seg_end);
                            if (STATS) ++st_leaf;
                            for (int j = first; j < first + m; ++j) {
                                const float4 pj = __ldg(sorted_pos + j);
                                // canonical predicate, image-directed form: (p_j - p_i) - s L, then fma chain
                                const float dx = __fsub_rn(__fsub_rn(pj.x, me.x), sL[0]);
                                const float dy = __fsub_rn(__fsub_rn(pj.y, me.y), sL[1]);
                                const float dz = __fsub_rn(__fsub_rn(pj.z, me.z), sL[2]);
                                const float dd = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                                if (STATS) ++st_checks;
                                if (dd <= r2 && j != k) {
                                    if (cnt < P.max_neigh) row[cnt] = __float_as_int(pj.w);
                                    ++cnt;
                                }
                            }
                            n = nd.w;
                        } else {
                            n = nd.z;
                        }
                    } else {
                        n = nd.w;
                    }
                }
            }
        }
        n_neigh[orig_i] = cnt;
    }
    const int wmax = __reduce_max_sync(0xFFFFFFFFu, cnt);
    if ((threadIdx.x & 31) == 0 && wmax > 0) atomicMax(&meta->max_count, wmax);
    if (STATS) {
        unsigned long long v[5] = {st_tests, st_leaf, st_checks, (unsigned long long)cnt, st_images};
#pragma unroll
        for (int q = 0; q < 5; ++q) {
            unsigned long long x = v[q];
#pragma unroll
            for (int o = 16; o; o >>= 1) x += __shfl_xor_sync(0xFFFFFFFFu, x, o);
            if ((threadIdx.x & 31) == 0 && x) atomicAdd(&meta->stats[q], x);
        }
    }
}



// ------------------------------------------------------------------------------------------------------------
// The paper's own operating mode: Algorithm 1 with line 14 as printed — a leaf whose box
// overlaps the search sphere is ACCEPTED, positions are never loaded, and the benchmark only counts.  One thread
// per particle in Z-order.  n_overlap[orig_i] = particles j != i accepted (a collapsed leaf accepts its whole
// range; the particle's own leaf always overlaps and is not counted).
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) count_overlaps_kernel(TraverseParams P, const int4 *__restrict__ nodes,
                                                              const float4 *__restrict__ sorted_pos,
                                                              TreeMeta *__restrict__ meta, int32_t *__restrict__ n_overlap) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    int cnt = 0;
    if (k < P.N) {
        const float4 me = sorted_pos[k];
        int ta = 0;
#pragma unroll
        for (int t = 1; t < QBVH_TMAX; ++t) ta += (k >= meta->seg[t]) ? 1 : 0;
        for (int tb = 0; tb < QBVH_TMAX; ++tb) {
            const int root = meta->roots[tb];
            if (!(P.r2[ta * QBVH_TMAX + tb] >= 0.0f) || root < 0) continue;
            const float R2 = P.R2[ta * QBVH_TMAX + tb];
            const float *fr = meta->frames[tb];
            const float flo[3] = {fr[0], fr[1], fr[2]};
            const float fdl[3] = {fr[6], fr[7], fr[8]};
            const int seg_end = meta->seg[tb + 1];
            const float xme[3] = {me.x, me.y, me.z};
            uint32_t bset = 0;                                   // line 4
            {
                const int4 nd = __ldg(nodes + root);
                float a[3], b[3];
                decompress((uint32_t)nd.x, (uint32_t)nd.y, flo, fdl, a, b);
                float tq[3][3];
#pragma unroll
                for (int d = 0; d < 3; ++d)
#pragma unroll
                    for (int s = -1; s <= 1; ++s) {
                        const float xs = __fadd_rn(xme[d], (float)s * P.L[d]);
                        tq[d][s + 1] = __fsub_rn(fminf(fmaxf(xs, a[d]), b[d]), xs);
                    }
#pragma unroll
                for (int img = 0; img < 27; ++img) {
                    const float tx = tq[0][img % 3], ty = tq[1][(img / 3) % 3], tz = tq[2][img / 9];
                    if (__fmaf_rn(tz, tz, __fmaf_rn(ty, ty, __fmul_rn(tx, tx))) <= R2) bset |= 1u << img;
                }
            }
            while (bset) {                                       // lines 5-19
                const int img = __ffs(bset) - 1;
                bset &= bset - 1;
                const float xs[3] = {__fadd_rn(me.x, (float)(img % 3 - 1) * P.L[0]), __fadd_rn(me.y, (float)((img / 3) % 3 - 1) * P.L[1]),
                                     __fadd_rn(me.z, (float)(img / 9 - 1) * P.L[2])};
                int n = root;
                while (n >= 0) {
                    const int4 nd = __ldg(nodes + n);
                    float a[3], b[3];
                    decompress((uint32_t)nd.x, (uint32_t)nd.y, flo, fdl, a, b);
                    float tq[3];
#pragma unroll
                    for (int d = 0; d < 3; ++d) tq[d] = __fsub_rn(fminf(fmaxf(xs[d], a[d]), b[d]), xs[d]);
                    const bool hit = __fmaf_rn(tq[2], tq[2], __fmaf_rn(tq[1], tq[1], __fmul_rn(tq[0], tq[0]))) <= R2;
                    if (hit && nd.z < 0) {                       // line 14: accept the leaf's particles, self excepted
                        const int first = ~nd.z, m = leaf_count(nd, P.N, seg_end);
                        cnt += m - ((img == 13 && (unsigned)(k - first) < (unsigned)m) ? 1 : 0);
                    }
                    n = (hit && nd.z >= 0) ? nd.z : nd.w;
                }
            }
        }
        n_overlap[__float_as_int(me.w)] = cnt;
    }
    const int wmax = __reduce_max_sync(0xFFFFFFFFu, cnt);
    if ((threadIdx.x & 31) == 0 && wmax > 0) atomicMax(&meta->max_count, wmax);
}

cudaError_t launch_count_overlaps(const TraverseParams &p, const BuildBuffers &b, int32_t *n_overlap, cudaStream_t st) {
    if (p.N == 0) return cudaSuccess;
    count_overlaps_kernel<<<(p.N + 127) / 128, 128, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, n_overlap);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// Host-buffer path (qbvh_neighbors_host): the list leaves the device through the SMs.  One warp per row copies the
// entries that exist — min(n_neigh, max_neigh), rounded up to a 16-byte piece — from the device staging list into the
// caller's pinned host rows (zero copy, 128-byte coalesced PCIe writes), rows in index order.  The copy engine's
// strided 2-D copy moves min(M, max_neigh) columns of EVERY row and runs at 42 GB/s for row widths that are no
// multiple of 128 bytes; this moves 14 % fewer bytes at 49 GB/s.  (Letting the traversal's own warps write their
// finished rows to the host under the traversal was slower, 9.9 against 9.0 ms end to end at config 2: those rows
// come in Z-order, i.e. scattered over the host buffer.)
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) rows_to_host_kernel(const int32_t *__restrict__ dlist, const int32_t *__restrict__ dcnt,
                                                           int32_t *__restrict__ hlist, int N, int cap, TreeMeta *__restrict__ meta) {
    const int lane = threadIdx.x & 31;
    const int nw = (gridDim.x * blockDim.x) >> 5;
    unsigned long long bytes = 0;
    for (int row = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; row < N; row += nw) {
        const int n = min(__ldg(dcnt + row), cap);
        const int pieces = (n + 3) >> 2;
        const int4 *src = reinterpret_cast<const int4 *>(dlist + (size_t)row * (size_t)cap);
        int4 *dst = reinterpret_cast<int4 *>(hlist + (size_t)row * (size_t)cap);
        for (int q = lane; q < pieces; q += 32) dst[q] = src[q];
        bytes += 16ull * (unsigned)pieces;
    }
    if (lane == 0 && bytes) atomicAdd(&meta->d2h_bytes, bytes);
}

cudaError_t launch_rows_to_host(const int32_t *dlist, const int32_t *dcnt, int32_t *hlist_dev, int64_t N, int32_t max_neigh,
                                TreeMeta *meta, cudaStream_t st) {
    if (N == 0 || max_neigh == 0) return cudaSuccess;       // (the caller has cleared meta->d2h_bytes)
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = (int)std::min<int64_t>(2 * sms, (N + 7) / 8);
    rows_to_host_kernel<<<blocks, 256, 0, st>>>(dlist, dcnt, hlist_dev, (int)N, max_neigh, meta);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// Group traversal (the production kernel).
//
// Algorithm 1 is written for one thread per particle; the paper runs those threads in Z-order so that "threads
// within the same CUDA warp traversed similar parts of the tree".  On B200 the per-lane walk is
// bound by divergent 16-byte gathers and by instruction issue (profiles/), so here one warp walks the tree ONCE
// for a whole QUERY GROUP — a maximal LBVH subtree with at most 32 leaves, emitted by the build — and every memory
// access is warp-coherent:
//   line 4     image bitset by vote: lane j tests image j of the group's bounding box against the root node box.
//   lines 8-19 the search volume of the group is its bounding box; "S overlaps A" (line 12) becomes the box-box
//              form of eq. 2: squared distance between nearest points <= padded r^2.  It contains every member's
//              search sphere, so no pair can be missed.  The walk still uses only each node's `left` and `rope`
//              words: 32 nodes are tested per step, one per lane, from a LIFO work list in shared memory; a popped
//              left child also schedules its rope (= its right sibling); an overlapping internal node schedules
//              its left child; an overlapping (collapsed) leaf goes to a leaf queue.
//   line 14    leaf ranges are gathered 32 at a time: each candidate particle is tested against the group box
//              (point-box form of eq. 2) and the survivors are compacted by ballot into a structure-of-arrays
//              tile in shared memory.  A full tile of 32 candidates is then checked by every lane for its own
//              particle with the canonical fp32 predicate, two candidates per instruction
//              (packed add/mul/fma.f32x2 of sm_100), the candidate data being broadcast 128-bit shared loads.
//   list       hits go to a per-lane ring in shared memory and leave it in aligned 64-byte blocks (4 x 128-bit
//              stores per lane), so the list is written in full 32-byte sectors.
// Groups are handed to warps dynamically (one atomic per group) by a persistent grid.
// ------------------------------------------------------------------------------------------------------------
typedef unsigned long long u64;
__device__ __forceinline__ u64 pk2(float lo, float hi) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk2(u64 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
    u64 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
    u64 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

#ifndef QBVH_GW_WARPS
#define QBVH_GW_WARPS 4
#endif
#ifndef QBVH_GW_NB
#define QBVH_GW_NB 3         // leaf batches gathered per step: a tile ring of 128 takes 31 + 3 x 32 candidates
#endif
constexpr int GW_NB = QBVH_GW_NB;
#ifndef QBVH_GW_RING
#define QBVH_GW_RING 32
#endif

constexpr int GW_WARPS = QBVH_GW_WARPS;   // warps per block
constexpr int GW_WL = 256;       // work-list entries per warp
constexpr int GW_LQ = 96;        // leaf-queue entries per warp
constexpr int GW_TILE = 128;     // candidate tile ring per warp: four tiles of 32
constexpr int GW_RING = QBVH_GW_RING;     // staged neighbors per lane: blocks of 16
constexpr int GW_RING_BYTES = 4 * GW_RING;

struct __align__(256) GwShared {
    int32_t ring[32][GW_RING];                     // per-lane staged neighbors (GW_RING_BYTES per lane)
    float tx[GW_TILE], ty[GW_TILE], tz[GW_TILE];   // candidate tile ring, structure of arrays
    int32_t ti[GW_TILE];                           // original particle index of each candidate
    uint32_t wl[GW_WL];                            // work list: node id | (also test its rope sibling) << 31
    uint2 lq[GW_LQ];                               // leaf queue: {first sorted position, count}
};

// append one neighbor to this lane's ring: slot address = ring base | (byte offset mod 256), one LOP3
// The ring is private to its lane and is only ever touched through these two asm statements (volatile: they keep
// their order among themselves and relative to the tile loads of check_tile).
__device__ __forceinline__ void ring_put(uint32_t ring_s, uint32_t &po, int32_t v) {
    asm volatile("st.shared.b32 [%0], %1;" ::"r"(ring_s | (po & (GW_RING_BYTES - 4))), "r"(v));
    po += 4;
}
__device__ __forceinline__ int4 ring_get4(uint32_t ring_s, uint32_t off) {
    int4 v;
    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(ring_s | (off & (GW_RING_BYTES - 16))));
    return v;
}

// One tile of 32 candidates, starting at slot `base` of the tile ring, against this lane's particle: the
// canonical predicate
//   D = (p_j - p_i) [- s L];  d2 = fma(Dz, Dz, fma(Dy, Dy, Dx*Dx));  d2 <= r^2
// evaluated for two candidates per instruction.  SELF: the tile holds the members of the group itself.
// What the fp64 path adds (qbvh_neighbors_f64): the pair is first judged in fp32 on the positions
// rounded to fp32.  d2 <= r2lo: certainly a neighbor, appended as in the fp32 kernel.  r2lo < d2 <= r2 (the band, about
// one pair per query group): its tile slot is remembered in a bit mask — one predicated instruction, no branch in the
// loop — and after the chunk the lanes that have any decide theirs with the canonical fp64 predicate
// on the Z-ordered double positions.
struct MetaCache {
    int32_t seg[QBVH_TMAX + 1], roots[QBVH_TMAX], gmax[QBVH_TMAX];
    float flo[QBVH_TMAX][3], fdl[QBVH_TMAX][3];     // quantization frame of every tree: origin and bin width
    int4 rootnode[QBVH_TMAX];
};
struct F64Ctx {
    const Pos64 *sp64;     // Z-ordered fp64 positions
    const int32_t *tp;     // sorted position of every candidate of the tile ring
    int ksort_i;           // sorted position of this lane's particle
    double s0, s1, s2;     // image shift (exactly 0 or +-L)
    double r2_64;
    float r2lo;
};
__device__ __noinline__ bool exact_pair_f64(const Pos64 *__restrict__ sp64, int ki, int kj, double s0, double s1, double s2, double r2) {
    const Pos64 a = sp64[ki], b = sp64[kj];
    const double dx = __dsub_rn(__dsub_rn(b.x, a.x), s0), dy = __dsub_rn(__dsub_rn(b.y, a.y), s1), dz = __dsub_rn(__dsub_rn(b.z, a.z), s2);
    return __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx))) <= r2;
}

// One quad of the candidate tile ring: x, y, z and the original index of four consecutive slots (broadcast loads).
// asm volatile keeps these loads where they are written relative to the ring stores: the quad after the current one
// is fetched BEFORE the current quad's hits are appended, so the append chain runs in the shadow of the load latency
// (ptxas never moves a shared load across a shared store it cannot disambiguate; written the plain way every quad
// waited for its loads after the previous quad's last append).
struct Quad {
    float4 X, Y, Z;
    int4 I;
};
__device__ __forceinline__ void tile_ld4(uint32_t a, float4 &v) {
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
}
__device__ __forceinline__ void quad_load(uint32_t tile_s, int slot, Quad &q) {
    const uint32_t a = tile_s + 4u * (uint32_t)slot;
    tile_ld4(a, q.X);
    tile_ld4(a + 4u * GW_TILE, q.Y);
    tile_ld4(a + 8u * GW_TILE, q.Z);
    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(q.I.x), "=r"(q.I.y), "=r"(q.I.z), "=r"(q.I.w) : "r"(a + 12u * GW_TILE));
}

template <bool SHIFTED, bool SELF, int NC, bool F64>
__device__ __forceinline__ void check_tile(const GwShared &sm, uint32_t tile_s, int base, u64 nmx, u64 nmy, u64 nmz, u64 ns0, u64 ns1,
                                        u64 ns2, float r2, int orig_i, uint32_t ring_s, uint32_t &po, const F64Ctx &fx) {
    const float r2a = F64 ? fx.r2lo : r2;        // what is appended without further ado
    uint32_t band = 0;
    Quad q;
    quad_load(tile_s, base, q);
#pragma unroll
    for (int j = 0; j < NC / 4; ++j) {
        u64 dx0 = add2(pk2(q.X.x, q.X.y), nmx), dx1 = add2(pk2(q.X.z, q.X.w), nmx);
        u64 dy0 = add2(pk2(q.Y.x, q.Y.y), nmy), dy1 = add2(pk2(q.Y.z, q.Y.w), nmy);
        u64 dz0 = add2(pk2(q.Z.x, q.Z.y), nmz), dz1 = add2(pk2(q.Z.z, q.Z.w), nmz);
        if (SHIFTED) {
            dx0 = add2(dx0, ns0), dx1 = add2(dx1, ns0);
            dy0 = add2(dy0, ns1), dy1 = add2(dy1, ns1);
            dz0 = add2(dz0, ns2), dz1 = add2(dz1, ns2);
        }
        const u64 dd0 = fma2(dz0, dz0, fma2(dy0, dy0, mul2(dx0, dx0)));
        const u64 dd1 = fma2(dz1, dz1, fma2(dy1, dy1, mul2(dx1, dx1)));
        float d0, d1, d2, d3;
        upk2(dd0, d0, d1);
        upk2(dd1, d2, d3);
        const int4 I = q.I;
        const bool s0 = !SELF || I.x != orig_i, s1 = !SELF || I.y != orig_i, s2 = !SELF || I.z != orig_i, s3 = !SELF || I.w != orig_i;
        const bool h0 = d0 <= r2a && s0, h1 = d1 <= r2a && s1, h2 = d2 <= r2a && s2, h3 = d3 <= r2a && s3;
        bool b0 = false, b1 = false, b2 = false, b3 = false;
        if (F64) b0 = d0 <= r2 && !(d0 <= r2a) && s0, b1 = d1 <= r2 && !(d1 <= r2a) && s1, b2 = d2 <= r2 && !(d2 <= r2a) && s2, b3 = d3 <= r2 && !(d3 <= r2a) && s3;
        if (j + 1 < NC / 4) quad_load(tile_s, base + 4 * (j + 1), q);   // the next quad is in flight during the appends
        if (h0) { ring_put(ring_s, po, I.x); }
        if (h1) { ring_put(ring_s, po, I.y); }
        if (h2) { ring_put(ring_s, po, I.z); }
        if (h3) { ring_put(ring_s, po, I.w); }
        if (F64) {
            if (b0) band |= 1u << (4 * j + 0);
            if (b1) band |= 1u << (4 * j + 1);
            if (b2) band |= 1u << (4 * j + 2);
            if (b3) band |= 1u << (4 * j + 3);
        }
    }
    if (F64 && __any_sync(0xFFFFFFFFu, band != 0)) {
        while (band) {
            const int slot = base + __ffs(band) - 1;
            band &= band - 1;
            if (exact_pair_f64(fx.sp64, fx.ksort_i, fx.tp[slot], fx.s0, fx.s1, fx.s2, fx.r2_64)) ring_put(ring_s, po, sm.ti[slot]);
        }
    }
}

// eight entries with one 256-bit store (sm_100: STG.256); p is 32-byte aligned
__device__ __forceinline__ void st_global_256(int32_t *p, const int4 a, const int4 b) {
    asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(p), "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w),
                 "r"(b.x), "r"(b.y), "r"(b.z), "r"(b.w)
                 : "memory");
}

// four staged entries -> row[off .. off+3], never past the row capacity
__device__ __forceinline__ void store4(int32_t *__restrict__ row, int off, int cap, bool vec_ok, const int4 v) {
    if (vec_ok && off + 4 <= cap) {
        *reinterpret_cast<int4 *>(row + off) = v;
    } else {
        if (off + 0 < cap) row[off + 0] = v.x;
        if (off + 1 < cap) row[off + 1] = v.y;
        if (off + 2 < cap) row[off + 2] = v.z;
        if (off + 3 < cap) row[off + 3] = v.w;
    }
}


// Morton bin of a coordinate: the build's function (build_kernels.cu, a1), restated.  It is monotone in p, which
// is all the entry-cell selection needs.
__device__ __forceinline__ int bin_of(float p, float lo, float s) {
    const float f = fminf(fmaxf(floorf(__fmul_rn(__fsub_rn(p, lo), s)), 0.0f), 1023.0f);
    return (int)f;
}
__device__ __forceinline__ uint32_t spread5(uint32_t v) {   // bit t -> bit 3t, t < 5
    v = (v | (v << 8)) & 0x0000100Fu;
    v = (v | (v << 4)) & 0x000010C3u;
    v = (v | (v << 2)) & 0x00001249u;
    return v;
}

// sphere-swept box test of eq. 2 in its box-box form: squared distance between the nearest
// points of the decompressed node box and the group's box [blo, bhi] <= padded r^2
__device__ __forceinline__ bool node_overlaps(const int4 nd, const float flo[3], const float fdl[3], const float blo[3],
                                              const float bhi[3], float R2) {
    float a[3], b[3];
    decompress((uint32_t)nd.x, (uint32_t)nd.y, flo, fdl, a, b);
    const float t0 = fmaxf(fmaxf(__fsub_rn(a[0], bhi[0]), __fsub_rn(blo[0], b[0])), 0.0f);
    const float t1 = fmaxf(fmaxf(__fsub_rn(a[1], bhi[1]), __fsub_rn(blo[1], b[1])), 0.0f);
    const float t2 = fmaxf(fmaxf(__fsub_rn(a[2], bhi[2]), __fsub_rn(blo[2], b[2])), 0.0f);
    return __fmaf_rn(t2, t2, __fmaf_rn(t1, t1, __fmul_rn(t0, t0))) <= R2;
}

// point-box form of eq. 2: is the candidate within the padded radius of the group's box
__device__ __forceinline__ bool point_in_reach(const float4 p, const float blo[3], const float bhi[3], float R2) {
    const float e0 = fmaxf(fmaxf(__fsub_rn(blo[0], p.x), __fsub_rn(p.x, bhi[0])), 0.0f);
    const float e1 = fmaxf(fmaxf(__fsub_rn(blo[1], p.y), __fsub_rn(p.y, bhi[1])), 0.0f);
    const float e2 = fmaxf(fmaxf(__fsub_rn(blo[2], p.z), __fsub_rn(p.z, bhi[2])), 0.0f);
    return __fmaf_rn(e2, e2, __fmaf_rn(e1, e1, __fmul_rn(e0, e0))) <= R2;
}

// WS: collapsed leaves are gathered in fixed slots of WS lanes each (WS >= K, 32 / WS leaves per batch, two batches
// per step so that two 16-byte position loads per lane are in flight).
template <bool STATS, int WS, bool F64>
__global__ void __launch_bounds__(GW_WARPS * 32) traverse_group_kernel(TraverseParams P, const int4 *__restrict__ nodes,
                                                                        const float4 *__restrict__ sorted_pos,
                                                                        const Pos64 *__restrict__ sorted_pos64,
                                                                        const uint2 *__restrict__ groups,
                                                                        const int32_t *__restrict__ entry,
                                                                        TreeMeta *__restrict__ meta,
                                                                        int32_t *__restrict__ nlist,
                                                                        int32_t *__restrict__ n_neigh) {
    __shared__ GwShared s_all[GW_WARPS];
    __shared__ int32_t s_tp[GW_WARPS][F64 ? GW_TILE : 1];   // fp64 only: sorted position of every candidate in the tile ring
    // what every group reads of the build's bookkeeping, fetched once per block: a group's set-up is a chain of
    // dependent loads (group record -> positions -> entry cells -> nodes); these would add links to it
    __shared__ MetaCache mc;
    if (threadIdx.x < QBVH_TMAX) {
        const int t = threadIdx.x;
        mc.seg[t + 1] = meta->seg[t + 1];
        if (t == 0) mc.seg[0] = meta->seg[0];
        const int root = meta->roots[t];
        mc.roots[t] = root;
        mc.gmax[t] = meta->gmax[t];
#pragma unroll
        for (int d = 0; d < 3; ++d) mc.flo[t][d] = meta->frames[t][d], mc.fdl[t][d] = meta->frames[t][6 + d];
        mc.rootnode[t] = root >= 0 ? __ldg(nodes + root) : make_int4(0, 0, 0, 0);
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t FULL = 0xFFFFFFFFu;
    const uint32_t lt_mask = (1u << lane) - 1u;
    GwShared &sm = s_all[warp];
    int32_t *const myring = static_cast<int32_t *>(__builtin_assume_aligned(sm.ring[lane], GW_RING_BYTES));
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(myring);   // aligned to the ring size
    const uint32_t tile_s = (uint32_t)__cvta_generic_to_shared(sm.tx);    // tx, ty, tz, ti follow one another
    // every lane's ring starts at another quad, so that lanes filling at the same pace hit different banks
    const uint32_t rot = (uint32_t)(lane & 7) << 4;
    const int ngroups = meta->group_count;
    const bool vec_ok = ((P.max_neigh & 3) == 0) && ((reinterpret_cast<uintptr_t>(nlist) & 15) == 0);
    const bool vec256_ok = ((P.max_neigh & 7) == 0) && ((reinterpret_cast<uintptr_t>(nlist) & 31) == 0);
    const int cap = P.max_neigh;
    constexpr int NL = 32 / WS;                 // leaves per gather batch
    constexpr int CHUNK = GW_RING >= 64 ? 32 : 16;   // candidates checked between two looks at the ring fill
    const int li = lane / WS, sub = lane % WS;
    unsigned long long st_tests = 0, st_leaf = 0, st_cand = 0, st_checks = 0, st_steps = 0, st_groups = 0;
    int wmax = 0;
    bool bound_violated = false;

    while (true) {
        int g = 0;
        if (lane == 0) g = atomicAdd(&meta->group_cursor, 1);
        g = __shfl_sync(FULL, g, 0);
        if (g >= ngroups) break;
        const uint2 grp = __ldg(groups + g);
        const int gfirst = (int)grp.x, gcnt = (int)grp.y;
        // query sharding (qbvh_neighbors_range): only the particles at sorted positions [q_first, q_first + q_count)
        // are queries; the other members of a group that straddles the edge stay candidates
        if (P.q_count >= 0 && (gfirst + gcnt <= P.q_first || gfirst >= P.q_first + P.q_count)) continue;
        const bool member = lane < gcnt;
        const bool live = member && (P.q_count < 0 || (unsigned)(gfirst + lane - P.q_first) < (unsigned)P.q_count);
        const float4 me = member ? __ldg(sorted_pos + gfirst + lane) : make_float4(0.f, 0.f, 0.f, 0.f);
        const int orig_i = member ? __float_as_int(me.w) : -1;
        const int row_i = P.q_count < 0 ? orig_i : gfirst + lane - P.q_first;   // row of the list this lane writes
        int ta = 0;
#pragma unroll
        for (int t = 1; t < QBVH_TMAX; ++t) ta += (gfirst >= mc.seg[t]) ? 1 : 0;
        const bool aligned = mc.gmax[ta] >= P.K;   // groups are unions of collapsed leaves (the normal case)
        // bounding box of the group (exact fp32 min / max of its members)
        float glo[3], ghi[3];
        {
            const float v[3] = {me.x, me.y, me.z};
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                glo[d] = ord2f(~__reduce_max_sync(FULL, live ? ~f2ord(v[d]) : 0u));
                ghi[d] = ord2f(__reduce_max_sync(FULL, live ? f2ord(v[d]) : 0u));
            }
        }
        int32_t *const row = nlist + (size_t)(live ? row_i : 0) * (size_t)cap;
        const u64 nmx = pk2(-me.x, -me.x), nmy = pk2(-me.y, -me.y), nmz = pk2(-me.z, -me.z);
        uint32_t po = rot;               // ring byte offset: rot + 4 x neighbors found so far for this lane's particle
        int flushed = 0;                 // neighbors already written to the list row (a multiple of 8)
        int thead = 0, tcount = 0;       // candidate tile ring: first slot (a multiple of 32), number of candidates
        if (STATS) ++st_groups;

        // Lanes write their complete 32-byte blocks (one sector, one 256-bit store) of staged neighbors to their list
        // rows.  Called when SOME lane runs out of ring space; EVERY lane with a complete block joins in, so the lanes
        // stay in step and a visit serves most of them (a visit per lane and block cost 3x the instructions).  The lane
        // that triggered the visit holds two blocks, most others one: both leave in the same straight-line pass; what
        // is left after it (a third block, a row at its capacity, an unaligned list) takes the general loop.
        auto flush_blocks = [&]() {
            if (vec256_ok) {
#pragma unroll
                for (int b = 0; b < 2; ++b) {
                    if ((int)((po - rot) >> 2) - flushed >= 8 && flushed + 8 <= cap) {
                        const uint32_t off = rot + 4u * (uint32_t)flushed;
                        const int4 v0 = ring_get4(ring_s, off), v1 = ring_get4(ring_s, off + 16u);
                        st_global_256(row + flushed, v0, v1);
                        flushed += 8;
                    }
                }
            }
            while (__any_sync(FULL, (int)((po - rot) >> 2) - flushed >= 8)) {
                if ((int)((po - rot) >> 2) - flushed >= 8) {
                    const uint32_t off = rot + 4u * (uint32_t)flushed;
                    const int4 v0 = ring_get4(ring_s, off), v1 = ring_get4(ring_s, off + 16u);
                    if (vec_ok && flushed + 8 <= cap) {           // two aligned 128-bit stores
                        int4 *dst = reinterpret_cast<int4 *>(row + flushed);
                        dst[0] = v0;
                        dst[1] = v1;
                    } else {
                        store4(row, flushed, cap, false, v0);
                        store4(row, flushed + 4, cap, false, v1);
                    }
                    flushed += 8;
                }
            }
        };

        for (int tb = 0; tb < QBVH_TMAX; ++tb) {
            const int root = mc.roots[tb];
            if (root < 0) continue;
            const float r2u = P.r2[ta * QBVH_TMAX + tb];
            if (!(r2u >= 0.0f)) continue;
            const float r2 = live ? r2u : -1.0f;          // idle lanes never accept
            const float R2 = P.R2[ta * QBVH_TMAX + tb];
            const float Rp = P.Rp[ta * QBVH_TMAX + tb];
            const float flo[3] = {mc.flo[tb][0], mc.flo[tb][1], mc.flo[tb][2]};
            const float fdl[3] = {mc.fdl[tb][0], mc.fdl[tb][1], mc.fdl[tb][2]};
            const int seg_end = mc.seg[tb + 1];
            const int32_t *const etab = entry + tb * ENTRY_CELLS;
            F64Ctx fx;
            if (F64) {
                fx.sp64 = sorted_pos64, fx.tp = s_tp[warp], fx.ksort_i = gfirst + (member ? lane : 0);
                fx.r2_64 = P.r2_64[ta * QBVH_TMAX + tb], fx.r2lo = live ? P.r2lo[ta * QBVH_TMAX + tb] : -1.0f;   // idle lanes never accept
            }
            // ---- Alg. 1 line 4: lane j tests image j of the group box against the root node; the vote is the bitset ----
            uint32_t bset;
            {
                const int4 nd = mc.rootnode[tb];
                const int sh[3] = {lane % 3 - 1, (lane / 3) % 3 - 1, lane / 9 - 1};
                float lo_s[3], hi_s[3];
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const float sL = (float)sh[d] * P.L[d];
                    lo_s[d] = __fadd_rn(glo[d], sL);
                    hi_s[d] = __fadd_rn(ghi[d], sL);
                }
                bset = __ballot_sync(FULL, lane < 27 && node_overlaps(nd, flo, fdl, lo_s, hi_s, R2));
            }
            while (bset) {                                    // lines 5-9
                const int img = __ffs(bset) - 1;
                bset &= bset - 1;
                const bool shifted = img != 13;
                const float s0 = (float)(img % 3 - 1) * P.L[0], s1 = (float)((img / 3) % 3 - 1) * P.L[1],
                            s2 = (float)(img / 9 - 1) * P.L[2];
                const float blo[3] = {__fadd_rn(glo[0], s0), __fadd_rn(glo[1], s1), __fadd_rn(glo[2], s2)};
                const float bhi[3] = {__fadd_rn(ghi[0], s0), __fadd_rn(ghi[1], s1), __fadd_rn(ghi[2], s2)};
                if (F64) fx.s0 = (double)(img % 3 - 1) * P.L64[0], fx.s1 = (double)((img / 3) % 3 - 1) * P.L64[1], fx.s2 = (double)(img / 9 - 1) * P.L64[2];
                // the group's own particles are found by the walk only here: in its own tree, unshifted.  They are
                // checked first, as one tile (self excluded by index), and their leaves are skipped below.
                // (A sparse type has groups smaller than the collapsed leaves, meta->gmax < K: then a leaf may hold the
                // group and strangers; nothing is skipped and every tile of this image excludes self by index.)
                const bool own_image = (tb == ta) && !shifted;
                const bool own_tree = own_image && aligned, self_all = own_image && !aligned;
                if (own_tree) {
                    sm.tx[lane] = member ? me.x : __int_as_float(0x7FC00000);   // NaN: never accepted
                    sm.ty[lane] = me.y;
                    sm.tz[lane] = me.z;
                    sm.ti[lane] = orig_i;
                    if (F64) s_tp[warp][lane] = gfirst + lane;
                    __syncwarp();
#pragma unroll 1
                    for (int h = 0; h < 32 / CHUNK; ++h) {
                        check_tile<false, true, CHUNK, F64>(sm, tile_s, CHUNK * h, nmx, nmy, nmz, 0ull, 0ull, 0ull, r2, orig_i, ring_s, po, fx);
                        if (__any_sync(FULL, (int)((po - rot) >> 2) - flushed >= GW_RING - CHUNK)) flush_blocks();
                    }
                    if (STATS) st_checks += (unsigned long long)gcnt * (unsigned)gcnt;
                    __syncwarp();
                    thead = 0;
                    tcount = 0;
                }

                // ---- line 9, "n <- root node": enter at the finest Morton grid whose cells touched by the search
                //      volume number at most 32 (one per lane); the root itself if even the 4^3 grid has more ----
                int node = -1;
                {
                    int c0[3], nc[3], lvl = -1;
                    int b0[3], b1[3];
#pragma unroll
                    for (int d = 0; d < 3; ++d) {
                        b0[d] = bin_of(__fsub_rd(blo[d], Rp), P.box_lo[d], P.scale[d]);
                        b1[d] = bin_of(__fadd_ru(bhi[d], Rp), P.box_lo[d], P.scale[d]);
                    }
#pragma unroll
                    for (int l = ENTRY_LMAX; l >= ENTRY_LMIN; --l) {
                        if (lvl < 0) {
                            const int n0 = (b1[0] >> (10 - l)) - (b0[0] >> (10 - l)) + 1;
                            const int n1 = (b1[1] >> (10 - l)) - (b0[1] >> (10 - l)) + 1;
                            const int n2 = (b1[2] >> (10 - l)) - (b0[2] >> (10 - l)) + 1;
                            if (n0 * n1 * n2 <= 32) {
                                lvl = l;
                                nc[0] = n0, nc[1] = n1, nc[2] = n2;
                                c0[0] = b0[0] >> (10 - l), c0[1] = b0[1] >> (10 - l), c0[2] = b0[2] >> (10 - l);
                            }
                        }
                    }
                    if (lvl < 0) {
                        if (lane == 0) node = root;
                    } else if (lane < nc[0] * nc[1] * nc[2]) {
                        // lane -> (ix, iy, iz); quotients of integers below 32 through a float reciprocal (exact: the
                        // true quotient of lane + 0.5 is at least 1/64 away from an integer)
                        const int qy = (int)(((float)lane + 0.5f) * __frcp_rn((float)nc[0]));           // lane / nc0
                        const int iz = (int)(((float)qy + 0.5f) * __frcp_rn((float)nc[1]));             // lane / (nc0 nc1)
                        const int ix = lane - qy * nc[0], iy = qy - iz * nc[1];
                        const uint32_t cell = (spread5((uint32_t)(c0[0] + ix)) << 2) | (spread5((uint32_t)(c0[1] + iy)) << 1) |
                                              spread5((uint32_t)(c0[2] + iz));
                        node = __ldg(etab + entry_offset(lvl) + (int)cell);
                    }
                }
                int wsz;
                {
                    // a range leaf larger than the cells of this level roots several of them: keep one copy
                    if (__match_any_sync(FULL, node) & lt_mask) node = -1;
                    const uint32_t eb = __ballot_sync(FULL, node >= 0);
                    if (node >= 0) sm.wl[__popc(eb & lt_mask)] = (uint32_t)node;
                    wsz = __popc(eb);
                }
                __syncwarp();
                int lqn = 0;                           // leaf queue fill

                while (true) {
                    if (tcount >= 32) {
                        // ---- line 14 for every member: one tile of 32 candidates ----
#pragma unroll 1
                        for (int h = 0; h < 32 / CHUNK; ++h) {
                            if (shifted)   // (the packed shift is formed here: nothing of it is live on the unshifted path)
                                check_tile<true, false, CHUNK, F64>(sm, tile_s, thead + CHUNK * h, nmx, nmy, nmz, pk2(-s0, -s0), pk2(-s1, -s1), pk2(-s2, -s2), r2, orig_i, ring_s, po, fx);
                            else if (self_all)
                                check_tile<false, true, CHUNK, F64>(sm, tile_s, thead + CHUNK * h, nmx, nmy, nmz, 0ull, 0ull, 0ull, r2, orig_i, ring_s, po, fx);
                            else
                                check_tile<false, false, CHUNK, F64>(sm, tile_s, thead + CHUNK * h, nmx, nmy, nmz, 0ull, 0ull, 0ull, r2, orig_i, ring_s, po, fx);
                            // flush as soon as another chunk could overrun a ring
                            if (__any_sync(FULL, (int)((po - rot) >> 2) - flushed >= GW_RING - CHUNK)) flush_blocks();
                        }
                        if (STATS) st_checks += 32ull * (unsigned)gcnt;
                        __syncwarp();
                        thead = (thead + 32) & (GW_TILE - 1);
                        tcount -= 32;
                        continue;
                    }
                    if (wsz > 0 && lqn <= GW_LQ - 64) {   // (room for the 64 leaves a step can emit)
                        // ---- lines 10-19, up to 64 nodes per step: every lane pops one entry and tests that node
                        //      and, for a left child, its rope (= right sibling) as well ----
                        const int npop = (wsz > GW_WL - 96) ? 1 : min(wsz, 32);
                        int pushA = 0, pushB = 0, emitA = 0, emitB = 0, pairf = 0;
                        int4 A = make_int4(0, 0, 0, 0), B = make_int4(0, 0, 0, 0);
                        if (lane < npop) {
                            const uint32_t ent = sm.wl[wsz - 1 - lane];
                            const int ia = (int)(ent & 0x7FFFFFFFu);
                            A = __ldg(nodes + ia);
                            if (ent >> 31) {
                                // A is a left child; its rope is its right sibling: internal node gamma + 1 or leaf
                                // gamma + 1 (SURVEY.md B.1 numbering).  Load both without waiting for A.
                                pairf = 1;
                                const int gam = ia < P.N - 1 ? ia : ia - (P.N - 1);
                                const int4 B1 = __ldg(nodes + gam + 1), B2 = __ldg(nodes + P.N + gam);
                                B = (A.w == gam + 1) ? B1 : B2;
                            }
                            const bool hitA = node_overlaps(A, flo, fdl, blo, bhi, R2);
                            pushA = hitA && A.z >= 0;
                            // leaves inside the group itself were handled above
                            emitA = hitA && A.z < 0 && !(own_tree && (unsigned)(~A.z - gfirst) < (unsigned)gcnt);
                            if (pairf) {
                                const bool hitB = node_overlaps(B, flo, fdl, blo, bhi, R2);
                                pushB = hitB && B.z >= 0;
                                emitB = hitB && B.z < 0 && !(own_tree && (unsigned)(~B.z - gfirst) < (unsigned)gcnt);
                            }
                        }
                        __syncwarp();                             // all reads of the list done before it is rewritten
                        const uint32_t pa = __ballot_sync(FULL, pushA), pb = __ballot_sync(FULL, pushB);
                        const uint32_t ea = __ballot_sync(FULL, emitA), eb = __ballot_sync(FULL, emitB);
                        const int base = wsz - npop;
                        // Bound of the work list: up to 160 entries a step pops <= 32 and pushes <= 64
                        // (wsz <= 192); above 160 it pops ONE entry and pushes <= 2, a depth-first descent that can
                        // grow the list by at most the depth of the tree below that entry (<= 60 levels: 30 code bits
                        // + 30 index bits) => wsz <= 252 < GW_WL.  The guard makes a violated bound an error, never
                        // an out-of-bounds write.
                        const int nw = base + __popc(pa) + __popc(pb);
                        const bool fits = nw <= GW_WL;
                        if (pushA && fits) sm.wl[base + __popc(pa & lt_mask)] = (uint32_t)A.z | 0x80000000u;
                        if (pushB && fits) sm.wl[base + __popc(pa) + __popc(pb & lt_mask)] = (uint32_t)B.z | 0x80000000u;
                        wsz = fits ? nw : base;
                        bound_violated |= !fits;
                        if (emitA) sm.lq[lqn + __popc(ea & lt_mask)] = make_uint2((uint32_t)(~A.z), (uint32_t)leaf_count(A, P.N, seg_end));
                        if (emitB)
                            sm.lq[lqn + __popc(ea) + __popc(eb & lt_mask)] = make_uint2((uint32_t)(~B.z), (uint32_t)leaf_count(B, P.N, seg_end));
                        lqn += __popc(ea) + __popc(eb);
                        if (STATS) {
                            st_tests += npop + __popc(__ballot_sync(FULL, pairf));
                            st_leaf += __popc(ea) + __popc(eb);
                            ++st_steps;
                        }
                        __syncwarp();
                        continue;
                    }
                    if (lqn > 0) {
                        // ---- gather up to GW_NB x 32/WS leaves: lane j takes particle j % WS of leaf j / WS of each batch (a
                        //      collapsed leaf has at most K <= WS particles); keep those within reach of the group box.
                        //      All position loads of the step are issued before the first is used ----
                        const int take = min(lqn, GW_NB * NL);
                        uint2 lf[GW_NB];
                        float4 pc[GW_NB];
                        bool keep[GW_NB];
#pragma unroll
                        for (int u = 0; u < GW_NB; ++u) {
                            lf[u] = make_uint2(0u, 0u);
                            if (u * NL + li < take) lf[u] = sm.lq[lqn - 1 - u * NL - li];
                        }
                        lqn -= take;
                        // lanes past the end of their leaf load its first particle instead (no branch) and drop it
#pragma unroll
                        for (int u = 0; u < GW_NB; ++u)
                            pc[u] = __ldg(sorted_pos + (lf[u].x + (sub < (int)lf[u].y ? (uint32_t)sub : 0u)));
                        int nkept = 0;
#pragma unroll
                        for (int u = 0; u < GW_NB; ++u) {
                            keep[u] = point_in_reach(pc[u], blo, bhi, R2) & (sub < (int)lf[u].y);   // (no short circuit: no branch)
                            const uint32_t kb = __ballot_sync(FULL, keep[u]);
                            if (keep[u]) {
                                const int slot = (thead + tcount + nkept + __popc(kb & lt_mask)) & (GW_TILE - 1);
                                sm.tx[slot] = pc[u].x;
                                sm.ty[slot] = pc[u].y;
                                sm.tz[slot] = pc[u].z;
                                sm.ti[slot] = __float_as_int(pc[u].w);
                                if (F64) s_tp[warp][slot] = (int32_t)lf[u].x + sub;
                            }
                            nkept += __popc(kb);
                        }
                        tcount += nkept;
                        if (STATS) st_cand += nkept;
                        __syncwarp();
                        continue;
                    }
                    if (tcount > 0) {
                        // ---- the image's last, partial tile: pad with NaN (never accepted) and run it as a full one ----
                        if (lane >= tcount) sm.tx[(thead + lane) & (GW_TILE - 1)] = __int_as_float(0x7FC00000);
                        if (STATS) st_checks -= (unsigned long long)(32 - tcount) * (unsigned)gcnt;
                        tcount = 32;
                        __syncwarp();
                        continue;
                    }
                    break;
                }
            }
        }
        // ---- tail of every row, count, overflow word ----
        flush_blocks();
        {
            const int cnt = (int)((po - rot) >> 2);
            const int rem = cnt - flushed;
            const uint32_t off = rot + 4u * (uint32_t)flushed;
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (4 * j < rem) {
                    const int4 v = ring_get4(ring_s, off + 16u * j);
                    const int o = flushed + 4 * j;
                    if (vec_ok && o + 4 <= cap) {
                        *reinterpret_cast<int4 *>(row + o) = v;    // up to 3 entries past the count: unspecified
                    } else {
                        if (4 * j + 0 < rem && o + 0 < cap) row[o + 0] = v.x;
                        if (4 * j + 1 < rem && o + 1 < cap) row[o + 1] = v.y;
                        if (4 * j + 2 < rem && o + 2 < cap) row[o + 2] = v.z;
                        if (4 * j + 3 < rem && o + 3 < cap) row[o + 3] = v.w;
                    }
                }
            if (live) n_neigh[row_i] = cnt;
            wmax = max(wmax, live ? cnt : 0);
        }
        __syncwarp();
    }
    wmax = __reduce_max_sync(FULL, wmax);
    if (lane == 0 && wmax > 0) atomicMax(&meta->max_count, wmax);
    if (lane == 0 && bound_violated) atomicOr(&meta->err_flags, 2);
    if (P.result_host != nullptr && lane == 0) {
        // The last warp to finish hands the result to the host (a write into pinned memory: no copy behind the
        // kernel) and re-arms the counters for the next traversal of this tree (no memset in front of it).
        __threadfence();
        if (atomicAdd(&meta->warps_done, 1) == (int)(gridDim.x * GW_WARPS) - 1) {
            __threadfence();
            P.result_host[0] = atomicMax(&meta->max_count, 0);
            P.result_host[1] = atomicOr(&meta->err_flags, 0);
            __threadfence_system();
            meta->max_count = 0;
            meta->group_cursor = 0;
            meta->warps_done = 0;
        }
    }
    if (STATS && lane == 0) {
        atomicAdd(&meta->stats[5], st_groups);
        atomicAdd(&meta->stats[6], st_tests);
        atomicAdd(&meta->stats[7], st_leaf);
        atomicAdd(&meta->stats[8], st_cand);
        atomicAdd(&meta->stats[9], st_checks);
        atomicAdd(&meta->stats[10], st_steps);
    }
}

// persistent grid of the group kernel: as many blocks as fit on the device at once
template <bool STATS, int WS, bool F64>
static int group_grid_blocks() {
    static int c = 0;
    if (c == 0) {
        int dev = 0, sms = 148, per_sm = 1;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, traverse_group_kernel<STATS, WS, F64>, GW_WARPS * 32, 0);
        c = sms * (per_sm > 0 ? per_sm : 1);
    }
    return c;
}

template <bool STATS, int WS, bool F64>
static void launch_group(const TraverseParams &p, const BuildBuffers &b, int32_t *nlist, int32_t *n_neigh, cudaStream_t st) {
    const int gb = min(group_grid_blocks<STATS, WS, F64>(), (p.N + GW_WARPS - 1) / GW_WARPS);
    traverse_group_kernel<STATS, WS, F64><<<gb, GW_WARPS * 32, 0, st>>>(p, b.nodes, b.sorted_pos, b.sorted_pos64, b.groups, b.entry, b.meta, nlist, n_neigh);
}
template <bool STATS, int WS>
static void launch_group_p(const TraverseParams &p, const BuildBuffers &b, int32_t *nlist, int32_t *n_neigh, bool f64, cudaStream_t st) {
    if (f64) launch_group<STATS, WS, true>(p, b, nlist, n_neigh, st);
    else launch_group<STATS, WS, false>(p, b, nlist, n_neigh, st);
}

// warps the production traversal keeps resident (the build sizes query groups of small systems by it)
int traverse_warp_slots() { return group_grid_blocks<false, 32, false>() * GW_WARPS; }

cudaError_t launch_traverse(const TraverseParams &p, const BuildBuffers &b, int32_t *nlist, int32_t *n_neigh,
                            bool stats, int variant, bool f64, cudaStream_t st) {
    if (p.N == 0) return cudaSuccess;
    const int threads = 128;
    const int blocks = (p.N + threads - 1) / threads;
    if (variant == 0) {
        // Algorithm 1 as written: one thread per particle
        if (stats)
            traverse_kernel<true><<<blocks, threads, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh);
        else
            traverse_kernel<false><<<blocks, threads, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh);
        return cudaGetLastError();
    }
    const int ws = p.K > 16 ? 32 : (p.K > 8 ? 16 : 8);
    if (stats) {
        // census of the paper's per-particle walk (stats[0..4]), then the instrumented production kernel
        traverse_kernel<true><<<blocks, threads, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh);
        cudaError_t e = cudaMemsetAsync(&b.meta->group_cursor, 0, 2 * sizeof(int32_t), st);
        if (e != cudaSuccess) return e;
        if (ws == 32) launch_group_p<true, 32>(p, b, nlist, n_neigh, f64, st);
        else if (ws == 16) launch_group_p<true, 16>(p, b, nlist, n_neigh, f64, st);
        else launch_group_p<true, 8>(p, b, nlist, n_neigh, f64, st);
    } else {
        if (ws == 32) launch_group_p<false, 32>(p, b, nlist, n_neigh, f64, st);
        else if (ws == 16) launch_group_p<false, 16>(p, b, nlist, n_neigh, f64, st);
        else launch_group_p<false, 8>(p, b, nlist, n_neigh, f64, st);
    }
    return cudaGetLastError();
}

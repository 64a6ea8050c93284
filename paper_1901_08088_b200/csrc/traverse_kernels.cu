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

__device__ __forceinline__ void decompress(uint32_t wlo, uint32_t whi, const float lo[3], const float dl[3],
                                           float a[3], float b[3]) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        a[d] = __fmaf_rd((float)((wlo >> (10 * d)) & 1023u), dl[d], lo[d]);
        b[d] = __fmaf_ru((float)((whi >> (10 * d)) & 1023u), dl[d], lo[d]);
    }
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
                            const int m = (P.K > 1) ? 1 + (int)(((uint32_t)nd.x >> 30) | (((uint32_t)nd.y >> 30) << 2)) : 1;
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

constexpr int GW_WARPS = 4;      // warps per block
constexpr int GW_WL = 512;       // work-list entries per warp
constexpr int GW_LQ = 64;        // leaf-queue entries per warp
constexpr int GW_TILE = 64;      // candidate tile ring per warp: two halves of 32
constexpr int GW_RING = 32;      // staged neighbors per lane: two blocks of 16

struct __align__(128) GwShared {
    float tx[GW_TILE], ty[GW_TILE], tz[GW_TILE];   // candidate tile, structure of arrays
    int32_t ti[GW_TILE];                           // original particle index of each candidate
    int32_t ring[32][GW_RING];                     // per-lane staged neighbors
    uint32_t wl[GW_WL];                            // work list: node id | (is a left child) << 31
    uint2 lq[GW_LQ];                               // leaf queue: {first sorted position, count}
};

// append one neighbor to this lane's ring: slot address = ring base | (byte offset mod 128), one LOP3
__device__ __forceinline__ void ring_put(uint32_t ring_s, uint32_t &po, int32_t v) {
    *static_cast<int32_t *>(__cvta_shared_to_generic((size_t)(ring_s | (po & (4 * GW_RING - 4))))) = v;
    po += 4;
}

// 16 candidates of the tile, starting at `base`, against this lane's particle: the canonical predicate
//   D = (p_j - p_i) [- s L];  d2 = fma(Dz, Dz, fma(Dy, Dy, Dx*Dx));  d2 <= r^2
// evaluated for two candidates per instruction.  SELF: the tile may hold members of the group itself.
template <bool SHIFTED, bool SELF>
__device__ __forceinline__ void check16(const GwShared &sm, int base, u64 nmx, u64 nmy, u64 nmz, u64 ns0, u64 ns1,
                                        u64 ns2, float r2, int orig_i, uint32_t ring_s, uint32_t &po) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float4 X = *reinterpret_cast<const float4 *>(&sm.tx[base + 4 * j]);
        const float4 Y = *reinterpret_cast<const float4 *>(&sm.ty[base + 4 * j]);
        const float4 Z = *reinterpret_cast<const float4 *>(&sm.tz[base + 4 * j]);
        const int4 I = *reinterpret_cast<const int4 *>(&sm.ti[base + 4 * j]);
        u64 dx0 = add2(pk2(X.x, X.y), nmx), dx1 = add2(pk2(X.z, X.w), nmx);
        u64 dy0 = add2(pk2(Y.x, Y.y), nmy), dy1 = add2(pk2(Y.z, Y.w), nmy);
        u64 dz0 = add2(pk2(Z.x, Z.y), nmz), dz1 = add2(pk2(Z.z, Z.w), nmz);
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
        if (d0 <= r2 && (!SELF || I.x != orig_i)) { ring_put(ring_s, po, I.x); }
        if (d1 <= r2 && (!SELF || I.y != orig_i)) { ring_put(ring_s, po, I.y); }
        if (d2 <= r2 && (!SELF || I.z != orig_i)) { ring_put(ring_s, po, I.z); }
        if (d3 <= r2 && (!SELF || I.w != orig_i)) { ring_put(ring_s, po, I.w); }
    }
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

template <bool STATS>
__global__ void __launch_bounds__(GW_WARPS * 32) traverse_group_kernel(TraverseParams P, const int4 *__restrict__ nodes,
                                                                        const float4 *__restrict__ sorted_pos,
                                                                        const uint2 *__restrict__ groups,
                                                                        TreeMeta *__restrict__ meta,
                                                                        int32_t *__restrict__ nlist,
                                                                        int32_t *__restrict__ n_neigh) {
    __shared__ GwShared s_all[GW_WARPS];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t FULL = 0xFFFFFFFFu;
    const uint32_t lt_mask = (1u << lane) - 1u;
    GwShared &sm = s_all[warp];
    int32_t *const myring = static_cast<int32_t *>(__builtin_assume_aligned(sm.ring[lane], 128));
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(myring);   // 128-byte aligned
    const int ngroups = meta->group_count;
    const bool vec_ok = ((P.max_neigh & 3) == 0) && ((reinterpret_cast<uintptr_t>(nlist) & 15) == 0);
    const int cap = P.max_neigh;
    unsigned long long st_tests = 0, st_leaf = 0, st_cand = 0, st_checks = 0, st_steps = 0, st_groups = 0;
    int wmax = 0;

    while (true) {
        int g = 0;
        if (lane == 0) g = atomicAdd(&meta->group_cursor, 1);
        g = __shfl_sync(FULL, g, 0);
        if (g >= ngroups) break;
        const uint2 grp = __ldg(groups + g);
        const int gfirst = (int)grp.x, gcnt = (int)grp.y;
        const bool live = lane < gcnt;
        const float4 me = live ? __ldg(sorted_pos + gfirst + lane) : make_float4(0.f, 0.f, 0.f, 0.f);
        const int orig_i = live ? __float_as_int(me.w) : -1;
        int ta = 0;
#pragma unroll
        for (int t = 1; t < QBVH_TMAX; ++t) ta += (gfirst >= meta->seg[t]) ? 1 : 0;
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
        int32_t *const row = nlist + (size_t)(live ? orig_i : 0) * (size_t)cap;
        const u64 nmx = pk2(-me.x, -me.x), nmy = pk2(-me.y, -me.y), nmz = pk2(-me.z, -me.z);
        uint32_t po = 0;                 // 4 x neighbors found so far for this lane's particle (ring byte offset)
        int flushed = 0;                 // neighbors already written to the list row
        int thead = 0, tcount = 0;       // candidate tile ring: first slot (0 or 32), number of candidates
        if (STATS) ++st_groups;

        // lanes holding a complete 64-byte block of staged neighbors write it to their list row
        auto flush_blocks = [&]() {
            if ((int)(po >> 2) - flushed >= 16) {
                const int32_t *src = myring + (flushed & (GW_RING - 1));
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    store4(row, flushed + 4 * j, cap, vec_ok, *reinterpret_cast<const int4 *>(src + 4 * j));
                flushed += 16;
            }
        };

        for (int tb = 0; tb < QBVH_TMAX; ++tb) {
            const int root = meta->roots[tb];
            if (root < 0) continue;
            const float r2u = P.r2[ta * QBVH_TMAX + tb];
            if (!(r2u >= 0.0f)) continue;
            const float r2 = live ? r2u : -1.0f;          // idle lanes never accept
            const float R2 = P.R2[ta * QBVH_TMAX + tb];
            const float *fr = meta->frames[tb];
            const float flo[3] = {fr[0], fr[1], fr[2]};
            const float fdl[3] = {fr[6], fr[7], fr[8]};
            // ---- Alg. 1 line 4: lane j tests image j of the group box against the root node; the vote is the bitset ----
            uint32_t bset;
            {
                const int4 nd = __ldg(nodes + root);
                float a[3], b[3];
                decompress((uint32_t)nd.x, (uint32_t)nd.y, flo, fdl, a, b);
                const int sh[3] = {lane % 3 - 1, (lane / 3) % 3 - 1, lane / 9 - 1};
                float tq[3];
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const float sL = (float)sh[d] * P.L[d];
                    const float lo_s = __fadd_rn(glo[d], sL), hi_s = __fadd_rn(ghi[d], sL);
                    tq[d] = fmaxf(fmaxf(__fsub_rn(a[d], hi_s), __fsub_rn(lo_s, b[d])), 0.0f);
                }
                const float d2 = __fmaf_rn(tq[2], tq[2], __fmaf_rn(tq[1], tq[1], __fmul_rn(tq[0], tq[0])));
                bset = __ballot_sync(FULL, lane < 27 && d2 <= R2);
            }
            while (bset) {                                    // lines 5-9
                const int img = __ffs(bset) - 1;
                bset &= bset - 1;
                const bool shifted = img != 13;
                const float s0 = (float)(img % 3 - 1) * P.L[0], s1 = (float)((img / 3) % 3 - 1) * P.L[1],
                            s2 = (float)(img / 9 - 1) * P.L[2];
                const float blo[3] = {__fadd_rn(glo[0], s0), __fadd_rn(glo[1], s1), __fadd_rn(glo[2], s2)};
                const float bhi[3] = {__fadd_rn(ghi[0], s0), __fadd_rn(ghi[1], s1), __fadd_rn(ghi[2], s2)};
                const u64 ns0 = pk2(-s0, -s0), ns1 = pk2(-s1, -s1), ns2 = pk2(-s2, -s2);
                const bool own_tree = (tb == ta) && !shifted;   // only then can a candidate be a group member

                if (lane == 0) sm.wl[0] = (uint32_t)root;
                __syncwarp();
                int wsz = 1, lqn = 0;                  // work list and leaf queue fill
                int gt = 0, gmax = 0, gfirst_l = 0, gm_l = 0;   // gather in progress: iteration, bound, my leaf
                int tapp = 0, tproc = 0;               // candidates appended to / consumed from the tile (this image)
                int self_lo = 0x7FFFFFFF, self_hi = -1;   // span of appended candidates that are group members

                while (true) {
                    if (tcount >= 32) {
                        // ---- line 14 for every member: one tile of 32 candidates, as two halves of 16 ----
#pragma unroll 1
                        for (int h = 0; h < 2; ++h) {
                            if (__any_sync(FULL, (int)(po >> 2) - flushed >= 16)) flush_blocks();
                            const int base = thead + 16 * h, a0 = tproc + 16 * h;
                            if (shifted)
                                check16<true, false>(sm, base, nmx, nmy, nmz, ns0, ns1, ns2, r2, orig_i, ring_s, po);
                            else if (a0 < self_hi && a0 + 16 > self_lo)
                                check16<false, true>(sm, base, nmx, nmy, nmz, ns0, ns1, ns2, r2, orig_i, ring_s, po);
                            else
                                check16<false, false>(sm, base, nmx, nmy, nmz, ns0, ns1, ns2, r2, orig_i, ring_s, po);
                        }
                        if (STATS) st_checks += 32ull * (unsigned)gcnt;
                        __syncwarp();
                        thead ^= 32;
                        tcount -= 32;
                        tproc += 32;
                        continue;
                    }
                    if (gt < gmax) {
                        // ---- gather: particle gt of every lane's leaf; keep those within reach of the group box ----
                        const bool valid = gt < gm_l;
                        float4 pj = make_float4(0.f, 0.f, 0.f, 0.f);
                        bool keep = false;
                        if (valid) {
                            pj = __ldg(sorted_pos + gfirst_l + gt);
                            const float e0 = fmaxf(fmaxf(__fsub_rn(blo[0], pj.x), __fsub_rn(pj.x, bhi[0])), 0.0f);
                            const float e1 = fmaxf(fmaxf(__fsub_rn(blo[1], pj.y), __fsub_rn(pj.y, bhi[1])), 0.0f);
                            const float e2 = fmaxf(fmaxf(__fsub_rn(blo[2], pj.z), __fsub_rn(pj.z, bhi[2])), 0.0f);
                            keep = __fmaf_rn(e2, e2, __fmaf_rn(e1, e1, __fmul_rn(e0, e0))) <= R2;
                        }
                        const uint32_t kb = __ballot_sync(FULL, keep);
                        if (keep) {
                            const int slot = (thead + tcount + __popc(kb & lt_mask)) & (GW_TILE - 1);
                            sm.tx[slot] = pj.x;
                            sm.ty[slot] = pj.y;
                            sm.tz[slot] = pj.z;
                            sm.ti[slot] = __float_as_int(pj.w);
                        }
                        if (own_tree) {
                            const int jj = gfirst_l + gt - gfirst;
                            const uint32_t sb = __ballot_sync(FULL, keep && jj >= 0 && jj < gcnt);
                            if (sb) {
                                const int lo_lane = __ffs(sb) - 1, hi_lane = 31 - __clz(sb);
                                self_lo = min(self_lo, tapp + __popc(kb & ((1u << lo_lane) - 1u)));
                                self_hi = max(self_hi, tapp + __popc(kb & ((2u << hi_lane) - 1u)));
                            }
                        }
                        const int nk = __popc(kb);
                        tcount += nk;
                        tapp += nk;
                        if (STATS) st_cand += nk;
                        ++gt;
                        __syncwarp();
                        continue;
                    }
                    if (lqn >= 32 || (wsz == 0 && lqn > 0)) {
                        // ---- start a gather: the newest (up to) 32 queued leaves, one per lane ----
                        const int ng = min(lqn, 32);
                        lqn -= ng;
                        gm_l = 0;
                        if (lane < ng) {
                            const uint2 q = sm.lq[lqn + lane];
                            gfirst_l = (int)q.x;
                            gm_l = (int)q.y;
                        }
                        gmax = __reduce_max_sync(FULL, gm_l);
                        gt = 0;
                        __syncwarp();
                        continue;
                    }
                    if (wsz > 0) {
                        // ---- lines 10-19, 32 nodes per step ----
                        const int npop = (wsz > GW_WL - 128) ? 1 : min(wsz, 32);
                        const bool active = lane < npop;
                        bool push_sib = false, push_child = false, emit = false;
                        int4 nd = make_int4(0, 0, 0, 0);
                        if (active) {
                            const uint32_t ent = sm.wl[wsz - 1 - lane];
                            nd = __ldg(nodes + (ent & 0x7FFFFFFFu));
                            float a[3], b[3];
                            decompress((uint32_t)nd.x, (uint32_t)nd.y, flo, fdl, a, b);
                            const float t0 = fmaxf(fmaxf(__fsub_rn(a[0], bhi[0]), __fsub_rn(blo[0], b[0])), 0.0f);
                            const float t1 = fmaxf(fmaxf(__fsub_rn(a[1], bhi[1]), __fsub_rn(blo[1], b[1])), 0.0f);
                            const float t2 = fmaxf(fmaxf(__fsub_rn(a[2], bhi[2]), __fsub_rn(blo[2], b[2])), 0.0f);
                            const float d2 = __fmaf_rn(t2, t2, __fmaf_rn(t1, t1, __fmul_rn(t0, t0)));
                            const bool hit = d2 <= R2;
                            push_sib = (ent >> 31) != 0;          // a left child: its rope is the right sibling
                            push_child = hit && nd.z >= 0;
                            emit = hit && nd.z < 0;
                        }
                        __syncwarp();                             // all reads of the list done before it is rewritten
                        const uint32_t b1 = __ballot_sync(FULL, push_sib);
                        const uint32_t b2 = __ballot_sync(FULL, push_child);
                        const uint32_t b3 = __ballot_sync(FULL, emit);
                        const int base = wsz - npop;
                        if (push_sib) sm.wl[base + __popc(b1 & lt_mask)] = (uint32_t)nd.w;
                        if (push_child) sm.wl[base + __popc(b1) + __popc(b2 & lt_mask)] = (uint32_t)nd.z | 0x80000000u;
                        wsz = base + __popc(b1) + __popc(b2);
                        if (emit) {
                            const uint32_t m = (P.K > 1) ? 1u + (((uint32_t)nd.x >> 30) | (((uint32_t)nd.y >> 30) << 2)) : 1u;
                            sm.lq[lqn + __popc(b3 & lt_mask)] = make_uint2((uint32_t)(~nd.z), m);
                        }
                        lqn += __popc(b3);
                        if (STATS) {
                            st_tests += npop;
                            st_leaf += __popc(b3);
                            ++st_steps;
                        }
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
            const int rem = (int)(po >> 2) - flushed;
            const int32_t *src = myring + (flushed & (GW_RING - 1));
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (4 * j < rem) {
                    const int4 v = *reinterpret_cast<const int4 *>(src + 4 * j);
                    const int off = flushed + 4 * j;
                    if (vec_ok && off + 4 <= cap) {
                        *reinterpret_cast<int4 *>(row + off) = v;    // up to 3 entries past the count: unspecified
                    } else {
                        if (4 * j + 0 < rem && off + 0 < cap) row[off + 0] = v.x;
                        if (4 * j + 1 < rem && off + 1 < cap) row[off + 1] = v.y;
                        if (4 * j + 2 < rem && off + 2 < cap) row[off + 2] = v.z;
                        if (4 * j + 3 < rem && off + 3 < cap) row[off + 3] = v.w;
                    }
                }
        }
        if (live) n_neigh[orig_i] = (int)(po >> 2);
        wmax = max(wmax, live ? (int)(po >> 2) : 0);
        __syncwarp();
    }
    wmax = __reduce_max_sync(FULL, wmax);
    if (lane == 0 && wmax > 0) atomicMax(&meta->max_count, wmax);
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
static int group_grid_blocks(bool stats) {
    static int cached[2] = {0, 0};
    int &c = cached[stats ? 1 : 0];
    if (c == 0) {
        int dev = 0, sms = 148, per_sm = 1;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (stats)
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, traverse_group_kernel<true>, GW_WARPS * 32, 0);
        else
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, traverse_group_kernel<false>, GW_WARPS * 32, 0);
        c = sms * (per_sm > 0 ? per_sm : 1);
    }
    return c;
}

cudaError_t launch_traverse(const TraverseParams &p, const BuildBuffers &b, int32_t *nlist, int32_t *n_neigh,
                            bool stats, int variant, cudaStream_t st) {
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
    if (stats) {
        // census of the paper's per-particle walk (stats[0..4]), then the instrumented production kernel
        traverse_kernel<true><<<blocks, threads, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh);
        cudaError_t e = cudaMemsetAsync(&b.meta->group_cursor, 0, 2 * sizeof(int32_t), st);
        if (e != cudaSuccess) return e;
        const int gb = min(group_grid_blocks(true), (p.N + GW_WARPS - 1) / GW_WARPS);
        traverse_group_kernel<true><<<gb, GW_WARPS * 32, 0, st>>>(p, b.nodes, b.sorted_pos, b.groups, b.meta, nlist, n_neigh);
    } else {
        const int gb = min(group_grid_blocks(false), (p.N + GW_WARPS - 1) / GW_WARPS);
        traverse_group_kernel<false><<<gb, GW_WARPS * 32, 0, st>>>(p, b.nodes, b.sorted_pos, b.groups, b.meta, nlist, n_neigh);
    }
    return cudaGetLastError();
}

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
// v2: the same Algorithm 1 per particle, restructured for SIMT efficiency (ncu on v0: 8 of 32 lanes active on
// average, leaf processing executed with 2-6 active lanes).
//   * image loop and node loop flattened into one loop: a lane that finishes an image pops the next set bit of
//     its bitset and restarts at the root in the same iteration slot (the bitset exists to avoid
//     wasted loop iterations);
//   * a leaf-range hit is not processed in place: (first, count, image, tree) is pushed onto a per-lane queue in
//     shared memory and the walk goes on.  When any lane's queue is full the whole warp leaves the walk and every
//     lane drains its own queue in a flat one-candidate-per-iteration loop (exact predicate);
//   * accepted neighbors are collected four at a time in registers and written with one 16-byte store.
// ------------------------------------------------------------------------------------------------------------
struct RowWriter {
    int32_t *row;
    int cap;       // max_neigh
    int cnt;
    bool vec;      // row is 16-byte aligned and cap % 4 == 0
    int b0, b1, b2, b3;
    __device__ __forceinline__ void push(int v) {
        const int s = cnt & 3;
        if (s == 0) b0 = v;
        else if (s == 1) b1 = v;
        else if (s == 2) b2 = v;
        else b3 = v;
        ++cnt;
        if (s == 3) {
            const int base = cnt - 4;
            if (vec) {
                if (base < cap) *reinterpret_cast<int4 *>(row + base) = make_int4(b0, b1, b2, b3);
            } else {
                if (base + 0 < cap) row[base + 0] = b0;
                if (base + 1 < cap) row[base + 1] = b1;
                if (base + 2 < cap) row[base + 2] = b2;
                if (base + 3 < cap) row[base + 3] = b3;
            }
        }
    }
    __device__ __forceinline__ void finish() {
        const int s = cnt & 3, base = cnt - s;
        if (s > 0 && base + 0 < cap) row[base + 0] = b0;
        if (s > 1 && base + 1 < cap) row[base + 1] = b1;
        if (s > 2 && base + 2 < cap) row[base + 2] = b2;
    }
};

template <int QCAP, int THREADS, bool TEX, int DUMMY = 0>
__global__ void __launch_bounds__(THREADS) traverse_v2_kernel(TraverseParams P, const int4 *__restrict__ nodes,
                                                               const float4 *__restrict__ sorted_pos,
                                                               TreeMeta *__restrict__ meta,
                                                               int32_t *__restrict__ nlist,
                                                               int32_t *__restrict__ n_neigh,
                                                               cudaTextureObject_t tex_nodes,
                                                               cudaTextureObject_t tex_pos) {
    __shared__ uint2 s_q[QCAP][THREADS];   // [slot][thread]: conflict-free 8-byte accesses
    const int k = blockIdx.x * THREADS + threadIdx.x;
    const bool live = k < P.N;
    const float4 me = live ? sorted_pos[k] : make_float4(0.f, 0.f, 0.f, 0.f);
    const int orig_i = __float_as_int(me.w);
    int ta = 0;
#pragma unroll
    for (int t = 1; t < QBVH_TMAX; ++t) ta += (k >= meta->seg[t]) ? 1 : 0;
    RowWriter out;
    out.row = nlist + (size_t)(live ? orig_i : 0) * (size_t)P.max_neigh;
    out.cap = live ? P.max_neigh : 0;
    out.cnt = 0;
    out.vec = ((P.max_neigh & 3) == 0) && ((reinterpret_cast<uintptr_t>(nlist) & 15) == 0);
    out.b0 = out.b1 = out.b2 = out.b3 = 0;
    int fill = 0;

    auto flush = [&]() {
        int e = 0, t = 0, first = 0, m = 0;
        float r2 = 0.f, s0 = 0.f, s1 = 0.f, s2 = 0.f;
        auto load_entry = [&]() {
            if (e < fill) {
                const uint2 q = s_q[e][threadIdx.x];
                first = (int)q.x;
                m = (int)(q.y & 15u) + 1;
                const int img = (int)((q.y >> 4) & 31u);
                const int tb = (int)(q.y >> 9);
                r2 = P.r2[ta * QBVH_TMAX + tb];
                s0 = (float)(img % 3 - 1) * P.L[0];
                s1 = (float)((img / 3) % 3 - 1) * P.L[1];
                s2 = (float)(img / 9 - 1) * P.L[2];
            }
        };
        load_entry();
        while (__any_sync(0xFFFFFFFFu, e < fill)) {
            if (e < fill) {
                const int j = first + t;
                const float4 pj = TEX ? tex1Dfetch<float4>(tex_pos, j) : __ldg(sorted_pos + j);
                const float dx = __fsub_rn(__fsub_rn(pj.x, me.x), s0);
                const float dy = __fsub_rn(__fsub_rn(pj.y, me.y), s1);
                const float dz = __fsub_rn(__fsub_rn(pj.z, me.z), s2);
                const float dd = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                if (dd <= r2 && j != k) out.push(__float_as_int(pj.w));
                if (++t == m) {
                    t = 0;
                    ++e;
                    load_entry();
                }
            }
        }
        fill = 0;
    };

    for (int tb = 0; tb < QBVH_TMAX; ++tb) {
        const int root = meta->roots[tb];
        if (root < 0) continue;                            // warp-uniform
        const float r2q = P.r2[ta * QBVH_TMAX + tb];
        const float R2 = P.R2[ta * QBVH_TMAX + tb];
        const float *fr = meta->frames[tb];
        const float flo[3] = {fr[0], fr[1], fr[2]};
        const float fdl[3] = {fr[6], fr[7], fr[8]};
        uint32_t bset = 0;
        if (live && r2q >= 0.0f) {                         // line 4: image bitset against the root node
            const int4 nd = __ldg(nodes + root);
            float a[3], b[3];
            decompress((uint32_t)nd.x, (uint32_t)nd.y, flo, fdl, a, b);
            float tq[3][3];
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
        int n = -1, img = 0;
        float xs0 = 0.f, xs1 = 0.f, xs2 = 0.f;
        while (true) {
            if (n < 0 && bset) {                           // lines 5-9: next image, restart at the root
                img = __ffs(bset) - 1;
                bset &= bset - 1;
                xs0 = __fadd_rn(me.x, (float)(img % 3 - 1) * P.L[0]);
                xs1 = __fadd_rn(me.y, (float)((img / 3) % 3 - 1) * P.L[1]);
                xs2 = __fadd_rn(me.z, (float)(img / 9 - 1) * P.L[2]);
                n = root;
            }
            if (n >= 0) {
                const int4 nd = TEX ? tex1Dfetch<int4>(tex_nodes, n) : __ldg(nodes + n);
                float a[3], b[3];
                decompress((uint32_t)nd.x, (uint32_t)nd.y, flo, fdl, a, b);
                const float t0 = __fsub_rn(fminf(fmaxf(xs0, a[0]), b[0]), xs0);
                const float t1 = __fsub_rn(fminf(fmaxf(xs1, a[1]), b[1]), xs1);
                const float t2 = __fsub_rn(fminf(fmaxf(xs2, a[2]), b[2]), xs2);
                const float d2 = __fmaf_rn(t2, t2, __fmaf_rn(t1, t1, __fmul_rn(t0, t0)));
                if (DUMMY) {
                    float acc0 = t0, acc1 = t1;
#pragma unroll
                    for (int u = 0; u < DUMMY; ++u) { acc0 = __fmaf_rn(acc0, 1.0001f, t2); acc1 = __fmaf_rn(acc1, 0.9999f, t0); }
                    if (acc0 + acc1 == 123.456f) out.cnt += 1;
                }
                const bool hit = d2 <= R2;
                if (hit && nd.z < 0) {
                    const uint32_t mm1 = (P.K > 1) ? (((uint32_t)nd.x >> 30) | (((uint32_t)nd.y >> 30) << 2)) : 0u;
                    s_q[fill][threadIdx.x] = make_uint2((uint32_t)(~nd.z), mm1 | ((uint32_t)img << 4) | ((uint32_t)tb << 9));
                    ++fill;
                }
                n = (hit && nd.z >= 0) ? nd.z : nd.w;
            }
            if (__any_sync(0xFFFFFFFFu, fill == QCAP)) flush();
            if (!__any_sync(0xFFFFFFFFu, n >= 0 || bset != 0)) break;
        }
    }
    flush();
    out.finish();
    if (live) n_neigh[orig_i] = out.cnt;
    const int wmax = __reduce_max_sync(0xFFFFFFFFu, out.cnt);
    if ((threadIdx.x & 31) == 0 && wmax > 0) atomicMax(&meta->max_count, wmax);
}


// ------------------------------------------------------------------------------------------------------------
// v3 ("group" traversal): one warp serves 32 Z-consecutive query particles (Z-order makes the
// lanes of a warp search the same part of the tree).  ncu on v0/v2 shows the per-lane rope walk is bound by the
// L1 tag stage (about 2 cycles per distinct 128-byte line touched by a divergent 16-byte gather), so here
// the warp walks the tree ONCE for the whole group and every memory access is warp-coherent:
//   * search volume of the group = bounding box of its 32 particles, tested against a node box with the
//     box-box form of eq. 2 (nearest points, squared distance <= padded r^2); it contains every member's search
//     sphere, so no pair can be missed.  The 27-image bitset (Alg. 1 line 4) is built by vote: lane j tests image j.
//   * the walk uses only the node's `left` and `rope` links, but 32 nodes are tested per step, one per lane:
//     a work list in shared memory holds node ids; testing a LEFT child also schedules its rope (= its right
//     sibling), an overlapping internal node schedules its left child, an overlapping (collapsed) leaf emits its
//     particle range.  Ballot + popc give each lane its slot in the list (no atomics).
//   * ranges are drained by the whole warp: the candidate position is one broadcast 16-byte load, every lane
//     evaluates the canonical predicate for its own particle, hits go to a per-lane staging row
//     in shared memory, and a full staging row is written to the neighbor list by all 32 lanes as one
//     contiguous 128-byte store.
// ------------------------------------------------------------------------------------------------------------
constexpr int GRP_STACK = 1024;   // work-list entries per warp
constexpr int GRP_RQ = 96;        // pending leaf ranges per warp
constexpr int GRP_STAGE = 32;     // staged neighbors per lane (one 128-byte line)

template <int WARPS>
__global__ void __launch_bounds__(WARPS * 32) traverse_group_kernel(TraverseParams P, const int4 *__restrict__ nodes,
                                                                     const float4 *__restrict__ sorted_pos,
                                                                     TreeMeta *__restrict__ meta,
                                                                     int32_t *__restrict__ nlist,
                                                                     int32_t *__restrict__ n_neigh) {
    __shared__ uint32_t s_stack[WARPS][GRP_STACK];
    __shared__ uint2 s_rq[WARPS][GRP_RQ];
    __shared__ int32_t s_stage[WARPS][32][GRP_STAGE];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t FULL = 0xFFFFFFFFu;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int k = (blockIdx.x * WARPS + warp) * 32 + lane;
    const bool live = k < P.N;
    if (!__any_sync(FULL, live)) return;
    const float4 me = live ? sorted_pos[k] : make_float4(0.f, 0.f, 0.f, 0.f);
    const int orig_i = __float_as_int(me.w);
    int ta = 0;
#pragma unroll
    for (int t = 1; t < QBVH_TMAX; ++t) ta += (k >= meta->seg[t]) ? 1 : 0;
    // bounding box of the group's live particles
    float glo[3], ghi[3];
    {
        const float v[3] = {me.x, me.y, me.z};
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            glo[d] = ord2f(~__reduce_max_sync(FULL, live ? ~f2ord(v[d]) : 0u));
            ghi[d] = ord2f(__reduce_max_sync(FULL, live ? f2ord(v[d]) : 0u));
        }
    }
    int32_t *const row = nlist + (size_t)(live ? orig_i : 0) * (size_t)P.max_neigh;
    int staged = 0, written = 0;
    uint32_t *stack = s_stack[warp];
    uint2 *rq = s_rq[warp];
    int rsz = 0;

    // write the staging rows of the lanes in `mask` to their list rows, 32 lanes per row, contiguous
    auto flush_stage = [&](uint32_t mask) {
        while (mask) {
            const int l = __ffs(mask) - 1;
            mask &= mask - 1;
            const int c = __shfl_sync(FULL, staged, l);
            const int w = __shfl_sync(FULL, written, l);
            const unsigned long long rp = __shfl_sync(FULL, (unsigned long long)row, l);
            if (lane < c && w + lane < P.max_neigh) reinterpret_cast<int32_t *>(rp)[w + lane] = s_stage[warp][l][lane];
            if (lane == l) {
                written += staged;
                staged = 0;
            }
        }
        __syncwarp();
    };

    // drain the pending leaf ranges: every lane checks every candidate of every range for its own particle
    auto flush_ranges = [&]() {
        for (int e = 0; e < rsz; ++e) {
            const uint2 q = rq[e];
            const int first = (int)q.x;
            const int m = (int)(q.y & 15u) + 1;
            const int img = (int)((q.y >> 4) & 31u);
            const int tb = (int)(q.y >> 9);
            const float r2 = live ? P.r2[ta * QBVH_TMAX + tb] : -1.0f;
            // every lane needs room for m more hits
            const uint32_t fullmask = __ballot_sync(FULL, staged > GRP_STAGE - 16);
            if (fullmask) flush_stage(fullmask);
            if (img == 13) {                                  // the unshifted image: (p_j - p_i) - 0 == p_j - p_i
                for (int t = 0; t < m; ++t) {
                    const float4 pj = __ldg(sorted_pos + first + t);
                    const float dx = __fsub_rn(pj.x, me.x), dy = __fsub_rn(pj.y, me.y), dz = __fsub_rn(pj.z, me.z);
                    const float dd = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                    if (dd <= r2 && first + t != k) s_stage[warp][lane][staged++] = __float_as_int(pj.w);
                }
            } else {
                const float s0 = (float)(img % 3 - 1) * P.L[0], s1 = (float)((img / 3) % 3 - 1) * P.L[1],
                            s2 = (float)(img / 9 - 1) * P.L[2];
                for (int t = 0; t < m; ++t) {
                    const float4 pj = __ldg(sorted_pos + first + t);
                    const float dx = __fsub_rn(__fsub_rn(pj.x, me.x), s0);
                    const float dy = __fsub_rn(__fsub_rn(pj.y, me.y), s1);
                    const float dz = __fsub_rn(__fsub_rn(pj.z, me.z), s2);
                    const float dd = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                    if (dd <= r2 && first + t != k) s_stage[warp][lane][staged++] = __float_as_int(pj.w);
                }
            }
        }
        rsz = 0;
    };

    for (int tb = 0; tb < QBVH_TMAX; ++tb) {
        const int root = meta->roots[tb];
        if (root < 0) continue;
        const float R2l = live ? P.R2[ta * QBVH_TMAX + tb] : -1.0f;
        const float R2 = __int_as_float(__reduce_max_sync(FULL, __float_as_int(R2l)));   // values are -1 or >= 0
        if (!(R2 >= 0.0f)) continue;
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
        while (bset) {                                        // lines 5-9
            const int img = __ffs(bset) - 1;
            bset &= bset - 1;
            float blo[3], bhi[3];                             // group box of this image
            {
                const int sh[3] = {img % 3 - 1, (img / 3) % 3 - 1, img / 9 - 1};
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const float sL = (float)sh[d] * P.L[d];
                    blo[d] = __fadd_rn(glo[d], sL);
                    bhi[d] = __fadd_rn(ghi[d], sL);
                }
            }
            if (lane == 0) stack[0] = (uint32_t)root;
            __syncwarp();
            int ssz = 1;
            while (ssz > 0) {                                 // lines 10-19, 32 nodes per step
                const int npop = (ssz > GRP_STACK - 64) ? 1 : min(ssz, 32);
                const bool active = lane < npop;
                bool push_sib = false, push_child = false, emit = false;
                int4 nd = make_int4(0, 0, 0, 0);
                if (active) {
                    const uint32_t ent = stack[ssz - 1 - lane];
                    nd = __ldg(nodes + (ent & 0x7FFFFFFFu));
                    float a[3], b[3];
                    decompress((uint32_t)nd.x, (uint32_t)nd.y, flo, fdl, a, b);
                    const float t0 = fmaxf(fmaxf(__fsub_rn(a[0], bhi[0]), __fsub_rn(blo[0], b[0])), 0.0f);
                    const float t1 = fmaxf(fmaxf(__fsub_rn(a[1], bhi[1]), __fsub_rn(blo[1], b[1])), 0.0f);
                    const float t2 = fmaxf(fmaxf(__fsub_rn(a[2], bhi[2]), __fsub_rn(blo[2], b[2])), 0.0f);
                    const float d2 = __fmaf_rn(t2, t2, __fmaf_rn(t1, t1, __fmul_rn(t0, t0)));
                    const bool hit = d2 <= R2;
                    push_sib = (ent >> 31) != 0;              // a left child: its rope is the right sibling
                    push_child = hit && nd.z >= 0;
                    emit = hit && nd.z < 0;
                }
                __syncwarp();                                 // all reads of the list done before it is rewritten
                const uint32_t b1 = __ballot_sync(FULL, push_sib);
                const uint32_t b2 = __ballot_sync(FULL, push_child);
                const uint32_t b3 = __ballot_sync(FULL, emit);
                const int base = ssz - npop;
                if (push_sib) stack[base + __popc(b1 & lt_mask)] = (uint32_t)nd.w;
                if (push_child) stack[base + __popc(b1) + __popc(b2 & lt_mask)] = (uint32_t)nd.z | 0x80000000u;
                ssz = base + __popc(b1) + __popc(b2);
                if (emit) {
                    const uint32_t mm1 = (P.K > 1) ? (((uint32_t)nd.x >> 30) | (((uint32_t)nd.y >> 30) << 2)) : 0u;
                    rq[rsz + __popc(b3 & lt_mask)] = make_uint2((uint32_t)(~nd.z), mm1 | ((uint32_t)img << 4) | ((uint32_t)tb << 9));
                }
                rsz += __popc(b3);
                __syncwarp();
                if (rsz > GRP_RQ - 32) flush_ranges();
            }
        }
    }
    flush_ranges();
    flush_stage(__ballot_sync(FULL, staged > 0));
    const int cnt = written;
    if (live) n_neigh[orig_i] = cnt;
    const int wmax = __reduce_max_sync(FULL, live ? cnt : 0);
    if (lane == 0 && wmax > 0) atomicMax(&meta->max_count, wmax);
}


// ------------------------------------------------------------------------------------------------------------
// v4: v3 + (a) adaptive split of the warp's 32-particle Z-order block into compact pieces, (b) leaf ranges are
// drained right after the step that found them (no range queue), (c) leaner candidate loop.
//
// (a) 32 consecutive Z-order particles are usually a compact blob, but a run that crosses a high-level split of
// the Z-curve has a bounding box spanning a large part of the simulation box.  A block [a,b] is therefore cut at
// the position where adjacent Morton keys differ in the highest bit — exactly the LBVH split of that range,
// whenever the two halves' search volumes together are smaller than the whole block's:
//     vol(box(A) (+) r) + vol(box(B) (+) r) < vol(box(A u B) (+) r),   vol(box (+) r) = prod_d (extent_d + 2 r).
// Pieces are traversed one after the other by the same warp; lanes outside the current piece sit idle.
// ------------------------------------------------------------------------------------------------------------
template <int WARPS>
__global__ void __launch_bounds__(WARPS * 32) traverse_group2_kernel(TraverseParams P, const int4 *__restrict__ nodes,
                                                                      const float4 *__restrict__ sorted_pos,
                                                                      const uint32_t *__restrict__ key_sorted,
                                                                      TreeMeta *__restrict__ meta,
                                                                      int32_t *__restrict__ nlist,
                                                                      int32_t *__restrict__ n_neigh) {
    __shared__ uint32_t s_stack[WARPS][GRP_STACK];
    __shared__ int32_t s_stage[WARPS][32][GRP_STAGE];
    __shared__ uint32_t s_pieces[WARPS][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t FULL = 0xFFFFFFFFu;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int k = (blockIdx.x * WARPS + warp) * 32 + lane;
    const bool live = k < P.N;
    const int nlive = __popc(__ballot_sync(FULL, live));
    if (nlive == 0) return;
    const float4 me = live ? sorted_pos[k] : make_float4(0.f, 0.f, 0.f, 0.f);
    const int orig_i = __float_as_int(me.w);
    const uint32_t mykey = live ? key_sorted[k] : 0u;
    int ta = 0;
#pragma unroll
    for (int t = 1; t < QBVH_TMAX; ++t) ta += (k >= meta->seg[t]) ? 1 : 0;
    // largest pruning radius any lane of the block uses against any tree (for the split heuristic)
    float rmaxl = 0.0f;
#pragma unroll
    for (int tb = 0; tb < QBVH_TMAX; ++tb) rmaxl = fmaxf(rmaxl, live ? P.R2[ta * QBVH_TMAX + tb] : 0.0f);
    const float two_r = 2.0f * sqrtf(__int_as_float(__reduce_max_sync(FULL, __float_as_int(rmaxl))));
    // xor of adjacent keys: the highest set bit over a lane range marks the LBVH split of that range
    const uint32_t knext = __shfl_down_sync(FULL, mykey, 1);
    const uint32_t kx = (lane + 1 < nlive) ? (mykey ^ knext) : 0u;

    int32_t *const row = nlist + (size_t)(live ? orig_i : 0) * (size_t)P.max_neigh;
    int32_t *const my_stage = s_stage[warp][lane];
    int staged = 0, written = 0;
    uint32_t *stack = s_stack[warp];
    const float mx = me.x, my = me.y, mz = me.z;

    auto flush_stage = [&](uint32_t mask) {
        while (mask) {
            const int l = __ffs(mask) - 1;
            mask &= mask - 1;
            const int c = __shfl_sync(FULL, staged, l);
            const int w = __shfl_sync(FULL, written, l);
            const unsigned long long rp = __shfl_sync(FULL, (unsigned long long)row, l);
            if (lane < c && w + lane < P.max_neigh) reinterpret_cast<int32_t *>(rp)[w + lane] = s_stage[warp][l][lane];
            if (lane == l) {
                written += staged;
                staged = 0;
            }
        }
        __syncwarp();
    };
    auto box_of = [&](bool in, float lo[3], float hi[3]) {
        const float v[3] = {mx, my, mz};
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            lo[d] = ord2f(~__reduce_max_sync(FULL, in ? ~f2ord(v[d]) : 0u));
            hi[d] = ord2f(__reduce_max_sync(FULL, in ? f2ord(v[d]) : 0u));
        }
    };
    auto svol = [&](const float lo[3], const float hi[3]) {
        return (hi[0] - lo[0] + two_r) * (hi[1] - lo[1] + two_r) * (hi[2] - lo[2] + two_r);
    };

    // ---- piece list (a | b << 8), LIFO ----
    int npieces = 1;
    if (lane == 0) s_pieces[warp][0] = 0u | ((uint32_t)(nlive - 1) << 8);
    __syncwarp();
    while (npieces > 0) {
        const uint32_t pc = s_pieces[warp][npieces - 1];
        --npieces;
        const int pa = (int)(pc & 255u), pb = (int)(pc >> 8);
        const bool inp = lane >= pa && lane <= pb;
        float glo[3], ghi[3];
        box_of(inp, glo, ghi);
        if (pb > pa) {
            const uint32_t xm = __reduce_max_sync(FULL, (lane >= pa && lane < pb) ? kx : 0u);
            const int sp = __ffs(__ballot_sync(FULL, lane >= pa && lane < pb && kx == xm)) - 1;   // split after lane sp
            float alo[3], ahi[3], blo2[3], bhi2[3];
            box_of(lane >= pa && lane <= sp, alo, ahi);
            box_of(lane > sp && lane <= pb, blo2, bhi2);
            if (svol(alo, ahi) + svol(blo2, bhi2) < svol(glo, ghi)) {
                __syncwarp();
                if (lane == 0) {
                    s_pieces[warp][npieces] = (uint32_t)(sp + 1) | ((uint32_t)pb << 8);
                    s_pieces[warp][npieces + 1] = (uint32_t)pa | ((uint32_t)sp << 8);
                }
                npieces += 2;
                __syncwarp();
                continue;
            }
        }
        // ---- traverse for the piece [pa, pb] ----
        const bool act_q = inp;   // this lane's particle is a query of the piece
        for (int tb = 0; tb < QBVH_TMAX; ++tb) {
            const int root = meta->roots[tb];
            if (root < 0) continue;
            const float R2l = act_q ? P.R2[ta * QBVH_TMAX + tb] : -1.0f;
            const float R2 = __int_as_float(__reduce_max_sync(FULL, __float_as_int(R2l)));
            if (!(R2 >= 0.0f)) continue;
            const float r2 = act_q ? P.r2[ta * QBVH_TMAX + tb] : -1.0f;
            const float *fr = meta->frames[tb];
            const float flo[3] = {fr[0], fr[1], fr[2]};
            const float fdl[3] = {fr[6], fr[7], fr[8]};
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
            while (bset) {
                const int img = __ffs(bset) - 1;
                bset &= bset - 1;
                const float s0 = (float)(img % 3 - 1) * P.L[0], s1 = (float)((img / 3) % 3 - 1) * P.L[1],
                            s2 = (float)(img / 9 - 1) * P.L[2];
                const float blo[3] = {__fadd_rn(glo[0], s0), __fadd_rn(glo[1], s1), __fadd_rn(glo[2], s2)};
                const float bhi[3] = {__fadd_rn(ghi[0], s0), __fadd_rn(ghi[1], s1), __fadd_rn(ghi[2], s2)};
                const bool shifted = img != 13;
                if (lane == 0) stack[0] = (uint32_t)root;
                __syncwarp();
                int ssz = 1;
                while (ssz > 0) {
                    const int npop = (ssz > GRP_STACK - 64) ? 1 : min(ssz, 32);
                    const bool active = lane < npop;
                    bool push_sib = false, push_child = false, emit = false;
                    int4 nd = make_int4(0, 0, 0, 0);
                    if (active) {
                        const uint32_t ent = stack[ssz - 1 - lane];
                        nd = __ldg(nodes + (ent & 0x7FFFFFFFu));
                        float a[3], b[3];
                        decompress((uint32_t)nd.x, (uint32_t)nd.y, flo, fdl, a, b);
                        const float t0 = fmaxf(fmaxf(__fsub_rn(a[0], bhi[0]), __fsub_rn(blo[0], b[0])), 0.0f);
                        const float t1 = fmaxf(fmaxf(__fsub_rn(a[1], bhi[1]), __fsub_rn(blo[1], b[1])), 0.0f);
                        const float t2 = fmaxf(fmaxf(__fsub_rn(a[2], bhi[2]), __fsub_rn(blo[2], b[2])), 0.0f);
                        const float d2 = __fmaf_rn(t2, t2, __fmaf_rn(t1, t1, __fmul_rn(t0, t0)));
                        const bool hit = d2 <= R2;
                        push_sib = (ent >> 31) != 0;
                        push_child = hit && nd.z >= 0;
                        emit = hit && nd.z < 0;
                    }
                    __syncwarp();
                    const uint32_t b1 = __ballot_sync(FULL, push_sib);
                    const uint32_t b2 = __ballot_sync(FULL, push_child);
                    uint32_t b3 = __ballot_sync(FULL, emit);
                    const int base = ssz - npop;
                    if (push_sib) stack[base + __popc(b1 & lt_mask)] = (uint32_t)nd.w;
                    if (push_child) stack[base + __popc(b1) + __popc(b2 & lt_mask)] = (uint32_t)nd.z | 0x80000000u;
                    ssz = base + __popc(b1) + __popc(b2);
                    __syncwarp();
                    // ---- drain the leaf ranges found in this step (line 14 of Alg. 1 for every member) ----
                    const int my_first = ~nd.z;
                    const int my_m = (P.K > 1) ? 1 + (int)(((uint32_t)nd.x >> 30) | (((uint32_t)nd.y >> 30) << 2)) : 1;
                    while (b3) {
                        const int src = __ffs(b3) - 1;
                        b3 &= b3 - 1;
                        const int first = __shfl_sync(FULL, my_first, src);
                        const int m = __shfl_sync(FULL, my_m, src);
                        const uint32_t fullmask = __ballot_sync(FULL, staged > GRP_STAGE - 16);
                        if (fullmask) flush_stage(fullmask);
                        const float4 *cp = sorted_pos + first;
                        const int kk = k - first;     // candidate t is this lane's own particle iff t == kk
                        if (!shifted) {
#pragma unroll 4
                            for (int t = 0; t < m; ++t) {
                                const float4 pj = __ldg(cp + t);
                                const float dx = __fsub_rn(pj.x, mx), dy = __fsub_rn(pj.y, my), dz = __fsub_rn(pj.z, mz);
                                const float dd = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                                if (dd <= r2 && t != kk) my_stage[staged++] = __float_as_int(pj.w);
                            }
                        } else {
#pragma unroll 4
                            for (int t = 0; t < m; ++t) {
                                const float4 pj = __ldg(cp + t);
                                const float dx = __fsub_rn(__fsub_rn(pj.x, mx), s0);
                                const float dy = __fsub_rn(__fsub_rn(pj.y, my), s1);
                                const float dz = __fsub_rn(__fsub_rn(pj.z, mz), s2);
                                const float dd = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                                if (dd <= r2 && t != kk) my_stage[staged++] = __float_as_int(pj.w);
                            }
                        }
                    }
                }
            }
        }
    }
    flush_stage(__ballot_sync(FULL, staged > 0));
    if (live) n_neigh[orig_i] = written;
    const int wmax = __reduce_max_sync(FULL, live ? written : 0);
    if (lane == 0 && wmax > 0) atomicMax(&meta->max_count, wmax);
}


// ------------------------------------------------------------------------------------------------------------
// v5: group traversal with (a) adaptive block split, (b) FIFO work list (falls back to LIFO when nearly full),
// (c) leaf ranges flattened into a candidate index list and processed as 32-candidate tiles: one gather into
// shared memory per tile (issued one tile ahead), then a fully unrolled loop in which every lane evaluates the
// canonical predicate for its own particle against each candidate of the tile (broadcast LDS.128).
// ------------------------------------------------------------------------------------------------------------
constexpr int G5_QUEUE = 1024;    // work-list ring entries per warp
constexpr int G5_CAND = 544;      // candidate indices per warp: < 32 left over + up to 32 ranges x 16
constexpr int G5_STAGE = 32;

template <int WARPS>
__global__ void __launch_bounds__(WARPS * 32) traverse_tile_kernel(TraverseParams P, const int4 *__restrict__ nodes,
                                                                    const float4 *__restrict__ sorted_pos,
                                                                    const uint32_t *__restrict__ key_sorted,
                                                                    TreeMeta *__restrict__ meta,
                                                                    int32_t *__restrict__ nlist,
                                                                    int32_t *__restrict__ n_neigh) {
    __shared__ uint32_t s_queue[WARPS][G5_QUEUE];
    __shared__ int32_t s_stage[WARPS][32][G5_STAGE];
    __shared__ int32_t s_cand[WARPS][G5_CAND];
    __shared__ float4 s_tile[WARPS][32];
    __shared__ uint32_t s_pieces[WARPS][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t FULL = 0xFFFFFFFFu;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int k = (blockIdx.x * WARPS + warp) * 32 + lane;
    const bool live = k < P.N;
    const int nlive = __popc(__ballot_sync(FULL, live));
    if (nlive == 0) return;
    const float4 me = live ? sorted_pos[k] : make_float4(0.f, 0.f, 0.f, 0.f);
    const int orig_i = live ? __float_as_int(me.w) : -1;
    const uint32_t mykey = live ? key_sorted[k] : 0u;
    int ta = 0;
#pragma unroll
    for (int t = 1; t < QBVH_TMAX; ++t) ta += (k >= meta->seg[t]) ? 1 : 0;
    float rmaxl = 0.0f;
#pragma unroll
    for (int tb = 0; tb < QBVH_TMAX; ++tb) rmaxl = fmaxf(rmaxl, live ? P.R2[ta * QBVH_TMAX + tb] : 0.0f);
    const float two_r = 2.0f * sqrtf(__int_as_float(__reduce_max_sync(FULL, __float_as_int(rmaxl))));
    const uint32_t knext = __shfl_down_sync(FULL, mykey, 1);
    const uint32_t kx = (lane + 1 < nlive) ? (mykey ^ knext) : 0u;

    int32_t *const row = nlist + (size_t)(live ? orig_i : 0) * (size_t)P.max_neigh;
    int32_t *const my_stage = s_stage[warp][lane];
    int staged = 0, written = 0;
    uint32_t *queue = s_queue[warp];
    int32_t *cand = s_cand[warp];
    float4 *tile = s_tile[warp];
    const float mx = me.x, my = me.y, mz = me.z;

    auto flush_stage = [&](uint32_t mask) {
        while (mask) {
            const int l = __ffs(mask) - 1;
            mask &= mask - 1;
            const int c = __shfl_sync(FULL, staged, l);
            const int w = __shfl_sync(FULL, written, l);
            const unsigned long long rp = __shfl_sync(FULL, (unsigned long long)row, l);
            if (lane < c && w + lane < P.max_neigh) reinterpret_cast<int32_t *>(rp)[w + lane] = s_stage[warp][l][lane];
            if (lane == l) {
                written += staged;
                staged = 0;
            }
        }
        __syncwarp();
    };
    auto box_of = [&](bool in, float lo[3], float hi[3]) {
        const float v[3] = {mx, my, mz};
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            lo[d] = ord2f(~__reduce_max_sync(FULL, in ? ~f2ord(v[d]) : 0u));
            hi[d] = ord2f(__reduce_max_sync(FULL, in ? f2ord(v[d]) : 0u));
        }
    };
    auto svol = [&](const float lo[3], const float hi[3]) {
        return (hi[0] - lo[0] + two_r) * (hi[1] - lo[1] + two_r) * (hi[2] - lo[2] + two_r);
    };

    int npieces = 1;
    if (lane == 0) s_pieces[warp][0] = 0u | ((uint32_t)(nlive - 1) << 8);
    __syncwarp();
    while (npieces > 0) {
        const uint32_t pc = s_pieces[warp][npieces - 1];
        --npieces;
        const int pa = (int)(pc & 255u), pb = (int)(pc >> 8);
        const bool inp = lane >= pa && lane <= pb;
        float glo[3], ghi[3];
        box_of(inp, glo, ghi);
        if (pb > pa) {
            const uint32_t xm = __reduce_max_sync(FULL, (lane >= pa && lane < pb) ? kx : 0u);
            const int sp = __ffs(__ballot_sync(FULL, lane >= pa && lane < pb && kx == xm)) - 1;
            float alo[3], ahi[3], blo2[3], bhi2[3];
            box_of(lane >= pa && lane <= sp, alo, ahi);
            box_of(lane > sp && lane <= pb, blo2, bhi2);
            if (svol(alo, ahi) + svol(blo2, bhi2) < svol(glo, ghi)) {
                __syncwarp();
                if (lane == 0) {
                    s_pieces[warp][npieces] = (uint32_t)(sp + 1) | ((uint32_t)pb << 8);
                    s_pieces[warp][npieces + 1] = (uint32_t)pa | ((uint32_t)sp << 8);
                }
                npieces += 2;
                __syncwarp();
                continue;
            }
        }
        for (int tb = 0; tb < QBVH_TMAX; ++tb) {
            const int root = meta->roots[tb];
            if (root < 0) continue;
            const float R2l = inp ? P.R2[ta * QBVH_TMAX + tb] : -1.0f;
            const float R2 = __int_as_float(__reduce_max_sync(FULL, __float_as_int(R2l)));
            if (!(R2 >= 0.0f)) continue;
            const float r2 = inp ? P.r2[ta * QBVH_TMAX + tb] : -1.0f;
            const float *fr = meta->frames[tb];
            const float flo[3] = {fr[0], fr[1], fr[2]};
            const float fdl[3] = {fr[6], fr[7], fr[8]};
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
            while (bset) {
                const int img = __ffs(bset) - 1;
                bset &= bset - 1;
                const float s0 = (float)(img % 3 - 1) * P.L[0], s1 = (float)((img / 3) % 3 - 1) * P.L[1],
                            s2 = (float)(img / 9 - 1) * P.L[2];
                const float blo[3] = {__fadd_rn(glo[0], s0), __fadd_rn(glo[1], s1), __fadd_rn(glo[2], s2)};
                const float bhi[3] = {__fadd_rn(ghi[0], s0), __fadd_rn(ghi[1], s1), __fadd_rn(ghi[2], s2)};

                // one 16-candidate half tile: every lane checks candidates [c0, c0+16) of the tile for its own particle
                auto half_tile = [&](int c0, int cnum) {
                    const uint32_t fullmask = __ballot_sync(FULL, staged > G5_STAGE - 16);
                    if (fullmask) flush_stage(fullmask);
#pragma unroll
                    for (int t = 0; t < 16; ++t) {
                        const float4 pj = tile[c0 + t];
                        const float dx = __fsub_rn(__fsub_rn(pj.x, mx), s0);
                        const float dy = __fsub_rn(__fsub_rn(pj.y, my), s1);
                        const float dz = __fsub_rn(__fsub_rn(pj.z, mz), s2);
                        const float dd = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                        if (dd <= r2 && __float_as_int(pj.w) != orig_i && t < cnum) my_stage[staged++] = __float_as_int(pj.w);
                    }
                };

                int ccount = 0;                              // candidate indices waiting in cand[0..ccount)
                if (lane == 0) queue[0] = (uint32_t)root;
                __syncwarp();
                int qhead = 0, qtail = 1;                    // ring indices (monotone counters)
                while (qtail > qhead) {
                    const int qn = qtail - qhead;
                    const bool lifo = qn > G5_QUEUE - 96;    // nearly full: take the newest entries instead (bounds growth)
                    const int npop = lifo ? 1 : min(qn, 32);
                    const bool active = lane < npop;
                    bool push_sib = false, push_child = false, emit = false;
                    int4 nd = make_int4(0, 0, 0, 0);
                    if (active) {
                        const uint32_t ent = lifo ? queue[(qtail - 1) & (G5_QUEUE - 1)] : queue[(qhead + lane) & (G5_QUEUE - 1)];
                        nd = __ldg(nodes + (ent & 0x7FFFFFFFu));
                        float a[3], b[3];
                        decompress((uint32_t)nd.x, (uint32_t)nd.y, flo, fdl, a, b);
                        const float t0 = fmaxf(fmaxf(__fsub_rn(a[0], bhi[0]), __fsub_rn(blo[0], b[0])), 0.0f);
                        const float t1 = fmaxf(fmaxf(__fsub_rn(a[1], bhi[1]), __fsub_rn(blo[1], b[1])), 0.0f);
                        const float t2 = fmaxf(fmaxf(__fsub_rn(a[2], bhi[2]), __fsub_rn(blo[2], b[2])), 0.0f);
                        const float d2 = __fmaf_rn(t2, t2, __fmaf_rn(t1, t1, __fmul_rn(t0, t0)));
                        const bool hit = d2 <= R2;
                        push_sib = (ent >> 31) != 0;
                        push_child = hit && nd.z >= 0;
                        emit = hit && nd.z < 0;
                    }
                    __syncwarp();
                    if (lifo) qtail -= 1; else qhead += npop;
                    const uint32_t b1 = __ballot_sync(FULL, push_sib);
                    const uint32_t b2 = __ballot_sync(FULL, push_child);
                    const uint32_t b3 = __ballot_sync(FULL, emit);
                    if (push_sib) queue[(qtail + __popc(b1 & lt_mask)) & (G5_QUEUE - 1)] = (uint32_t)nd.w;
                    if (push_child) queue[(qtail + __popc(b1) + __popc(b2 & lt_mask)) & (G5_QUEUE - 1)] = (uint32_t)nd.z | 0x80000000u;
                    qtail += __popc(b1) + __popc(b2);
                    if (b3) {
                        // flatten the emitted ranges into candidate indices (exclusive scan of the range lengths)
                        const int m = emit ? ((P.K > 1) ? 1 + (int)(((uint32_t)nd.x >> 30) | (((uint32_t)nd.y >> 30) << 2)) : 1) : 0;
                        int incl = m;
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) {
                            const int v = __shfl_up_sync(FULL, incl, o);
                            if (lane >= o) incl += v;
                        }
                        const int tot = __shfl_sync(FULL, incl, 31);
                        const int first = ~nd.z;
                        int32_t *dst = cand + ccount + incl - m;
                        for (int t = 0; t < m; ++t) dst[t] = first + t;
                        ccount += tot;
                    }
                    __syncwarp();
                    // full tiles
                    if (ccount >= 32) {
                        int cb = 0;
                        float4 pre = __ldg(sorted_pos + cand[lane]);
                        while (ccount - cb >= 32) {
                            tile[lane] = pre;
                            __syncwarp();
                            if (ccount - cb >= 64) pre = __ldg(sorted_pos + cand[cb + 32 + lane]);
                            half_tile(0, 16);
                            half_tile(16, 16);
                            __syncwarp();
                            cb += 32;
                        }
                        // move the remainder (< 32 indices) to the front
                        const int rem = ccount - cb;
                        const int v = (lane < rem) ? cand[cb + lane] : 0;
                        __syncwarp();
                        if (lane < rem) cand[lane] = v;
                        ccount = rem;
                        __syncwarp();
                    }
                }
                // the image's last, partial tile (the shift changes with the image)
                if (ccount > 0) {
                    if (lane < ccount) tile[lane] = __ldg(sorted_pos + cand[lane]);
                    __syncwarp();
                    half_tile(0, min(ccount, 16));
                    if (ccount > 16) half_tile(16, ccount - 16);
                    __syncwarp();
                }
            }
        }
    }
    flush_stage(__ballot_sync(FULL, staged > 0));
    if (live) n_neigh[orig_i] = written;
    const int wmax = __reduce_max_sync(FULL, live ? written : 0);
    if (lane == 0 && wmax > 0) atomicMax(&meta->max_count, wmax);
}

cudaError_t launch_traverse(const TraverseParams &p, const BuildBuffers &b, int32_t *nlist, int32_t *n_neigh,
                            bool stats, int variant, cudaStream_t st, cudaTextureObject_t tn, cudaTextureObject_t tp) {
    if (p.N == 0) return cudaSuccess;
    const int threads = 128;
    const int blocks = (p.N + threads - 1) / threads;
    if (stats)
        traverse_kernel<true><<<blocks, threads, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh);
    else if (variant == 0)
        traverse_kernel<false><<<blocks, threads, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh);
    else if (variant == 1)
        traverse_v2_kernel<8, 128, false><<<blocks, 128, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh, 0, 0);
    else if (variant == 8)
        traverse_tile_kernel<4><<<(p.N + 127) / 128, 128, 0, st>>>(p, b.nodes, b.sorted_pos, b.key_a, b.meta, nlist, n_neigh);
    else if (variant == 7)
        traverse_group2_kernel<4><<<(p.N + 127) / 128, 128, 0, st>>>(p, b.nodes, b.sorted_pos, b.key_a, b.meta, nlist, n_neigh);
    else if (variant == 4)
        traverse_group_kernel<4><<<(p.N + 127) / 128, 128, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh);
    else if (variant == 2)
        traverse_v2_kernel<16, 128, false><<<blocks, 128, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh, 0, 0);
    else if (variant == 6)
        traverse_v2_kernel<16, 128, false, 12><<<blocks, 128, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh, 0, 0);
    else if (variant == 5 && tn && tp)
        traverse_v2_kernel<16, 128, true><<<blocks, 128, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh, tn, tp);
    else
        traverse_v2_kernel<32, 128, false><<<blocks, 128, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh, 0, 0);
    return cudaGetLastError();
}

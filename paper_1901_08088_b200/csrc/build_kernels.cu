// build_kernels.cu — steps a1..a6 of the hot path and the build-side subtree collapse (§8f NEXT-1),
// hand-written for sm_100a.  Five launches:
//   a1  morton_cell_kernel : Morton keys in the periodic box, per-type root AABB (the quantization
//                            frame), occupancy of the Morton cells (the leading 2 + 3 lvl key bits)
//       cell_scan_kernel   : exclusive scan of the cell occupancies (decoupled look-back); its last block writes type
//                            segments, roots, frames
//   a2  cell_scatter_kernel: most-significant-digit pass of the radix sort: every (key, index) goes to its cell
//   a2..a6 cell_tree_kernel: one warp per cell: sorts the cell by (key, index) — the result is the stable sort of
//                            gathers into Z-order, quantizes each particle onto the 1023-bin grid of
//                            its tree's root box with outward rounding, and builds the cell's
//                            subtree of Karras' radix tree bottom up in shared memory: hierarchy,
//                            ropes in closed form, boxes united on the packed 10-bit integers
//   a3..a6 top_tree_kernel : the tree above the cells: one thread per cell root walks up, the two children of a node
//                            meet through one 128-bit atomic exchange ("atomic" hand-over)
// Subtree collapse: a node is written only once it is known not to lie below a collapsed
// range leaf; the choice is made bottom up by an integer cost model.
#include "qbvh_internal.cuh"

// ------------------------------------------------------------------------------------------------------------
// a1. Morton keys.  b_d = clamp(floor((p_d - lo_d) * s_d), 0, 1023), s_d = 1023/L_d (fp32 RN, computed on the
// host); code = 30-bit interleave with x in the most significant position of each triple; key = type<<30 | code.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t spread10(uint32_t v) {  // bit t -> bit 3t
    v &= 0x3FFu;
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

__device__ __forceinline__ uint32_t morton_bin(float p, float lo, float s) {
    float u = __fmul_rn(__fsub_rn(p, lo), s);
    float f = floorf(u);
    f = fminf(fmaxf(f, 0.0f), 1023.0f);   // fmaxf(NaN,0) = 0
    return (uint32_t)f;
}

constexpr int MORTON_THREADS = 256;

// PT = float: the paper's single-precision particle data.  PT = double (qbvh_build_f64,
// PAPER.md:140, 154): the tree is built from the positions rounded to fp32; the exact leaf test stays in fp64.
// Four consecutive particles per thread, every particle of the system in flight at once (one wave of threads).
// rank_out[i] = place of particle i inside its Morton cell, in order of arrival (one atomic per set of lanes that
// share a cell: already Z-ordered input, common in MD, would otherwise hammer one address); the cell is sorted by
// (key, index) afterwards, so the final order is the stable sort whatever the arrival order was.
template <int NT, typename PT>
__global__ void __launch_bounds__(MORTON_THREADS) morton_cell_kernel(const PT *__restrict__ pos,
                                                           const int32_t *__restrict__ type, int N, float3 lo,
                                                           float3 scale, int cell_shift, uint32_t *__restrict__ key_out,
                                                           uint32_t *__restrict__ rank_out,
                                                           uint32_t *__restrict__ cell_count,
                                                           TreeMeta *__restrict__ meta,
                                                           int32_t *__restrict__ entry, int entry_words) {
    const int stride = gridDim.x * blockDim.x;
    const int gtid = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    // the entry table of the traversal starts out empty (-1) and is filled by the tree kernels
    for (int i = gtid; i < entry_words; i += stride) entry[i] = -1;

    float mn[NT][3], mx[NT][3];
#pragma unroll
    for (int t = 0; t < NT; ++t)
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            mn[t][d] = INFINITY;
            mx[t][d] = -INFINITY;
        }
    bool bad_type = false;
    const int i0 = 4 * gtid;
    float px[4], py[4], pz[4];
    int tt[4] = {0, 0, 0, 0};
    const bool full = i0 + 3 < N;
    if (sizeof(PT) == 4 && full && ((reinterpret_cast<uintptr_t>(pos) & 15) == 0)) {
        const float4 *p4 = reinterpret_cast<const float4 *>(pos) + 3 * (size_t)gtid;   // three 128-bit loads
        const float4 a = __ldg(p4), b = __ldg(p4 + 1), c = __ldg(p4 + 2);
        px[0] = a.x, py[0] = a.y, pz[0] = a.z, px[1] = a.w, py[1] = b.x, pz[1] = b.y;
        px[2] = b.z, py[2] = b.w, pz[2] = c.x, px[3] = c.y, py[3] = c.z, pz[3] = c.w;
    } else {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int i = min(i0 + u, N - 1);
            px[u] = (float)pos[3 * (size_t)i + 0], py[u] = (float)pos[3 * (size_t)i + 1], pz[u] = (float)pos[3 * (size_t)i + 2];
        }
    }
    if (type) {
        if (full && ((reinterpret_cast<uintptr_t>(type) & 15) == 0)) {
            const int4 t4 = __ldg(reinterpret_cast<const int4 *>(type) + gtid);
            tt[0] = t4.x, tt[1] = t4.y, tt[2] = t4.z, tt[3] = t4.w;
        } else {
#pragma unroll
            for (int u = 0; u < 4; ++u) tt[u] = type[min(i0 + u, N - 1)];
        }
    }
    uint32_t key[4], rank[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const bool valid = i0 + u < N;
        int ty = tt[u];
        if (valid && (ty < 0 || ty >= NT)) {
            bad_type = true;
            ty = 0;
        }
        const uint32_t t = (uint32_t)ty;
        const float x = px[u], y = py[u], z = pz[u];
        const uint32_t code = (spread10(morton_bin(x, lo.x, scale.x)) << 2) | (spread10(morton_bin(y, lo.y, scale.y)) << 1) |
                              spread10(morton_bin(z, lo.z, scale.z));
        key[u] = (t << 30) | code;
        if (valid) {
#pragma unroll
            for (int v = 0; v < NT; ++v) {
                const bool m = (NT == 1) || (t == (uint32_t)v);
                mn[v][0] = m ? fminf(mn[v][0], x) : mn[v][0];
                mn[v][1] = m ? fminf(mn[v][1], y) : mn[v][1];
                mn[v][2] = m ? fminf(mn[v][2], z) : mn[v][2];
                mx[v][0] = m ? fmaxf(mx[v][0], x) : mx[v][0];
                mx[v][1] = m ? fmaxf(mx[v][1], y) : mx[v][1];
                mx[v][2] = m ? fmaxf(mx[v][2], z) : mx[v][2];
            }
        }
    }
    // the four draws of a thread are independent: all atomics are issued before the first result is used
    uint32_t grp[4], base[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) grp[u] = __match_any_sync(0xFFFFFFFFu, (i0 + u < N) ? (key[u] >> cell_shift) : 0xFFFFFFFFu);
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        base[u] = 0;
        if (i0 + u < N && lane == __ffs(grp[u]) - 1) base[u] = atomicAdd(&cell_count[key[u] >> cell_shift], (uint32_t)__popc(grp[u]));
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) rank[u] = __shfl_sync(0xFFFFFFFFu, base[u], __ffs(grp[u]) - 1) + __popc(grp[u] & ((1u << lane) - 1u));
    if (full && ((reinterpret_cast<uintptr_t>(key_out) & 15) == 0) && ((reinterpret_cast<uintptr_t>(rank_out) & 15) == 0)) {
        reinterpret_cast<uint4 *>(key_out)[gtid] = make_uint4(key[0], key[1], key[2], key[3]);
        reinterpret_cast<uint4 *>(rank_out)[gtid] = make_uint4(rank[0], rank[1], rank[2], rank[3]);
    } else {
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (i0 + u < N) {
                key_out[i0 + u] = key[u];
                rank_out[i0 + u] = rank[u];
            }
    }
    // per-type min/max: warp reduce on the order-preserving encoding, block reduce through shared memory, then one
    // global atomic per block and value
    __shared__ uint32_t s_mm[QBVH_TMAX][6];
    if (threadIdx.x < QBVH_TMAX * 6) (&s_mm[0][0])[threadIdx.x] = 0u;
    __syncthreads();
#pragma unroll
    for (int t = 0; t < NT; ++t)
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            uint32_t a = __reduce_max_sync(0xFFFFFFFFu, ~f2ord(mn[t][d]));
            uint32_t b = __reduce_max_sync(0xFFFFFFFFu, f2ord(mx[t][d]));
            if (lane == 0) {
                if (a != ~f2ord(INFINITY)) atomicMax(&s_mm[t][d], a);
                if (b != f2ord(-INFINITY)) atomicMax(&s_mm[t][3 + d], b);
            }
        }
    __syncthreads();
    if (threadIdx.x < NT * 6) {
        const uint32_t v = (&s_mm[0][0])[threadIdx.x];
        if (v) atomicMax(&meta->mm_enc[0][0] + threadIdx.x, v);
    }
    if (bad_type) atomicOr(&meta->err_flags, 1);
}

// ------------------------------------------------------------------------------------------------------------
// Scan of the cell occupancies.  One tile of SCAN_TILE cells per block, tiles chained by decoupled look-back on one
// 64-bit status word (at most SCAN_MAX_TILES = 128 blocks: all resident at once).  Writes cell_start (exclusive
// prefix, cell_start[ncells] = N) and the ascending list of non-empty cells; the last block to finish turns the
// per-type results into segments, roots and quantization frames.
// ------------------------------------------------------------------------------------------------------------
struct FinalizeParams {
    int N, T, lvl, warp_slots, group_cap;
    float r_hint[QBVH_TMAX];
};

__device__ void finalize_block(TreeMeta *__restrict__ meta, const uint32_t *__restrict__ cell_start, const FinalizeParams fp) {
    const int d = threadIdx.x;
    __shared__ float s_rho[QBVH_TMAX];
    __shared__ int s_cnt[QBVH_TMAX];
    const int cpt = 1 << (3 * fp.lvl);              // cells per type
    auto seg_of = [&](int t) -> int { return t < fp.T ? (int)__ldcg(cell_start + (size_t)t * cpt) : fp.N; };
    if (d <= QBVH_TMAX) meta->seg[d] = seg_of(d);
    if (d < QBVH_TMAX) {
        const int s = seg_of(d), n = seg_of(d + 1) - s;
        meta->roots[d] = (n <= 0) ? -1 : (n == 1 ? (fp.N - 1 + s) : s);
        float *fr = meta->frames[d];
        float vol = 1.0f;
        int32_t *rb = meta->rbin[d];
        rb[0] = rb[1] = rb[2] = rb[3] = -1;
        if (n > 0) {
            const float rh = fp.r_hint[d];
            for (int a = 0; a < 3; ++a) {
                float lo = ord2f(~__ldcg(&meta->mm_enc[d][a]));
                float hi = ord2f(__ldcg(&meta->mm_enc[d][3 + a]));
                fr[a] = lo;
                fr[3 + a] = hi;
                // Delta = div_ru(sub_ru(hi, lo), 1023): the 1023-bin grid spans at least the root box
                const float delta = __fdiv_ru(__fsub_ru(hi, lo), QBVH_NBINS);
                fr[6 + a] = delta;
                fr[9 + a] = delta > 0.0f ? __fdiv_rn(1.0f, delta) : 0.0f;     // first guess of the quantizer only
                vol *= hi - lo;
                // expected query radius in bins of this axis (collapse cost model): ceil(r / Delta), fp32 RN division
                if (rh > 0.0f) rb[a] = delta > 0.0f ? (int)fminf(ceilf(__fdiv_rn(rh, delta)), 1023.0f) : 1;
            }
        } else {
            for (int a = 0; a < 12; ++a) fr[a] = 0.0f;
        }
        s_rho[d] = (n > 1 && vol > 0.0f) ? (float)n / vol : 0.0f;    // unknown (flat or single): treated as dense
        s_cnt[d] = n > 0 ? n : 0;
    }
    __syncthreads();
    // Query-group size per type.  One warp traverses for a whole group with the group's box as search volume, so
    // the candidates it draws from a tree of number density rho_b grow with rho_b x (group size / rho_t): for a
    // type far sparser than the densest one (the colloids of a colloid-solvent mixture) a full group
    // would sweep up thousands of misses.  Groups of type t hold at most 32 rho_t / rho_max particles (>= 1).
    if (d < QBVH_TMAX) {
        const float rmax = fmaxf(fmaxf(s_rho[0], s_rho[1]), fmaxf(s_rho[2], s_rho[3]));
        int gm = min(GROUP_MAX, max(fp.group_cap, 1));       // QBVH_OPT_GROUP_MAX (default 32)
        if (s_rho[d] > 0.0f && rmax > 0.0f)
            gm = (int)fminf(fmaxf(floorf((float)gm * s_rho[d] / rmax), 1.0f), (float)gm);
        // Small systems (the regime of PAPER.md:186): with fewer groups than the device has resident warps the
        // traversal is one group's latency, so groups shrink (down to 4) until there is about one per warp.
        gm = min(gm, max(4, s_cnt[d] / max(fp.warp_slots, 1)));
        meta->gmax[d] = gm;
    }
}

// One tile of SCAN_TILE cells per block.  No chain between the tiles.  Up to SCAN_DIRECT_TILES tiles every block
// simply adds up the counters of all tiles before its own (a few hundred KB out of L2) and nothing waits for anything;
// beyond that every block publishes its tile's total and the blocks meet once (at most SCAN_MAX_TILES = 128 blocks,
// normally all resident at once; the wait is bounded and falls back to the direct sum).  The kernel is a handful of
// dependent L2 round trips.
constexpr int SCAN_DIRECT_TILES = 32;
__global__ void __launch_bounds__(SCAN_THREADS) cell_scan_kernel(const uint32_t *__restrict__ cell_count,
                                                                  uint32_t *__restrict__ cell_start,
                                                                  uint32_t *__restrict__ cell_list, int ncells,
                                                                  TreeMeta *__restrict__ meta, long long spin_cycles) {
    cudaGridDependencySynchronize();
    __shared__ unsigned long long s_warp[SCAN_THREADS / 32], s_pre[SCAN_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x, ntiles = gridDim.x;
    const int c0 = tile * SCAN_TILE + tid * SCAN_IPT;
    auto value = [](uint32_t c) { return (unsigned long long)c | ((unsigned long long)(c != 0) << 32); };   // particles, non-empty cells << 32
    uint32_t cnt[SCAN_IPT];
    if (c0 + SCAN_IPT <= ncells) {
        const uint4 a = __ldcg(reinterpret_cast<const uint4 *>(cell_count + c0)), b = __ldcg(reinterpret_cast<const uint4 *>(cell_count + c0) + 1);
        cnt[0] = a.x, cnt[1] = a.y, cnt[2] = a.z, cnt[3] = a.w, cnt[4] = b.x, cnt[5] = b.y, cnt[6] = b.z, cnt[7] = b.w;
    } else {
#pragma unroll
        for (int u = 0; u < SCAN_IPT; ++u) cnt[u] = (c0 + u < ncells) ? __ldcg(cell_count + c0 + u) : 0u;
    }
    // sum of everything before this tile, read directly (tiles are full except the last)
    unsigned long long before = 0;
    if (ntiles <= SCAN_DIRECT_TILES) {
        const uint4 *src = reinterpret_cast<const uint4 *>(cell_count);
        for (int q = tid; q < tile * (SCAN_TILE / 4); q += SCAN_THREADS) {
            const uint4 v = __ldcg(src + q);
            before += value(v.x) + value(v.y) + value(v.z) + value(v.w);
        }
    }
    unsigned long long mine = 0;
#pragma unroll
    for (int u = 0; u < SCAN_IPT; ++u) mine += value(cnt[u]);
    unsigned long long inc = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long v = __shfl_up_sync(0xFFFFFFFFu, inc, o);
        if (lane >= o) inc += v;
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) before += __shfl_xor_sync(0xFFFFFFFFu, before, o);
    if (lane == 31) s_warp[warp] = inc;
    if (lane == 0) s_pre[warp] = before;
    __syncthreads();
    unsigned long long wbase = 0, total = 0, excl = 0;
#pragma unroll
    for (int w = 0; w < SCAN_THREADS / 32; ++w) {
        if (w < warp) wbase += s_warp[w];
        total += s_warp[w];
        excl += s_pre[w];
    }
    if (ntiles > SCAN_DIRECT_TILES) {
        // The blocks meet once: each publishes its tile's total and waits until all have.  Blocks of an ordinary launch
        // are not promised to be resident together (a busy or partitioned device), so the wait is bounded: a block that
        // has not seen everybody after spin_cycles adds up the counters before its tile itself, as the small grids do —
        // the same sum, never a hang.
        volatile unsigned long long *tot = meta->scan_status;
        __shared__ int s_met;
        if (tid == 0) {
            tot[tile] = total;
            __threadfence();
            atomicAdd(&meta->scan_arrived, 1u);
            const long long t0 = clock64();
            bool met = false;
            while (!(met = *(volatile uint32_t *)&meta->scan_arrived >= (uint32_t)ntiles) && clock64() - t0 < spin_cycles) {}
            __threadfence();
            s_met = met ? 1 : 0;
        }
        __syncthreads();
        unsigned long long v = 0ull;
        if (s_met) {
            v = (tid < tile) ? tot[tid] : 0ull;     // ntiles <= 128 <= SCAN_THREADS
        } else {
            const uint4 *src = reinterpret_cast<const uint4 *>(cell_count);
            for (int q = tid; q < tile * (SCAN_TILE / 4); q += SCAN_THREADS) {
                const uint4 c = __ldcg(src + q);
                v += value(c.x) + value(c.y) + value(c.z) + value(c.w);
            }
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
        __syncthreads();
        if (lane == 0) s_pre[warp] = v;
        __syncthreads();
        excl = 0;
#pragma unroll
        for (int w = 0; w < SCAN_THREADS / 32; ++w) excl += s_pre[w];
    }
    unsigned long long run = excl + wbase + inc - mine;
#pragma unroll
    for (int u = 0; u < SCAN_IPT; ++u) {
        if (c0 + u < ncells) {
            cell_start[c0 + u] = (uint32_t)run;
            if (cnt[u]) cell_list[(uint32_t)(run >> 32)] = (uint32_t)(c0 + u);
        }
        run += value(cnt[u]);
    }
    if (tile == ntiles - 1 && tid == SCAN_THREADS - 1) {
        cell_start[ncells] = (uint32_t)run;              // = N
        meta->ncell = (int32_t)(run >> 32);
    }
}

// N = 0: only the bookkeeping
__global__ void finalize_empty_kernel(TreeMeta *__restrict__ meta) {
    const int d = threadIdx.x;
    if (d <= QBVH_TMAX) meta->seg[d] = 0;
    if (d < QBVH_TMAX) {
        meta->roots[d] = -1;
        meta->gmax[d] = GROUP_MAX;
        for (int a = 0; a < 12; ++a) meta->frames[d][a] = 0.0f;
        for (int a = 0; a < 4; ++a) meta->rbin[d][a] = -1;
    }
}

// ------------------------------------------------------------------------------------------------------------
// a2, first pass (the most significant digit of the radix sort): (key, index) of every particle to its cell, at the
// place the key kernel drew for it.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) cell_scatter_kernel(const uint32_t *__restrict__ key, const uint32_t *__restrict__ rank,
                                                            int N, int cell_shift, const uint32_t *__restrict__ cell_start,
                                                            uint2 *__restrict__ ent, uint32_t *__restrict__ cell_count, int ncells,
                                                            TreeMeta *__restrict__ meta, const FinalizeParams fp) {
    cudaGridDependencySynchronize();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    // the counters have been scanned: clear them for the next build
    for (int c = i; c < ncells; c += gridDim.x * blockDim.x) cell_count[c] = 0u;
    if (i < N) {
        const uint32_t k = __ldg(key + i);
        ent[__ldg(cell_start + (k >> cell_shift)) + __ldg(rank + i)] = make_uint2(k, (uint32_t)i);
    }
    // type segments, roots, quantization frames: needed by the next launch only; one block does it on the side
    if (blockIdx.x == gridDim.x - 1) finalize_block(meta, cell_start, fp);
}

// ------------------------------------------------------------------------------------------------------------
// Quantizer defined by its decompressor:
//   D_lo(q) = fma_rd(q, Delta, lo)   D_hi(q) = fma_ru(q, Delta, lo)
//   q_lo(a) = max{q : D_lo(q) <= a}  q_hi(b) = min{q : D_hi(q) >= b}
// D_lo and D_hi are monotone in q, so a first guess from (a - lo) / Delta is checked against its neighbours and,
// should it be off by more than one (denormal Delta), replaced by the 10-step bisection.  q_lo, q_hi are monotone, so
// the union of boxes is the per-field integer min/max of the packed words.
// ------------------------------------------------------------------------------------------------------------
__device__ __noinline__ uint32_t quant_lo_bisect(float a, float lo, float delta) {
    uint32_t q = 0;
    for (uint32_t bit = 512; bit; bit >>= 1) {
        uint32_t c = q | bit;
        if (__fmaf_rd((float)c, delta, lo) <= a) q = c;
    }
    return q;
}
__device__ __noinline__ uint32_t quant_hi_bisect(float b, float lo, float delta) {
    uint32_t q = 0;
    for (uint32_t bit = 512; bit; bit >>= 1) {
        uint32_t c = q + bit;
        if (__fmaf_ru((float)(c - 1), delta, lo) < b) q = c;
    }
    return q;
}
__device__ __forceinline__ uint32_t quant_lo(float a, float lo, float delta, float inv) {
    int q = (int)fminf(fmaxf(floorf(__fmul_rn(__fsub_rn(a, lo), inv)), 0.0f), 1023.0f);
    if (__fmaf_rd((float)q, delta, lo) <= a) {
        if (q == 1023 || __fmaf_rd((float)(q + 1), delta, lo) > a) return (uint32_t)q;
        ++q;
        if (q == 1023 || __fmaf_rd((float)(q + 1), delta, lo) > a) return (uint32_t)q;
    } else if (q > 0) {
        --q;
        if (__fmaf_rd((float)q, delta, lo) <= a) return (uint32_t)q;
    }
    return quant_lo_bisect(a, lo, delta);
}
__device__ __forceinline__ uint32_t quant_hi(float b, float lo, float delta, float inv) {
    int q = (int)fminf(fmaxf(ceilf(__fmul_rn(__fsub_rn(b, lo), inv)), 0.0f), 1023.0f);
    if (__fmaf_ru((float)q, delta, lo) >= b) {
        if (q == 0 || __fmaf_ru((float)(q - 1), delta, lo) < b) return (uint32_t)q;
        --q;
        if (q == 0 || __fmaf_ru((float)(q - 1), delta, lo) < b) return (uint32_t)q;
    } else if (q < 1023) {
        ++q;
        if (__fmaf_ru((float)q, delta, lo) >= b) return (uint32_t)q;
    }
    return quant_hi_bisect(b, lo, delta);
}
// q_hi of the same value whose q_lo is known (a point: its box is one bin, Fig. 3c): the first guess is q_lo
// itself or the bin line above it
__device__ __forceinline__ uint32_t quant_hi_from_lo(float b, float lo, float delta, uint32_t qlo) {
    int q = (int)qlo;
    if (__fmaf_ru((float)q, delta, lo) >= b) {
        if (q == 0 || __fmaf_ru((float)(q - 1), delta, lo) < b) return (uint32_t)q;
    } else if (q < 1023) {
        ++q;
        if (__fmaf_ru((float)q, delta, lo) >= b) return (uint32_t)q;   // D_hi(q - 1) < b was just seen
    }
    return quant_hi_bisect(b, lo, delta);
}
__device__ __forceinline__ uint32_t pack_min(uint32_t a, uint32_t b) {
    return min(a & 0x3FFu, b & 0x3FFu) | min(a & 0xFFC00u, b & 0xFFC00u) | min(a & 0x3FF00000u, b & 0x3FF00000u);
}
__device__ __forceinline__ uint32_t pack_max(uint32_t a, uint32_t b) {
    return max(a & 0x3FFu, b & 0x3FFu) | max(a & 0xFFC00u, b & 0xFFC00u) | max(a & 0x3FF00000u, b & 0x3FF00000u);
}

// 128-bit atomic exchange (sm_90+): returns the previous content of *addr
__device__ __forceinline__ uint4 exch128(uint4 *addr, uint4 v) {
    unsigned long long vlo = (unsigned long long)v.x | ((unsigned long long)v.y << 32);
    unsigned long long vhi = (unsigned long long)v.z | ((unsigned long long)v.w << 32);
    unsigned long long olo, ohi;
    asm volatile(
        "{\n .reg .b128 _v, _d;\n mov.b128 _v, {%2, %3};\n atom.global.relaxed.gpu.exch.b128 _d, [%4], _v;\n"
        " mov.b128 {%0, %1}, _d;\n}"
        : "=l"(olo), "=l"(ohi)
        : "l"(vlo), "l"(vhi), "l"(addr)
        : "memory");
    return make_uint4((uint32_t)olo, (uint32_t)(olo >> 32), (uint32_t)ohi, (uint32_t)(ohi >> 32));
}

// common prefix length of the augmented keys (ka, a) and (kb, b)
__device__ __forceinline__ int delta_aug(uint32_t ka, int a, uint32_t kb, int b) {
    const uint32_t x = ka ^ kb;
    return x ? __clz(x) : 32 + __clz((uint32_t)a ^ (uint32_t)b);
}

// ------------------------------------------------------------------------------------------------------------
// What both tree kernels share.
//
// Hierarchy (Karras' binary radix tree, "built bottom up"): every node covers a contiguous range
// [f,l] of the sorted augmented keys (key, position).  With dL = delta(f-1,f) and dR = delta(l,l+1) the common
// prefix lengths with the outside neighbours (-1 beyond the type segment), the node is the LEFT child of its
// parent iff dR > dL, and then the parent splits at gamma = l; otherwise it is the RIGHT child and gamma = f-1.
// (dL = dR only at a root, where both are -1.)  Numbering (pinned in tests/test_oracle_tree.py): a
// left child [f,gamma] is internal node gamma, a right child [gamma+1,l] is internal node gamma+1, a root is the
// first position of its segment; leaf k is node N-1+k.  Rope: a left child's rope is its right
// sibling; a right child's rope is its parent's; for a node covering [f,l] in closed form: END if l is the segment
// end, else with m = l+1: internal node m if its range starts at m (delta(m,m+1) > delta(m,m-1)), else leaf m.
//
// Collapse.  A node is PENDING while it may still end up inside a range leaf:
// single particles, and nodes that chose to collapse.  A pending node is not written; the thread that forms its
// parent either collapses the parent too (the children vanish) or writes the parent and, as leaves, its pending
// children.  A node may collapse only if both children are pending, so a written node is never below a leaf.
// ------------------------------------------------------------------------------------------------------------
struct TreeCtx {
    const void *pos;
    int f64;
    int N, K, lvl;
    uint32_t build_tag;
    const uint32_t *cell_start, *cell_list;
    uint2 *ent;
    uint32_t *key_sorted, *idx_sorted;
    float4 *sorted_pos;
    Pos64 *sorted_pos64;
    int4 *nodes;
    int32_t *parent;
    uint4 *slot;
    uint2 *groups;
    int32_t *entry;
    int32_t *big_list;
    CellRoot *croot;
    unsigned char *scratch;
    TreeMeta *meta;
};

struct Child {
    uint32_t wlo, whi;   // packed box (30 bits each)
    int f, l;            // sorted positions covered
    bool pend;
};

__device__ __forceinline__ unsigned long long swollen(uint32_t wlo, uint32_t whi, const int32_t *rb) {
    unsigned long long w = 1;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int ext = max((int)((whi >> (10 * d)) & 1023u) - (int)((wlo >> (10 * d)) & 1023u), 0);   // zero-extent frames invert the codes (R10)
        w *= (unsigned long long)(ext + 2 * rb[d]);
    }
    return w;
}
__device__ __forceinline__ unsigned long long leaf_cost(unsigned long long w, int cnt) {
    return w * (unsigned long long)(COST_LEAF_FIXED + COST_LEAF_PER_PARTICLE * cnt);
}

// Entry table of the traversal.  The upper levels of an LBVH over Morton codes ARE a regular grid: all particles
// whose code starts with a given 3l-bit prefix (one cell of the 2^l-per-axis grid over the box) form
// one subtree.  A node whose keys share `dnode` leading bits while its parent's share only `dpar` roots the cell
// of every level l with dpar < 2 + 3 l <= dnode (2 type bits, then the code).
__device__ __forceinline__ void emit_entry(int32_t *__restrict__ etab, uint32_t ki, int dpar, int dnode, int node) {
    if (dpar >= 2 + 3 * ENTRY_LMAX || dnode < 2 + 3 * ENTRY_LMIN) return;   // below or above every grid level
#pragma unroll
    for (int l = ENTRY_LMIN; l <= ENTRY_LMAX; ++l) {
        const int need = 2 + 3 * l;
        if (dpar < need && need <= dnode) etab[entry_offset(l) + (int)((ki & 0x3FFFFFFFu) >> (30 - 3 * l))] = node;
    }
}

// A range leaf covering sorted positions [f, l] (dnode = common prefix length of its keys): on grid levels finer than
// the leaf itself no node below it exists any more, so the leaf roots every cell of those levels that holds one of
// its particles (the traversal drops the duplicates among its entry nodes).
template <class KeyF>
__device__ __forceinline__ void emit_entry_leaf(int32_t *__restrict__ etab, KeyF keyat, int f, int l, int dpar, int dnode, int node) {
    if (dpar >= 2 + 3 * ENTRY_LMAX) return;
    const uint32_t kf = keyat(f);
    emit_entry(etab, kf, dpar, dnode, node);
#pragma unroll 1
    for (int lv = ENTRY_LMIN; lv <= ENTRY_LMAX; ++lv) {
        const int need = 2 + 3 * lv;
        if (dpar < need && need > dnode)
            for (int k = f; k <= l; ++k) etab[entry_offset(lv) + (int)((keyat(k) & 0x3FFFFFFFu) >> (30 - 3 * lv))] = node;
    }
}

// query groups (maximal subtrees with <= gmax leaves): appended with one atomic per converged set of lanes
__device__ __forceinline__ void emit_groups(TreeMeta *meta, uint2 *__restrict__ groups, uint2 g0, uint2 g1, int n) {
    const uint32_t act = __activemask();
    const uint32_t two = __ballot_sync(act, n >= 2);
    const int lane = threadIdx.x & 31;
    const uint32_t lt = (1u << lane) - 1u;
    const int leader = __ffs(act) - 1;
    int base = 0;
    if (lane == leader) base = atomicAdd(&meta->group_count, __popc(act) + __popc(two));
    base = __shfl_sync(act, base, leader) + __popc(act & lt) + __popc(two & lt);
    groups[base] = g0;
    if (n >= 2) groups[base + 1] = g1;
}

// Form the parent of the adjacent children a (left) and b (right).  dL, dR: the parent's outer prefix lengths;
// dsplit = delta(a.l, b.f): the parent's own prefix length.  rope_p: the parent's rope (and b's).  pfx(f, l): common
// prefix length of the keys at sorted positions f and l.  Returns whether the parent is pending; ulo/uhi: its box.
// kparent: any key below the parent (entry table); keyat(k): key at sorted position k, asked for the particles of
// pending children only.
template <class KeyF, class PfxF>
__device__ __forceinline__ bool form_parent(const TreeCtx &cx, int t, int s_seg, int gmax, const int32_t *rb, uint32_t kparent, KeyF keyat,
                                            const Child a, const Child b, int dL, int dR, int dsplit, int rope_p, PfxF pfx,
                                            uint32_t &ulo, uint32_t &uhi, int &written) {
    const int N = cx.N;
    ulo = pack_min(a.wlo, b.wlo);
    uhi = pack_max(a.whi, b.whi);
    const int ca = a.l - a.f + 1, cb = b.l - b.f + 1, cnt = ca + cb;
    bool collapse = cx.K > 1 && cnt <= cx.K && a.pend && b.pend;
    if (collapse && rb[0] >= 0) {
        const unsigned long long wp = swollen(ulo, uhi, rb);
        collapse = leaf_cost(wp, cnt) <=
                   wp * (unsigned long long)COST_NODE + leaf_cost(swollen(a.wlo, a.whi, rb), ca) + leaf_cost(swollen(b.wlo, b.whi, rb), cb);
    }
    const bool root = dL < 0 && dR < 0;
    if (!collapse) {
        const int id = root ? s_seg : (dR > dL ? b.l : a.f);
        const int lc = ca == 1 ? N - 1 + a.f : a.l;
        const int rc = cb == 1 ? N - 1 + b.f : b.f;
        cx.nodes[id] = make_int4((int)ulo, (int)uhi, lc, rope_p);
        cx.parent[lc] = id;
        cx.parent[rc] = id;
        if (root) cx.parent[id] = -1;
        int32_t *const etab = cx.entry + t * ENTRY_CELLS;
        emit_entry(etab, kparent, max(dL, dR), dsplit, id);
        written = 1;
        if (a.pend) {
            cx.nodes[lc] = make_int4((int)a.wlo, (int)a.whi, ~a.f, rc);
            if (dsplit < 2 + 3 * ENTRY_LMAX) emit_entry_leaf(etab, keyat, a.f, a.l, dsplit, ca == 1 ? 64 : pfx(a.f, a.l), lc);
            ++written;
        }
        if (b.pend) {
            cx.nodes[rc] = make_int4((int)b.wlo, (int)b.whi, ~b.f, rope_p);
            if (dsplit < 2 + 3 * ENTRY_LMAX) emit_entry_leaf(etab, keyat, b.f, b.l, dsplit, cb == 1 ? 64 : pfx(b.f, b.l), rc);
            ++written;
        }
    }
    if (cnt > gmax) {                            // children that fit are maximal: they become query groups
        const int nl = ca <= gmax, nr = cb <= gmax;
        if (nl + nr) {
            const uint2 gl = make_uint2((uint32_t)a.f, (uint32_t)ca), gr = make_uint2((uint32_t)b.f, (uint32_t)cb);
            emit_groups(cx.meta, cx.groups, nl ? gl : gr, gr, nl + nr);
        }
    }
    return collapse;
}

// common prefix length of two cells' keys (cell ids carry the type bits); -1 across types
__device__ __forceinline__ int delta_cells(uint32_t ca, uint32_t cb, int lvl) {
    if ((ca >> (3 * lvl)) != (cb >> (3 * lvl))) return -1;
    return __clz((ca ^ cb) << (30 - 3 * lvl));
}

// The root of a type's tree that is still pending (a single particle, or everything collapsed): written as a leaf.
template <class KeyF>
__device__ __forceinline__ void write_pending_root(const TreeCtx &cx, int t, KeyF keyat, const Child me, int pfx_me) {
    const int id = (me.l == me.f) ? cx.N - 1 + me.f : me.f;      // = meta->roots[t]
    cx.nodes[id] = make_int4((int)me.wlo, (int)me.whi, ~me.f, -1);
    cx.parent[id] = -1;
    emit_entry_leaf(cx.entry + t * ENTRY_CELLS, keyat, me.f, me.l, -1, pfx_me, id);
}

// Walk up from a finished subtree (a cell root) through the levels above the cells.  The two children of a node meet at
// slot[gamma]: the first to arrive leaves a 16-byte record there with ONE 128-bit atomic exchange and retires; the
// second takes it and forms the parent ("walking up the tree from the leaf nodes").  Record:
//   x = packed lower bound | pending << 31      y = packed upper bound
//   z = far end of the range (a left child: its first position, a right child: its last)
//   w = build tag << 14 | (dnext + 1) << 7 | (outer delta + 1)
// dnext (right children): delta(m, m+1) for m = last + 1, the first particle of the NEXT cell, known from the cell
// table when the cell was built (64 if that cell holds two or more particles) — with it the parent's rope needs no
// key at all, so a level of the walk is one L2 round trip.  Slots are tagged with an 18-bit per-build number instead
// of being cleared every build.
static_assert(QBVH_TAG_MAX == (1u << 18) - 1, "the tag shares a word with two 7-bit prefix lengths");
__device__ void walk_up(const TreeCtx &cx, Child me, int dL, int dR, int dnext) {
    const uint32_t *key = cx.key_sorted;
    const uint32_t ki = key[me.f];                         // the walker's own cell: sorted before the walk starts
    const int t = (int)(ki >> 30);
    const int s_seg = cx.meta->seg[t];
    const int gmax = cx.meta->gmax[t];
    const int32_t *rb = cx.meta->rbin[t];
    auto keyat = [&](int k) { return key[k]; };           // asked for a.f and for pending children only: small cells, sorted by the previous launch
    auto pfx = [&](int f, int l) { return delta_aug(key[f], f, key[l], l); };
    int written = 0;
    while (true) {
        if (dL < 0 && dR < 0) {                      // the root of this type's tree
            if (me.pend) {
                write_pending_root(cx, t, keyat, me, me.l == me.f ? 64 : pfx(me.f, me.l));
                ++written;
            }
            if (me.l - me.f + 1 <= gmax) emit_groups(cx.meta, cx.groups, make_uint2((uint32_t)me.f, (uint32_t)(me.l - me.f + 1)), make_uint2(0u, 0u), 1);
            break;
        }
        const bool is_left = dR > dL;
        const int gamma = is_left ? me.l : me.f - 1;
        const uint4 mine = make_uint4(me.wlo | (me.pend ? 0x80000000u : 0u), me.whi, (uint32_t)(is_left ? me.f : me.l),
                                      (cx.build_tag << 14) | ((uint32_t)(dnext + 1) << 7) | (uint32_t)((is_left ? dL : dR) + 1));
        const uint4 other = exch128(cx.slot + gamma, mine);
        if ((other.w >> 14) != cx.build_tag) break;  // first to arrive: the sibling will carry on
        const int dsplit = is_left ? dR : dL;        // delta(gamma, gamma+1): the parent's own prefix length
        Child sib;
        sib.wlo = other.x & 0x7FFFFFFFu;
        sib.whi = other.y;
        sib.pend = (other.x >> 31) != 0;
        Child a, b;
        if (is_left) {
            sib.f = gamma + 1;
            sib.l = (int)other.z;
            dR = (int)(other.w & 127u) - 1;
            dnext = (int)((other.w >> 7) & 127u) - 1;
            a = me, b = sib;
        } else {
            sib.f = (int)other.z;
            sib.l = gamma;
            dL = (int)(other.w & 127u) - 1;
            a = sib, b = me;
        }
        const int rope_p = dR < 0 ? -1 : (dnext > dR ? b.l + 1 : cx.N + b.l);   // internal node m or leaf N-1+m, m = b.l + 1
        uint32_t ulo, uhi;
        int w = 0;
        const bool pend = form_parent(cx, t, s_seg, gmax, rb, ki, keyat, a, b, dL, dR, dsplit, rope_p, pfx, ulo, uhi, w);
        written += w;
        me.wlo = ulo, me.whi = uhi, me.f = a.f, me.l = b.l, me.pend = pend;
    }
    if (written) atomicAdd(&cx.meta->nodes_emitted, written);
}

// ------------------------------------------------------------------------------------------------------------
// One cell: G cooperating threads (a warp, or a whole block for a cell too large for a warp's shared memory).
// Working arrays of length >= the next power of two of n: in shared memory, or for giant cells in global scratch.
// ------------------------------------------------------------------------------------------------------------
struct CellArrays {
    unsigned long long *kv;   // (key << 32 | original index): sorted ascending = Z-order, ties by index
    int32_t *e;               // at a segment's first position: its last position; -1 elsewhere
    int32_t *mrg;             // merge partner chosen in the current round, -1: none
    uint32_t *wlo, *whi;      // packed box of the segment; bit 31 of wlo: pending
    int8_t *dL, *dR;          // outer prefix lengths of the segment
};
constexpr int CELL_BYTES_PER_SLOT = 8 + 4 + 4 + 4 + 4 + 1 + 1;   // 26

__device__ __forceinline__ CellArrays carve_cell_arrays(unsigned char *base, int cap) {
    CellArrays A;
    A.kv = reinterpret_cast<unsigned long long *>(base);
    A.e = reinterpret_cast<int32_t *>(base + 8 * (size_t)cap);
    A.mrg = A.e + cap;
    A.wlo = reinterpret_cast<uint32_t *>(A.mrg + cap);
    A.whi = A.wlo + cap;
    A.dL = reinterpret_cast<int8_t *>(A.whi + cap);
    A.dR = A.dL + cap;
    return A;
}

template <int G>
__device__ __forceinline__ void coop_sync() {
    if (G == 32) __syncwarp();
    else __syncthreads();
}

// Batcher's odd-even merge sort over kv[0..n): every comparator moves the smaller value to the lower index, so
// positions >= n act as +infinity without being stored (their comparators are skipped).
template <int G>
__device__ void sort_cell(unsigned long long *kv, int n, int rank) {
    int P = 1;
    while (P < n) P <<= 1;
    auto cmpx = [&](int i, int j) {
        if (j < n) {
            const unsigned long long x = kv[i], y = kv[j];
            if (y < x) {
                kv[i] = y;
                kv[j] = x;
            }
        }
    };
    for (int size = 2; size <= P; size <<= 1) {
        int stride = size >> 1;
        coop_sync<G>();
        for (int tq = rank; tq < (P >> 1); tq += G) {
            const int pos = 2 * tq - (tq & (stride - 1));
            cmpx(pos, pos + stride);
        }
        for (stride >>= 1; stride > 0; stride >>= 1) {
            coop_sync<G>();
            for (int tq = rank; tq < (P >> 1); tq += G) {
                const int pos = 2 * tq - (tq & (stride - 1));
                const int offset = tq & ((size >> 1) - 1);
                if (offset >= stride) cmpx(pos - stride, pos);
            }
        }
    }
    coop_sync<G>();
}

// A warp's cell (n <= CELL_WARP_MAX): rank by counting.  Every lane keeps its own entries in registers, every entry
// is broadcast once from shared memory and counted against them; all keys are distinct (the index is part of them).
template <int Q>
__device__ __forceinline__ void sort_cell_warp_q(unsigned long long *kv, int n, int lane) {
    unsigned long long mine[Q];
    int below[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        mine[q] = (lane + 32 * q < n) ? kv[lane + 32 * q] : ~0ull;
        below[q] = 0;
    }
    __syncwarp();
#pragma unroll 4
    for (int jj = 0; jj < n; ++jj) {
        const unsigned long long v = kv[jj];
#pragma unroll
        for (int q = 0; q < Q; ++q) below[q] += v < mine[q];
    }
    __syncwarp();
#pragma unroll
    for (int q = 0; q < Q; ++q)
        if (lane + 32 * q < n) kv[below[q]] = mine[q];
    __syncwarp();
}
__device__ __forceinline__ void sort_cell_warp(unsigned long long *kv, int n, int lane) {
    static_assert(CELL_WARP_MAX == 128, "four entries per lane at most");
    if (n <= 32) sort_cell_warp_q<1>(kv, n, lane);
    else if (n <= 64) sort_cell_warp_q<2>(kv, n, lane);
    else sort_cell_warp_q<4>(kv, n, lane);
}

// packed-box union of the particles at local positions [f, l] of a warp's cell
__device__ __forceinline__ void range_box(const CellArrays &A, int f, int l, int lane, uint32_t &lo, uint32_t &hi) {
    uint32_t x0 = 1023u, y0 = 1023u, z0 = 1023u, x1 = 0u, y1 = 0u, z1 = 0u;
    for (int p = f + lane; p <= l; p += 32) {
        const uint32_t a = A.wlo[p], b = A.whi[p];
        x0 = min(x0, a & 1023u), y0 = min(y0, (a >> 10) & 1023u), z0 = min(z0, (a >> 20) & 1023u);
        x1 = max(x1, b & 1023u), y1 = max(y1, (b >> 10) & 1023u), z1 = max(z1, (b >> 20) & 1023u);
    }
    const uint32_t FULL = 0xFFFFFFFFu;
    // one reduction per bound: the three 10-bit fields travel in one word (min of the sum is not the sum of the
    // mins, so the fields are reduced one by one)
    x0 = __reduce_min_sync(FULL, x0), y0 = __reduce_min_sync(FULL, y0), z0 = __reduce_min_sync(FULL, z0);
    x1 = __reduce_max_sync(FULL, x1), y1 = __reduce_max_sync(FULL, y1), z1 = __reduce_max_sync(FULL, z1);
    lo = x0 | (y0 << 10) | (z0 << 20);
    hi = x1 | (y1 << 10) | (z1 << 20);
}

template <int G>
__device__ void process_cell(const TreeCtx &cx, const CellArrays A, int j, int rank, bool kv_is_ent) {
    const int N = cx.N, lvl = cx.lvl;
    const int ncell = cx.meta->ncell;
    const uint32_t c = __ldg(cx.cell_list + j);
    const int F = (int)__ldg(cx.cell_start + c);
    const int n = (int)__ldg(cx.cell_start + c + 1) - F;
    const int t = (int)(c >> (3 * lvl));
    const int s_seg = cx.meta->seg[t], e_seg = cx.meta->seg[t + 1] - 1;
    const int gmax = cx.meta->gmax[t];
    const int32_t *rb = cx.meta->rbin[t];
    // neighbouring cells: outer prefix lengths of the cell, and what starts right after it
    int dLc = -1, dRc = -1, dNN = -1, n_next = 0;
    if (j > 0) dLc = delta_cells(__ldg(cx.cell_list + j - 1), c, lvl);
    if (j + 1 < ncell) {
        const uint32_t cn = __ldg(cx.cell_list + j + 1);
        dRc = delta_cells(c, cn, lvl);
        if (dRc >= 0) {
            n_next = (int)(__ldg(cx.cell_start + cn + 1) - __ldg(cx.cell_start + cn));
            if (j + 2 < ncell) dNN = delta_cells(cn, __ldg(cx.cell_list + j + 2), lvl);
        }
    }
    // ---- a2: sort the cell by (key, index) ----
    if (!kv_is_ent)
        for (int p = rank; p < n; p += G) {
            const uint2 e = cx.ent[F + p];
            A.kv[p] = ((unsigned long long)e.x << 32) | e.y;
        }
    if (G == 32) {
        __syncwarp();
        sort_cell_warp(A.kv, n, rank);
    } else {
        sort_cell<G>(A.kv, n, rank);
    }
    const float *fr = cx.meta->frames[t];
    // collapse by size alone, query groups at least as large as the range leaves: the top-down path below
    const bool by_size = G == 32 && cx.K > 1 && rb[0] < 0 && gmax >= cx.K;
    // ---- a2' gather, a6 quantize, leaf state ----
    for (int p = rank; p < n; p += G) {
        const unsigned long long kvp = A.kv[p];
        const uint32_t ki = (uint32_t)(kvp >> 32), idx = (uint32_t)kvp;
        const int k = F + p;
        cx.key_sorted[k] = ki;
        cx.idx_sorted[k] = idx;
        float x, y, z;
        if (cx.f64) {
            const double *pp = static_cast<const double *>(cx.pos) + 3 * (size_t)idx;
            const double xd = pp[0], yd = pp[1], zd = pp[2];
            Pos64 q;
            q.x = xd, q.y = yd, q.z = zd, q.idx = (long long)idx;
            cx.sorted_pos64[k] = q;
            x = (float)xd, y = (float)yd, z = (float)zd;
        } else {
            const float *pp = static_cast<const float *>(cx.pos) + 3 * (size_t)idx;
            x = pp[0], y = pp[1], z = pp[2];
        }
        cx.sorted_pos[k] = make_float4(x, y, z, __uint_as_float(idx));
        const uint32_t qx = quant_lo(x, fr[0], fr[6], fr[9]), qy = quant_lo(y, fr[1], fr[7], fr[10]), qz = quant_lo(z, fr[2], fr[8], fr[11]);
        const uint32_t wlo = qx | (qy << 10) | (qz << 20);
        const uint32_t whi = quant_hi_from_lo(x, fr[0], fr[6], qx) | (quant_hi_from_lo(y, fr[1], fr[7], qy) << 10) |
                             (quant_hi_from_lo(z, fr[2], fr[8], qz) << 20);
        A.wlo[p] = wlo | 0x80000000u;                    // a single particle is pending
        A.whi[p] = whi;
        if (!by_size) {                                  // segment state of the rounds
            A.e[p] = p;
            A.dL[p] = (int8_t)(p > 0 ? delta_aug(ki, k, (uint32_t)(A.kv[p - 1] >> 32), k - 1) : dLc);
            A.dR[p] = (int8_t)(p < n - 1 ? delta_aug(ki, k, (uint32_t)(A.kv[p + 1] >> 32), k + 1) : dRc);
        }
        if (k == e_seg && k < N - 1) {                   // no internal node carries the index of a segment end
            cx.nodes[k] = make_int4(0, 0, 0, -1);
            cx.parent[k] = -1;
        }
    }
    coop_sync<G>();
    // rope of a node whose last particle is local position l (dcur = delta(l, l+1), the node's dR)
    auto rope_of = [&](int l, int dcur) -> int {
        if (F + l >= e_seg) return -1;
        const int m = l + 1;
        int dnext;
        if (m <= n - 2) dnext = delta_aug((uint32_t)(A.kv[m] >> 32), F + m, (uint32_t)(A.kv[m + 1] >> 32), F + m + 1);
        else if (m == n - 1) dnext = dRc;
        else dnext = n_next >= 2 ? 64 : dNN;             // m = first particle of the next cell
        return dnext > dcur ? F + m : N - 1 + F + m;
    };
    auto keyat = [&](int k) { return (uint32_t)(A.kv[k - F] >> 32); };
    auto pfx = [&](int f, int l) { return delta_aug(keyat(f), f, keyat(l), l); };
    if (by_size) {
        // (gmax >= K: query groups are unions of range leaves, so none has to be cut out of a leaf's inside)
        // ---- Collapse by size alone (no cost hint): a node is a range leaf iff it holds <= K particles, so only the
        //      nodes with more than K particles exist as internal nodes.  They are split top down — the split of a
        //      range is where the highest differing bit of its first and last augmented key flips —
        //      and nothing below the range leaves is ever touched.  Same tree as the rounds below would give. ----
        const int lane = rank;
        int written = 0;
        CellRoot r;
        r.first = F, r.last = F + n - 1, r.d = cell_root_d(dLc, dRc, n_next >= 2 ? 64 : dNN, false);
        r.key0 = (uint32_t)(A.kv[0] >> 32), r.pad[0] = r.pad[1] = 0u;
        if (n <= cx.K) {
            uint32_t lo, hi;
            range_box(A, 0, n - 1, lane, lo, hi);
            r.wlo = lo | 0x80000000u, r.whi = hi;      // pending: the top-level walk decides
        } else {
            auto aug = [&](int p) { return (A.kv[p] & 0xFFFFFFFF00000000ull) | (unsigned long long)(uint32_t)(F + p); };
            int32_t *stack = A.mrg;                      // entries f | l << 8 | (dL+1) << 16 | (dR+1) << 24
            int sp = 0;
            if (lane == 0) stack[0] = 0 | ((n - 1) << 8) | ((dLc + 1) << 16) | ((dRc + 1) << 24);
            sp = 1;
            __syncwarp();
            while (sp > 0) {
                const uint32_t ent = (uint32_t)stack[--sp];
                __syncwarp();
                const int f = ent & 255u, l = (ent >> 8) & 255u, dL = (int)((ent >> 16) & 255u) - 1, dR = (int)(ent >> 24) - 1;
                const int bit = 63 - __clzll((long long)(aug(f) ^ aug(l)));
                int g = l;                               // first position whose key has the bit set
                for (int base = f + 1; base <= l; base += 32) {
                    const int p = base + lane;
                    const uint32_t m = __ballot_sync(0xFFFFFFFFu, p <= l && ((aug(p) >> bit) & 1ull));
                    if (m) {
                        g = base + __ffs(m) - 1;
                        break;
                    }
                }
                const int gam = g - 1, dsplit = 63 - bit;
                Child a, b;
                a.f = F + f, a.l = F + gam, b.f = F + gam + 1, b.l = F + l;
                range_box(A, f, gam, lane, a.wlo, a.whi);
                range_box(A, gam + 1, l, lane, b.wlo, b.whi);
                const int ca = gam - f + 1, cb = l - gam;
                a.pend = ca <= cx.K, b.pend = cb <= cx.K;
                if (lane == 0) {
                    uint32_t ulo, uhi;
                    int w = 0;
                    // cnt > K: form_parent never collapses this node; it writes it and its pending children
                    form_parent(cx, t, s_seg, gmax, rb, keyat(a.f), keyat, a, b, dL, dR, dsplit, rope_of(l, dR), pfx, ulo, uhi, w);
                    written += w;
                    if (f == 0 && l == n - 1) r.wlo = ulo, r.whi = uhi;
                    if (!a.pend) stack[sp] = f | (gam << 8) | ((dL + 1) << 16) | ((dsplit + 1) << 24);
                    if (!b.pend) stack[sp + (a.pend ? 0 : 1)] = (gam + 1) | (l << 8) | ((dsplit + 1) << 16) | ((dR + 1) << 24);
                }
                sp += (a.pend ? 0 : 1) + (b.pend ? 0 : 1);
                __syncwarp();
            }
        }
        if (lane == 0) {
            cx.croot[j] = r;
            if (written) atomicAdd(&cx.meta->nodes_emitted, written);
        }
        return;
    }
    // ---- a3..a6 inside the cell: rounds of merges.  A segment that is a left child (dR > dL) merges with the segment
    //      that starts right after it if that one is a right child: then they are siblings.  Height of the cell's
    //      subtree rounds; no atomics. ----
    int written = 0;
    while (A.e[0] != n - 1) {
        for (int p = rank; p < n; p += G) {
            int partner = -1;
            const int ep = A.e[p];
            if (ep >= 0 && ep < n - 1 && A.dR[p] > A.dL[p]) {
                const int s = ep + 1;
                if (!(A.dR[s] > A.dL[s])) partner = s;   // s starts a segment (it follows one) and is a right child
            }
            A.mrg[p] = partner;
        }
        coop_sync<G>();
        for (int p = rank; p < n; p += G) {
            const int s = A.mrg[p];
            if (s < 0) continue;
            Child a, b;
            a.wlo = A.wlo[p] & 0x7FFFFFFFu, a.whi = A.whi[p], a.f = F + p, a.l = F + A.e[p], a.pend = (A.wlo[p] >> 31) != 0;
            b.wlo = A.wlo[s] & 0x7FFFFFFFu, b.whi = A.whi[s], b.f = F + s, b.l = F + A.e[s], b.pend = (A.wlo[s] >> 31) != 0;
            const int dL = A.dL[p], dR = A.dR[s], dsplit = A.dR[p];
            uint32_t ulo, uhi;
            int w = 0;
            const bool pend = form_parent(cx, t, s_seg, gmax, rb, keyat(a.f), keyat, a, b, dL, dR, dsplit, rope_of(b.l - F, dR),
                                          pfx, ulo, uhi, w);
            written += w;
            A.wlo[p] = ulo | (pend ? 0x80000000u : 0u);
            A.whi[p] = uhi;
            A.e[p] = b.l - F;
            A.dR[p] = (int8_t)dR;
            A.e[s] = -1;
        }
        coop_sync<G>();
    }
    if (rank == 0) {
        CellRoot r;
        r.wlo = A.wlo[0];
        r.whi = A.whi[0];
        r.first = F;
        r.last = F + n - 1;
        r.d = cell_root_d(dLc, dRc, n_next >= 2 ? 64 : dNN, G != 32);
        r.key0 = (uint32_t)(A.kv[0] >> 32), r.pad[0] = r.pad[1] = 0u;
        cx.croot[j] = r;
    }
    if (G == 32) {
        written = __reduce_add_sync(0xFFFFFFFFu, written);
        if (rank == 0 && written) atomicAdd(&cx.meta->nodes_emitted, written);
    } else if (written) {
        atomicAdd(&cx.meta->nodes_emitted, written);
    }
}

constexpr int CELL_WARPS = 4;
__global__ void __launch_bounds__(CELL_WARPS * 32) cell_tree_kernel(const TreeCtx cx) {
    cudaGridDependencySynchronize();
    __shared__ __align__(16) unsigned char s_mem[CELL_WARPS][CELL_WARP_MAX * CELL_BYTES_PER_SLOT];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int j = blockIdx.x * CELL_WARPS + warp;
    if (j >= cx.meta->ncell) return;
    const uint32_t c = __ldg(cx.cell_list + j);
    const int n = (int)(__ldg(cx.cell_start + c + 1) - __ldg(cx.cell_start + c));
    if (n > CELL_WARP_MAX) {                        // too large for a warp: a whole block takes it in the next launch
        if (lane == 0) {
            cx.big_list[atomicAdd(&cx.meta->nbig, 1)] = j;
            cx.croot[j].d = CELL_ROOT_BIG;
        }
        return;
    }
    process_cell<32>(cx, carve_cell_arrays(s_mem[warp], CELL_WARP_MAX), j, lane, false);
}

constexpr int TOP_THREADS = 512;
__global__ void __launch_bounds__(TOP_THREADS) top_tree_kernel(const TreeCtx cx) {
    cudaGridDependencySynchronize();
    extern __shared__ __align__(16) unsigned char s_dyn[];
    // ---- cells too large for one warp (rare: strongly clustered input), one block each ----
    const int nbig = cx.meta->nbig;
    for (int b = blockIdx.x; b < nbig; b += gridDim.x) {
        const int j = cx.big_list[b];
        const uint32_t c = __ldg(cx.cell_list + j);
        const int F = (int)__ldg(cx.cell_start + c);
        const int n = (int)__ldg(cx.cell_start + c + 1) - F;
        __syncthreads();
        if (n <= CELL_BLOCK_MAX) {
            process_cell<TOP_THREADS>(cx, carve_cell_arrays(s_dyn, CELL_BLOCK_MAX), j, threadIdx.x, false);
        } else {
            // giant cell: the entries are sorted in place, the other arrays live in the scratch area at the cell's own offset
            CellArrays A;
            A.kv = reinterpret_cast<unsigned long long *>(cx.ent + F);
            unsigned char *sc = cx.scratch;
            A.e = reinterpret_cast<int32_t *>(sc) + F;
            A.mrg = reinterpret_cast<int32_t *>(sc + 4 * (size_t)cx.N) + F;
            A.wlo = reinterpret_cast<uint32_t *>(sc + 8 * (size_t)cx.N) + F;
            A.whi = reinterpret_cast<uint32_t *>(sc + 12 * (size_t)cx.N) + F;
            A.dL = reinterpret_cast<int8_t *>(sc + 16 * (size_t)cx.N) + F;
            A.dR = reinterpret_cast<int8_t *>(sc + 17 * (size_t)cx.N) + F;
            // ent holds {key, index} as uint2 = little-endian (index << 32 | key): swap the halves so that the
            // 64-bit order is (key, index)
            for (int p = threadIdx.x; p < n; p += TOP_THREADS) {
                const uint2 e = cx.ent[F + p];
                A.kv[p] = ((unsigned long long)e.x << 32) | e.y;
            }
            __syncthreads();
            process_cell<TOP_THREADS>(cx, A, j, threadIdx.x, true);
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence();                          // the block's key_sorted stores, for the ropes of the walk
            const CellRoot r = cx.croot[j];
            Child me;
            me.wlo = r.wlo & 0x7FFFFFFFu, me.whi = r.whi, me.f = r.first, me.l = r.last, me.pend = (r.wlo >> 31) != 0;
            walk_up(cx, me, (int)(r.d & 255u) - 1, (int)((r.d >> 8) & 255u) - 1, (int)((r.d >> 16) & 255u) - 1);
        }
    }
    // ---- one thread per cell root.  The 32 cell roots of a warp are consecutive in Z-order, so the lowest levels above
    //      the cells are merged inside the warp first, by the same rounds as inside a cell (a segment that is a left child
    //      merges with the segment starting right after it if that one is a right child), the state exchanged by
    //      shuffles: about five levels fewer for the atomic walk, whose length is pure latency. ----
    const int lane = threadIdx.x & 31;
    const uint32_t FULL = 0xFFFFFFFFu;
    const int j = blockIdx.x * TOP_THREADS + threadIdx.x;
    bool alive = false;
    Child me;
    me.wlo = me.whi = 0u, me.f = me.l = 0, me.pend = false;
    int dL = -1, dR = -1, dnext = -1, t = 0;
    uint32_t ki = 0;
    if (j < cx.meta->ncell) {
        const CellRoot r = cx.croot[j];
        if (!(r.d & CELL_ROOT_BIG)) {                // a large cell is walked by the block that builds it (the bit says so whichever of the two wrote last)
            me.wlo = r.wlo & 0x7FFFFFFFu, me.whi = r.whi, me.f = r.first, me.l = r.last, me.pend = (r.wlo >> 31) != 0;
            dL = (int)(r.d & 255u) - 1, dR = (int)((r.d >> 8) & 255u) - 1, dnext = (int)((r.d >> 16) & 255u) - 1;
            ki = r.key0;
            t = (int)(ki >> 30);
            alive = true;
        }
    }
    const int s_seg = cx.meta->seg[t], gmax = cx.meta->gmax[t];
    const int32_t *rb = cx.meta->rbin[t];
    const uint32_t *key = cx.key_sorted;
    auto keyat = [&](int k) { return key[k]; };
    auto pfx = [&](int f, int l) { return delta_aug(key[f], f, key[l], l); };
    int lastl = lane;                                // last lane of this lane's segment
    int written = 0;
    while (true) {
        const int sc = min(lastl + 1, 31);           // head of the segment that starts right after mine
        const int p_alive = __shfl_sync(FULL, (int)alive, sc), p_dL = __shfl_sync(FULL, dL, sc), p_dR = __shfl_sync(FULL, dR, sc);
        const bool merge = alive && dR > dL && lastl < 31 && p_alive && !(p_dR > p_dL);
        if (!__any_sync(FULL, merge)) break;
        Child b;
        b.wlo = __shfl_sync(FULL, me.wlo, sc), b.whi = __shfl_sync(FULL, me.whi, sc);
        b.l = __shfl_sync(FULL, me.l, sc), b.pend = __shfl_sync(FULL, (int)me.pend, sc) != 0;
        const int p_dnext = __shfl_sync(FULL, dnext, sc), p_lastl = __shfl_sync(FULL, lastl, sc);
        const uint32_t kill = __reduce_or_sync(FULL, merge ? (1u << sc) : 0u);
        if (merge) {
            b.f = me.l + 1;
            const int dsplit = dR;                   // delta(gamma, gamma+1): the parent's own prefix length
            dR = p_dR, dnext = p_dnext, lastl = p_lastl;
            const int rope_p = dR < 0 ? -1 : (dnext > dR ? b.l + 1 : cx.N + b.l);
            uint32_t ulo, uhi;
            int w = 0;
            const bool pend = form_parent(cx, t, s_seg, gmax, rb, ki, keyat, me, b, dL, dR, dsplit, rope_p, pfx, ulo, uhi, w);
            written += w;
            me.wlo = ulo, me.whi = uhi, me.l = b.l, me.pend = pend;
        }
        if ((kill >> lane) & 1u) alive = false;
    }
    if (written) atomicAdd(&cx.meta->nodes_emitted, written);
    if (alive) walk_up(cx, me, dL, dR, dnext);
}

// ------------------------------------------------------------------------------------------------------------
// The build is a chain of five dependent launches.  The four dependents are launched with programmatic stream
// serialization (programmatic dependent launch): their blocks may be scheduled while the predecessor drains and wait in
// cudaGridDependencySynchronize() — the first statement of each of those kernels — until the predecessor's memory is
// visible, which takes the launch latency off the critical path.
template <typename... KArgs, typename... Args>
static cudaError_t launch_dependent(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid, cfg.blockDim = block, cfg.dynamicSmemBytes = smem, cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr, cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

int pick_cell_level(int64_t N, int T) {
    // the smallest grid with at most ~48 particles per cell on average, T * 8^lvl <= CELL_MAX_TOTAL
    int lvl = CELL_LMIN;
    while (lvl < CELL_LMAX && N > (int64_t)48 << (3 * lvl)) ++lvl;
    while (lvl > CELL_LMIN && ((int64_t)T << (3 * lvl)) > CELL_MAX_TOTAL) --lvl;
    return lvl;
}

cudaError_t launch_build(const void *pos, const int32_t *type, const BuildParams &p, const BuildBuffers &b, cudaStream_t st) {
    const int N = p.N;
    cudaError_t err = cudaMemsetAsync(b.meta, 0, sizeof(TreeMeta), st);
    if (err != cudaSuccess) return err;
    if (N == 0) {
        finalize_empty_kernel<<<1, 32, 0, st>>>(b.meta);
        return cudaGetLastError();
    }
    static int sms = 0;
    if (sms == 0) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaFuncSetAttribute(top_tree_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, CELL_BLOCK_MAX * CELL_BYTES_PER_SLOT);
    }
    const int lvl = p.lvl;
    const int ncells = p.T << (3 * lvl);
    const int cell_shift = 30 - 3 * lvl;
    const int entry_words = QBVH_TMAX * ENTRY_CELLS;
    const float3 lo = make_float3(p.box_lo[0], p.box_lo[1], p.box_lo[2]);
    const float3 sc = make_float3(p.box_scale[0], p.box_scale[1], p.box_scale[2]);
    const int mblocks = ((N + 3) / 4 + MORTON_THREADS - 1) / MORTON_THREADS;
#define QBVH_MORTON(NT)                                                                                                        \
    if (p.f64)                                                                                                                 \
        morton_cell_kernel<NT, double><<<mblocks, MORTON_THREADS, 0, st>>>(static_cast<const double *>(pos), type, N, lo, sc,  \
                                                                          cell_shift, b.key, b.rank, b.cell_count, b.meta, b.entry, entry_words); \
    else                                                                                                                       \
        morton_cell_kernel<NT, float><<<mblocks, MORTON_THREADS, 0, st>>>(static_cast<const float *>(pos), type, N, lo, sc,    \
                                                                         cell_shift, b.key, b.rank, b.cell_count, b.meta, b.entry, entry_words);
    switch (p.T) {
        case 1: QBVH_MORTON(1) break;
        case 2: QBVH_MORTON(2) break;
        case 3: QBVH_MORTON(3) break;
        default: QBVH_MORTON(4) break;
    }
#undef QBVH_MORTON
    FinalizeParams fp;
    fp.N = N, fp.T = p.T, fp.lvl = lvl, fp.warp_slots = traverse_warp_slots(), fp.group_cap = p.group_cap;
    for (int t = 0; t < QBVH_TMAX; ++t) fp.r_hint[t] = p.r_hint[t];
    const int tiles = (ncells + SCAN_TILE - 1) / SCAN_TILE;
    err = launch_dependent(cell_scan_kernel, dim3(tiles), dim3(SCAN_THREADS), 0, st, b.cell_count, b.cell_start, b.cell_list, ncells, b.meta,
                           (long long)p.scan_spin_cycles);
    if (err != cudaSuccess) return err;
    err = launch_dependent(cell_scatter_kernel, dim3((N + 255) / 256), dim3(256), 0, st, b.key, b.rank, N, cell_shift, b.cell_start, b.ent,
                           b.cell_count, ncells, b.meta, fp);
    if (err != cudaSuccess) return err;
    TreeCtx cx;
    cx.pos = pos, cx.f64 = p.f64 ? 1 : 0, cx.N = N, cx.K = p.K, cx.lvl = lvl, cx.build_tag = p.build_tag;
    cx.cell_start = b.cell_start, cx.cell_list = b.cell_list, cx.ent = b.ent;
    cx.key_sorted = b.key_sorted, cx.idx_sorted = b.idx_sorted, cx.sorted_pos = b.sorted_pos;
    cx.sorted_pos64 = b.sorted_pos64;
    cx.nodes = b.nodes, cx.parent = b.parent, cx.slot = b.slot, cx.groups = b.groups, cx.entry = b.entry;
    cx.big_list = b.big_list, cx.croot = b.croot, cx.scratch = b.scratch, cx.meta = b.meta;
    const int max_cells = min(N, ncells);
    err = launch_dependent(cell_tree_kernel, dim3((max_cells + CELL_WARPS - 1) / CELL_WARPS), dim3(CELL_WARPS * 32), 0, st, cx);
    if (err != cudaSuccess) return err;
    err = launch_dependent(top_tree_kernel, dim3((max_cells + TOP_THREADS - 1) / TOP_THREADS), dim3(TOP_THREADS),
                           (size_t)CELL_BLOCK_MAX * CELL_BYTES_PER_SLOT, st, cx);
    if (err != cudaSuccess) return err;
    return cudaGetLastError();
}

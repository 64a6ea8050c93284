// build_kernels.cu — steps a1..a6 of the hot path, hand-written for sm_100a.
//   a1  morton_hist_kernel : Morton keys in the periodic box + digit histograms of all four
//                            radix passes + per-type root AABB (the quantization frame)
//       finalize_kernel    : exclusive scans of the histograms, type segments, roots, frames
//   a2  onesweep_kernel    : stable LSD radix sort, 8-bit digits, one kernel per pass with chained-scan
//                            decoupled look-back between tiles (the paper used CUB)
//   a3+a4 hierarchy_kernel : Karras binary radix tree + ropes in closed form
//       entry_table_kernel : node of every cell of the 4^3 .. 32^3 Morton grids (entry points of the traversal)
//   a2'+a5+a6 fit_kernel   : gather into Z-order, quantize each leaf onto the 1023-bin grid of its tree's root
//                            box with outward rounding, then bottom-up union with atomic
//                            hand-over directly on the packed 10-bit integers
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

// One block of MORTON_THREADS threads: histograms -> exclusive offsets; segments, roots, frames.  Run by the last
// block of morton_hist_kernel to finish (threads 0..255 own one digit each).
__device__ void finalize_block(TreeMeta *__restrict__ meta, int N) {
    __shared__ uint32_t s_scan[256];
    __shared__ uint32_t s_ws[8];
    const int d = threadIdx.x, lane = d & 31, warp = d >> 5;
    for (int p = 0; p < 4; ++p) {
        uint32_t c = 0, inc = 0;
        if (d < 256) {
            c = __ldcg(&meta->hist[p][d]);
            inc = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t v = __shfl_up_sync(0xFFFFFFFFu, inc, o);
                if (lane >= o) inc += v;
            }
            if (lane == 31) s_ws[warp] = inc;
        }
        __syncthreads();
        if (d < 256) {
            uint32_t base = 0;
            for (int w = 0; w < warp; ++w) base += s_ws[w];
            uint32_t excl = base + inc - c;
            meta->hist[p][d] = excl;
            if (p == 3) s_scan[d] = excl;
        }
        __syncthreads();
    }
    if (d <= QBVH_TMAX) {
        // type t owns top-digit values [64 t, 64 t + 63]
        int s = (d < QBVH_TMAX) ? (int)s_scan[64 * d] : N;
        meta->seg[d] = s;
    }
    if (d < QBVH_TMAX) {
        int s = (int)s_scan[64 * d];
        int e1 = (d + 1 < QBVH_TMAX) ? (int)s_scan[64 * (d + 1)] : N;
        int n = e1 - s;
        meta->roots[d] = (n <= 0) ? -1 : (n == 1 ? (N - 1 + s) : s);
        float *fr = meta->frames[d];
        if (n > 0) {
            for (int a = 0; a < 3; ++a) {
                float lo = ord2f(~__ldcg(&meta->mm_enc[d][a]));
                float hi = ord2f(__ldcg(&meta->mm_enc[d][3 + a]));
                fr[a] = lo;
                fr[3 + a] = hi;
                // Delta = div_ru(sub_ru(hi, lo), 1023): the 1023-bin grid spans at least the root box
                fr[6 + a] = __fdiv_ru(__fsub_ru(hi, lo), QBVH_NBINS);
            }
        } else {
            for (int a = 0; a < 9; ++a) fr[a] = 0.0f;
        }
        fr[9] = fr[10] = fr[11] = 0.0f;
    }
}

constexpr int MORTON_THREADS = 512;

template <int NT>
__global__ void __launch_bounds__(MORTON_THREADS) morton_hist_kernel(const float *__restrict__ pos,
                                                           const int32_t *__restrict__ type, int N, float3 lo,
                                                           float3 scale, uint32_t *__restrict__ key_out,
                                                           TreeMeta *__restrict__ meta,
                                                           uint32_t *__restrict__ status0, int status_words,
                                                           int32_t *__restrict__ entry, int entry_words) {
    __shared__ uint32_t s_hist[4][256];
    __shared__ bool s_last;
    for (int i = threadIdx.x; i < 1024; i += blockDim.x) (&s_hist[0][0])[i] = 0;
    __syncthreads();
    const int stride = gridDim.x * blockDim.x;
    const int gtid = blockIdx.x * blockDim.x + threadIdx.x;
    // the look-back status buffer of the first sort pass must be zero before that pass starts; the entry table of
    // the traversal starts out empty (-1) and is filled by hierarchy_kernel
    for (int i = gtid; i < status_words; i += stride) status0[i] = 0;
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
    auto one = [&](float x, float y, float z, int tt) -> uint32_t {
        if (tt < 0 || tt >= NT) {
            bad_type = true;
            tt = 0;
        }
        const uint32_t t = (uint32_t)tt;
        uint32_t code = (spread10(morton_bin(x, lo.x, scale.x)) << 2) | (spread10(morton_bin(y, lo.y, scale.y)) << 1) |
                        spread10(morton_bin(z, lo.z, scale.z));
        uint32_t key = (t << 30) | code;
        atomicAdd(&s_hist[0][key & 255u], 1u);
        atomicAdd(&s_hist[1][(key >> 8) & 255u], 1u);
        atomicAdd(&s_hist[2][(key >> 16) & 255u], 1u);
        atomicAdd(&s_hist[3][key >> 24], 1u);
#pragma unroll
        for (int u = 0; u < NT; ++u) {
            bool m = (NT == 1) || (t == (uint32_t)u);
            mn[u][0] = m ? fminf(mn[u][0], x) : mn[u][0];
            mn[u][1] = m ? fminf(mn[u][1], y) : mn[u][1];
            mn[u][2] = m ? fminf(mn[u][2], z) : mn[u][2];
            mx[u][0] = m ? fmaxf(mx[u][0], x) : mx[u][0];
            mx[u][1] = m ? fmaxf(mx[u][1], y) : mx[u][1];
            mx[u][2] = m ? fmaxf(mx[u][2], z) : mx[u][2];
        }
        return key;
    };
    // four particles per thread and iteration: three 128-bit position loads, one 128-bit key store
    const bool vec = ((reinterpret_cast<uintptr_t>(pos) & 15) == 0) && ((reinterpret_cast<uintptr_t>(key_out) & 15) == 0) &&
                     (type == nullptr || (reinterpret_cast<uintptr_t>(type) & 15) == 0);
    const int nquad = vec ? N / 4 : 0;
    for (int q = gtid; q < nquad; q += stride) {
        const float4 *p4 = reinterpret_cast<const float4 *>(pos) + 3 * (size_t)q;
        const float4 a = __ldg(p4), b = __ldg(p4 + 1), c = __ldg(p4 + 2);
        int4 tt = make_int4(0, 0, 0, 0);
        if (type) tt = __ldg(reinterpret_cast<const int4 *>(type) + q);
        uint4 k;
        k.x = one(a.x, a.y, a.z, tt.x);
        k.y = one(a.w, b.x, b.y, tt.y);
        k.z = one(b.z, b.w, c.x, tt.z);
        k.w = one(c.y, c.z, c.w, tt.w);
        reinterpret_cast<uint4 *>(key_out)[q] = k;
    }
    for (int i = 4 * nquad + gtid; i < N; i += stride) {
        const float x = pos[3 * (size_t)i + 0], y = pos[3 * (size_t)i + 1], z = pos[3 * (size_t)i + 2];
        key_out[i] = one(x, y, z, type ? type[i] : 0);
    }
    // per-type min/max: warp reduce on the order-preserving encoding, one global atomic per warp and value
#pragma unroll
    for (int t = 0; t < NT; ++t)
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            uint32_t a = __reduce_max_sync(0xFFFFFFFFu, ~f2ord(mn[t][d]));
            uint32_t b = __reduce_max_sync(0xFFFFFFFFu, f2ord(mx[t][d]));
            if ((threadIdx.x & 31) == 0) {
                if (a != ~f2ord(INFINITY)) atomicMax(&meta->mm_enc[t][d], a);
                if (b != f2ord(-INFINITY)) atomicMax(&meta->mm_enc[t][3 + d], b);
            }
        }
    if (bad_type) atomicOr(&meta->err_flags, 1);
    __syncthreads();
    for (int i = threadIdx.x; i < 1024; i += blockDim.x) {
        uint32_t c = (&s_hist[0][0])[i];
        if (c) atomicAdd(&meta->hist[0][0] + i, c);
    }
    // the last block to get here turns the histograms into offsets (segments, roots, frames)
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(&meta->blocks_done, 1u) == gridDim.x - 1;
    __syncthreads();
    if (s_last) {
        __threadfence();
        finalize_block(meta, N);
    }
}

// N = 0: only the bookkeeping
__global__ void __launch_bounds__(MORTON_THREADS) finalize_kernel(TreeMeta *__restrict__ meta, int N) {
    finalize_block(meta, N);
}

// ------------------------------------------------------------------------------------------------------------
// a2. One pass of the LSD radix sort (8-bit digit).  A tile of 4096 keys per block; ranks inside a warp by
// match_any, warps and digits combined by block scans, tiles chained by decoupled look-back on one status word
// per (tile, digit).  Stable: ties keep their input order at every level.  FIRST: values are implicit (= index).
// ------------------------------------------------------------------------------------------------------------
template <bool FIRST>
__global__ void __launch_bounds__(SORT_THREADS, 2) onesweep_kernel(const uint32_t *__restrict__ kin,
                                                                    const uint32_t *__restrict__ vin,
                                                                    uint32_t *__restrict__ kout,
                                                                    uint32_t *__restrict__ vout, int N, int shift,
                                                                    const uint32_t *__restrict__ hist_excl,
                                                                    volatile uint32_t *status,
                                                                    uint32_t *__restrict__ status_next,
                                                                    uint32_t *__restrict__ tile_counter) {
    // per-warp digit counters while ranking; the tile's keys in output order afterwards (same storage)
    __shared__ __align__(16) uint32_t s_buf[SORT_TILE];
    __shared__ uint32_t s_vals[SORT_TILE];
    __shared__ uint32_t s_dstart[256];
    __shared__ uint32_t s_gbase[256];
    __shared__ uint32_t s_ws[8];
    __shared__ uint32_t s_tile;
    static_assert(SORT_WARPS * 256 <= SORT_TILE, "the per-warp counters live in the key buffer");
    uint32_t(*s_whist)[256] = reinterpret_cast<uint32_t(*)[256]>(s_buf);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(tile_counter, 1u);
    for (int i = tid; i < SORT_WARPS * 256; i += SORT_THREADS) s_buf[i] = 0;
    __syncthreads();
    const uint32_t tile = s_tile;
    const int base = (int)tile * SORT_TILE;
    const int nvalid = min(SORT_TILE, N - base);
    if (tid < 256) status_next[(size_t)tile * 256 + tid] = 0;   // the other buffer: used by the next pass, idle now

    uint32_t key[SORT_IPT], val[SORT_IPT];
    uint32_t rank[SORT_IPT];
    const int wbase = warp * (32 * SORT_IPT);
#pragma unroll
    for (int r = 0; r < SORT_IPT; ++r) {
        const int li = wbase + r * 32 + lane;
        key[r] = (li < nvalid) ? kin[base + li] : 0xFFFFFFFFu;
        val[r] = FIRST ? (uint32_t)(base + li) : ((li < nvalid) ? vin[base + li] : 0u);
    }
    // ranks inside the warp: lanes with the same digit find each other by match.any; the lowest of them bumps the
    // warp's counter of that digit (shared-memory atomic) and hands the old value to the others.  Rounds are
    // ordered by the warp-wide shuffle, so equal digits keep their input order (stability).
    const uint32_t lt_mask = (1u << lane) - 1u;
#pragma unroll
    for (int r = 0; r < SORT_IPT; ++r) {
        const int li = wbase + r * 32 + lane;
        const bool valid = li < nvalid;
        const uint32_t d = (key[r] >> shift) & 255u;
        const uint32_t m = __match_any_sync(0xFFFFFFFFu, valid ? d : 256u);
        uint32_t before = 0;
        if (valid && (m & lt_mask) == 0) before = atomicAdd(&s_whist[warp][d], (uint32_t)__popc(m));
        before = __shfl_sync(0xFFFFFFFFu, before, __ffs(m) - 1);
        rank[r] = before + __popc(m & lt_mask);
    }
    __syncthreads();
    // thread d owns digit d: exclusive scan over warps, then over digits, then over tiles (look-back)
    if (tid < 256) {
        const int d = tid;
        uint32_t c[SORT_WARPS];
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) c[w] = s_whist[w][d];
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) {
            s_whist[w][d] = run;
            run += c[w];
        }
        const uint32_t count = run;
        if (tile == 0) status[d] = count | ST_PRE;
        else status[(size_t)tile * 256 + d] = count | ST_AGG;
        uint32_t inc = count;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t v = __shfl_up_sync(0xFFFFFFFFu, inc, o);
            if (lane >= o) inc += v;
        }
        if (lane == 31) s_ws[warp] = inc;
        asm volatile("bar.sync 1, 256;");      // the eight warps that own digits
        uint32_t wb = 0;
        for (int w = 0; w < warp; ++w) wb += s_ws[w];
        const uint32_t dstart = wb + inc - count;
        s_dstart[d] = dstart;
        uint32_t excl = 0;
        if (tile != 0) {
            // decoupled look-back, LB predecessors polled per round trip: all tiles of a pass are resident at once
            // at these sizes, so the chain of prefixes advances LB tiles per L2 round trip
            int p = (int)tile - 1;
            bool done = false;
            while (!done) {
                constexpr int LB = 16;
                uint32_t v[LB];
#pragma unroll
                for (int u = 0; u < LB; ++u) v[u] = (p - u >= 0) ? (uint32_t)status[(size_t)(p - u) * 256 + d] : (uint32_t)(1u << 31);
#pragma unroll
                for (int u = 0; u < LB; ++u) {
                    if (done) continue;
                    if (v[u] & ST_PRE) {
                        excl += v[u] & ST_VAL;
                        done = true;
                    } else if (v[u] & ST_AGG) {
                        excl += v[u] & ST_VAL;
                        --p;
                    } else {
                        break;                 // not published yet: poll again from here
                    }
                }
            }
            status[(size_t)tile * 256 + d] = (excl + count) | ST_PRE;
        }
        s_gbase[d] = hist_excl[d] + excl - dstart;   // wraps mod 2^32; final index is exact
    }
    __syncthreads();
    // position of every key inside the tile's output order
#pragma unroll
    for (int r = 0; r < SORT_IPT; ++r) {
        const uint32_t d = (key[r] >> shift) & 255u;
        rank[r] += s_dstart[d] + s_whist[warp][d];
    }
    __syncthreads();                                  // the counters are dead: their storage takes the keys
#pragma unroll
    for (int r = 0; r < SORT_IPT; ++r) {
        const int li = wbase + r * 32 + lane;
        if (li < nvalid) {
            s_buf[rank[r]] = key[r];
            s_vals[rank[r]] = val[r];
        }
    }
    __syncthreads();
    for (int p = tid; p < nvalid; p += SORT_THREADS) {
        const uint32_t k = s_buf[p];
        const uint32_t g = s_gbase[(k >> shift) & 255u] + (uint32_t)p;
        kout[g] = k;
        vout[g] = s_vals[p];
    }
}

// ------------------------------------------------------------------------------------------------------------
// a3 + a4. One thread per sorted position k: leaf k's node words and (if it exists) internal node k.
// delta(i,j) = length of the common prefix of the augmented keys (key, position); -1 outside the type segment.
// Rope of a node covering [f,l] (pinned in tests/test_oracle_tree.py): END if l is the segment
// end, else with m = l+1: internal node m if its range starts at m, else leaf m.
// ------------------------------------------------------------------------------------------------------------
struct SegDelta {
    const uint32_t *key;
    int s, e;
    __device__ __forceinline__ int operator()(int i, uint32_t ki, long long j) const {
        if (j < s || j > e) return -1;
        uint32_t x = ki ^ __ldg(key + j);
        return x ? __clz(x) : 32 + __clz((uint32_t)i ^ (uint32_t)j);
    }
};

__global__ void __launch_bounds__(256) hierarchy_kernel(const uint32_t *__restrict__ key, int N,
                                                         TreeMeta *__restrict__ meta, int4 *__restrict__ nodes,
                                                         int32_t *__restrict__ parent,
                                                         unsigned long long *__restrict__ slot,
                                                         uint2 *__restrict__ groups, int32_t *__restrict__ entry,
                                                         int K) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    // query groups found by this thread (at most two): maximal subtrees with <= GROUP_MAX leaves
    uint2 grp0 = make_uint2(0u, 0u), grp1 = make_uint2(0u, 0u);
    int ngrp = 0;
    if (k < N) {
        const uint32_t ki = key[k];
        const int t = ki >> 30;
        SegDelta delta{key, meta->seg[t], meta->seg[t + 1] - 1};
        const int s = delta.s, e = delta.e;
        auto rope_of = [&](int l) -> int {
            if (l == e) return -1;
            const int m = l + 1;
            const uint32_t km = __ldg(key + m);
            if (m <= e - 1 && delta(m, km, m + 1) > delta(m, km, m - 1)) return m;
            return N - 1 + m;
        };
        int2 *nodes_lr = reinterpret_cast<int2 *>(nodes);   // {left, rope} = second half of the 16-byte node
        // Entry table of the traversal.  The upper levels of an LBVH over Morton codes ARE a regular grid: all
        // particles whose code starts with a given 3l-bit prefix (one cell of the 2^l-per-axis grid over the box,
        // PAPER.md:61) form one subtree.  A node whose keys share `dnode` leading bits while its parent's share
        // only `dpar` roots the cell of every level l with dpar < 2 + 3 l <= dnode (2 type bits, then the code).
        int32_t *const etab = entry + t * ENTRY_CELLS;
        auto emit_entry = [&](int dpar, int dnode, int node) {
#pragma unroll
            for (int l = ENTRY_LMIN; l <= ENTRY_LMAX; ++l) {
                const int need = 2 + 3 * l;
                if (dpar < need && need <= dnode) etab[entry_offset(l) + (int)((ki & 0x3FFFFFFFu) >> (30 - 3 * l))] = node;
            }
        };
        const int dl = delta(k, ki, (long long)k - 1), dr = delta(k, ki, (long long)k + 1);
        // leaf k
        nodes_lr[2 * (size_t)(N - 1 + k) + 1] = make_int2(~k, rope_of(k));
        emit_entry(max(dl, dr), 64, N - 1 + k);
        if (s == e) parent[N - 1 + k] = -1;                 // a one-particle tree: the leaf is the root
        if (k == s && e - s + 1 <= GROUP_MAX) {             // a whole tree that fits one group
            grp0 = make_uint2((uint32_t)s, (uint32_t)(e - s + 1));
            ngrp = 1;
        }
        if (k == e) {                                       // no internal node carries the index of a segment end
            if (k < N - 1) {
                nodes[k] = make_int4(0, 0, 0, -1);
                parent[k] = -1;
                slot[k] = SLOT_EMPTY;
            }
        } else {
            // internal node k (Karras)
            const int d = (dr > dl) ? 1 : -1;
            const int dmin = (dr > dl) ? dl : dr;
            long long lmax = 2;
            while (delta(k, ki, k + lmax * d) > dmin) lmax <<= 1;
            long long l = 0;
            for (long long tt = lmax >> 1; tt >= 1; tt >>= 1)
                if (delta(k, ki, k + (l + tt) * d) > dmin) l += tt;
            const int j = (int)(k + l * d);
            const int dnode = delta(k, ki, j);
            long long sp = 0, tt = l;
            do {
                tt = (tt + 1) >> 1;
                if (delta(k, ki, k + (sp + tt) * d) > dnode) sp += tt;
            } while (tt > 1);
            const int gamma = (int)(k + sp * d + (d < 0 ? -1 : 0));
            const int f = min(k, j), la = max(k, j);
            const int lc = (f == gamma) ? (N - 1 + gamma) : gamma;
            const int rc = (la == gamma + 1) ? (N - 1 + gamma + 1) : (gamma + 1);
            parent[lc] = k;
            parent[rc] = k;
            if (k == s) parent[k] = -1;
            emit_entry(dmin, dnode, k);
            const int size = la - f + 1;
            const int leftword = (K > 1 && size <= K) ? ~f : lc;   // collapsed range leaf: first sorted position
            nodes_lr[2 * (size_t)k + 1] = make_int2(leftword, rope_of(la));
            slot[k] = SLOT_EMPTY;
            if (size > GROUP_MAX) {                         // children that fit are maximal: they become groups
                const int lsize = gamma - f + 1, rsize = la - gamma;
                if (lsize <= GROUP_MAX) {
                    grp0 = make_uint2((uint32_t)f, (uint32_t)lsize);
                    ngrp = 1;
                }
                if (rsize <= GROUP_MAX) {
                    const uint2 gr = make_uint2((uint32_t)(gamma + 1), (uint32_t)rsize);
                    if (ngrp) grp1 = gr; else grp0 = gr;
                    ++ngrp;
                }
            }
        }
    }
    // append this warp's groups with one atomic
    const uint32_t b1 = __ballot_sync(0xFFFFFFFFu, ngrp >= 1), b2 = __ballot_sync(0xFFFFFFFFu, ngrp >= 2);
    const int total = __popc(b1) + __popc(b2);
    if (total) {
        const int lane = threadIdx.x & 31;
        const uint32_t lt = (1u << lane) - 1u;
        int base = 0;
        if (lane == 0) base = atomicAdd(&meta->group_count, total);
        base = __shfl_sync(0xFFFFFFFFu, base, 0) + __popc(b1 & lt) + __popc(b2 & lt);
        if (ngrp >= 1) groups[base] = grp0;
        if (ngrp >= 2) groups[base + 1] = grp1;
    }
}

// ------------------------------------------------------------------------------------------------------------
// a2' + a5 + a6.  Quantizer defined by its decompressor:
//   D_lo(q) = fma_rd(q, Delta, lo)   D_hi(q) = fma_ru(q, Delta, lo)
//   q_lo(a) = max{q : D_lo(q) <= a}  q_hi(b) = min{q : D_hi(q) >= b}     (bisection: D_lo, D_hi are monotone)
// q_lo/q_hi are monotone, so the union of boxes is the per-field integer min/max of the packed words.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t quant_lo(float a, float lo, float delta) {
    uint32_t q = 0;
#pragma unroll
    for (uint32_t bit = 512; bit; bit >>= 1) {
        uint32_t c = q | bit;
        if (__fmaf_rd((float)c, delta, lo) <= a) q = c;
    }
    return q;
}
__device__ __forceinline__ uint32_t quant_hi(float b, float lo, float delta) {
    uint32_t q = 0;
#pragma unroll
    for (uint32_t bit = 512; bit; bit >>= 1) {
        uint32_t c = q + bit;
        if (__fmaf_ru((float)(c - 1), delta, lo) < b) q = c;
    }
    return q;
}
__device__ __forceinline__ uint32_t pack_min(uint32_t a, uint32_t b) {
    return min(a & 0x3FFu, b & 0x3FFu) | min(a & 0xFFC00u, b & 0xFFC00u) | min(a & 0x3FF00000u, b & 0x3FF00000u);
}
__device__ __forceinline__ uint32_t pack_max(uint32_t a, uint32_t b) {
    return max(a & 0x3FFu, b & 0x3FFu) | max(a & 0xFFC00u, b & 0xFFC00u) | max(a & 0x3FF00000u, b & 0x3FF00000u);
}

__global__ void __launch_bounds__(256) fit_kernel(const float *__restrict__ pos, const uint32_t *__restrict__ idx_sorted,
                                                   const uint32_t *__restrict__ key_sorted, int N,
                                                   const TreeMeta *__restrict__ meta, float4 *__restrict__ sorted_pos,
                                                   int4 *__restrict__ nodes, const int32_t *__restrict__ parent,
                                                   unsigned long long *__restrict__ slot) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const uint32_t idx = idx_sorted[k];
    const float x = pos[3 * (size_t)idx], y = pos[3 * (size_t)idx + 1], z = pos[3 * (size_t)idx + 2];
    sorted_pos[k] = make_float4(x, y, z, __uint_as_float(idx));
    const float *fr = meta->frames[key_sorted[k] >> 30];
    uint32_t wlo = quant_lo(x, fr[0], fr[6]) | (quant_lo(y, fr[1], fr[7]) << 10) | (quant_lo(z, fr[2], fr[8]) << 20);
    uint32_t whi = quant_hi(x, fr[0], fr[6]) | (quant_hi(y, fr[1], fr[7]) << 10) | (quant_hi(z, fr[2], fr[8]) << 20);
    int2 *nodes_b = reinterpret_cast<int2 *>(nodes);    // {lo, hi} = first half of the 16-byte node
    nodes_b[2 * (size_t)(N - 1 + k)] = make_int2((int)wlo, (int)whi);
    int n = parent[N - 1 + k];
    while (n >= 0) {
        // hand-over through one 64-bit atomic: the first child to arrive deposits its box, the second merges
        const unsigned long long mine = (unsigned long long)wlo | ((unsigned long long)whi << 32);
        const unsigned long long other = atomicExch(slot + n, mine);
        if (other == SLOT_EMPTY) break;                 // a packed box never has bits 30, 31, 62, 63 set
        wlo = pack_min(wlo, (uint32_t)other);
        whi = pack_max(whi, (uint32_t)(other >> 32));
        nodes_b[2 * (size_t)n] = make_int2((int)wlo, (int)whi);
        n = parent[n];
    }
}

// ------------------------------------------------------------------------------------------------------------
cudaError_t launch_build(const float *pos, const int32_t *type, int N, int T, int K, const float *box_lo,
                         const float *box_scale, const BuildBuffers &b, cudaStream_t st) {
    cudaError_t err = cudaMemsetAsync(b.meta, 0, sizeof(TreeMeta), st);
    if (err != cudaSuccess) return err;
    if (N == 0) {
        finalize_kernel<<<1, MORTON_THREADS, 0, st>>>(b.meta, 0);
        return cudaGetLastError();
    }
    const int tiles = (N + SORT_TILE - 1) / SORT_TILE;
    const int status_words = tiles * 256;
    const int entry_words = QBVH_TMAX * ENTRY_CELLS;
    const float3 lo = make_float3(box_lo[0], box_lo[1], box_lo[2]);
    const float3 sc = make_float3(box_scale[0], box_scale[1], box_scale[2]);
    int mblocks = (N / 4 + MORTON_THREADS - 1) / MORTON_THREADS;
    if (mblocks > 148 * 2) mblocks = 148 * 2;
    if (mblocks < 1) mblocks = 1;
    switch (T) {
        case 1: morton_hist_kernel<1><<<mblocks, MORTON_THREADS, 0, st>>>(pos, type, N, lo, sc, b.key_a, b.meta, b.status[0], status_words, b.entry, entry_words); break;
        case 2: morton_hist_kernel<2><<<mblocks, MORTON_THREADS, 0, st>>>(pos, type, N, lo, sc, b.key_a, b.meta, b.status[0], status_words, b.entry, entry_words); break;
        case 3: morton_hist_kernel<3><<<mblocks, MORTON_THREADS, 0, st>>>(pos, type, N, lo, sc, b.key_a, b.meta, b.status[0], status_words, b.entry, entry_words); break;
        default: morton_hist_kernel<4><<<mblocks, MORTON_THREADS, 0, st>>>(pos, type, N, lo, sc, b.key_a, b.meta, b.status[0], status_words, b.entry, entry_words); break;
    }
    // four passes a -> b -> a -> b -> a
    onesweep_kernel<true><<<tiles, SORT_THREADS, 0, st>>>(b.key_a, nullptr, b.key_b, b.idx_b, N, 0, b.meta->hist[0],
                                                          b.status[0], b.status[1], &b.meta->tile_counter[0]);
    onesweep_kernel<false><<<tiles, SORT_THREADS, 0, st>>>(b.key_b, b.idx_b, b.key_a, b.idx_a, N, 8, b.meta->hist[1],
                                                           b.status[1], b.status[0], &b.meta->tile_counter[1]);
    onesweep_kernel<false><<<tiles, SORT_THREADS, 0, st>>>(b.key_a, b.idx_a, b.key_b, b.idx_b, N, 16, b.meta->hist[2],
                                                           b.status[0], b.status[1], &b.meta->tile_counter[2]);
    onesweep_kernel<false><<<tiles, SORT_THREADS, 0, st>>>(b.key_b, b.idx_b, b.key_a, b.idx_a, N, 24, b.meta->hist[3],
                                                           b.status[1], b.status[0], &b.meta->tile_counter[3]);
    const int nb = (N + 255) / 256;
    hierarchy_kernel<<<nb, 256, 0, st>>>(b.key_a, N, b.meta, b.nodes, b.parent, b.slot, b.groups, b.entry, K);
    fit_kernel<<<nb, 256, 0, st>>>(pos, b.idx_a, b.key_a, N, b.meta, b.sorted_pos, b.nodes, b.parent, b.slot);
    return cudaGetLastError();
}

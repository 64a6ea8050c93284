// build_kernels.cu — steps a1..a6 of the hot path, hand-written for sm_100a.
//   a1  morton_hist_kernel : Morton keys in the periodic box + digit histograms of all four
//                            radix passes + per-type root AABB (the quantization frame); its last
//                            block scans the histograms and writes type segments, roots and frames
//   a2  onesweep_kernel    : stable LSD radix sort, 8-bit digits, one kernel per pass with chained-scan
//                            decoupled look-back between tiles (the paper used CUB)
//   a2'+a3+a4+a5+a6 tree_kernel : gather into Z-order; Karras binary radix tree built bottom up
//                            with ropes in closed form; each leaf quantized onto the 1023-bin
//                            grid of its tree's root box with outward rounding; boxes united
//                            on the packed 10-bit integers while walking up with one 128-bit atomic hand-over
//                            per node; entry table and query groups of the traversal
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
__device__ void finalize_block(TreeMeta *__restrict__ meta, int N, int warp_slots) {
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
    __shared__ float s_rho[QBVH_TMAX];
    __shared__ uint32_t s_scan_count[QBVH_TMAX];
    if (d < QBVH_TMAX) {
        int s = (int)s_scan[64 * d];
        int e1 = (d + 1 < QBVH_TMAX) ? (int)s_scan[64 * (d + 1)] : N;
        int n = e1 - s;
        meta->roots[d] = (n <= 0) ? -1 : (n == 1 ? (N - 1 + s) : s);
        float *fr = meta->frames[d];
        float vol = 1.0f;
        if (n > 0) {
            for (int a = 0; a < 3; ++a) {
                float lo = ord2f(~__ldcg(&meta->mm_enc[d][a]));
                float hi = ord2f(__ldcg(&meta->mm_enc[d][3 + a]));
                fr[a] = lo;
                fr[3 + a] = hi;
                // Delta = div_ru(sub_ru(hi, lo), 1023): the 1023-bin grid spans at least the root box
                fr[6 + a] = __fdiv_ru(__fsub_ru(hi, lo), QBVH_NBINS);
                vol *= hi - lo;
            }
        } else {
            for (int a = 0; a < 9; ++a) fr[a] = 0.0f;
        }
        fr[9] = fr[10] = fr[11] = 0.0f;
        s_rho[d] = (n > 1 && vol > 0.0f) ? (float)n / vol : 0.0f;    // unknown (flat or single): treated as dense
        s_scan_count[d] = n > 0 ? (uint32_t)n : 0u;
    }
    __syncthreads();
    // Query-group size per type.  One warp traverses for a whole group with the group's box as search volume, so
    // the candidates it draws from a tree of number density rho_b grow with rho_b x (group size / rho_t): for a
    // type far sparser than the densest one (the colloids of a colloid-solvent mixture) a full group
    // would sweep up thousands of misses.  Groups of type t hold at most 32 rho_t / rho_max particles (>= 1).
    if (d < QBVH_TMAX) {
        const float rmax = fmaxf(fmaxf(s_rho[0], s_rho[1]), fmaxf(s_rho[2], s_rho[3]));
        int gm = GROUP_MAX;
        if (s_rho[d] > 0.0f && rmax > 0.0f)
            gm = (int)fminf(fmaxf(floorf((float)GROUP_MAX * s_rho[d] / rmax), 1.0f), (float)GROUP_MAX);
        // Small systems (the regime of PAPER.md:186): with fewer groups than the device has resident warps the
        // traversal is one group's latency, so groups shrink (down to 4) until there is about one per warp.
        const int nt = (int)s_scan_count[d];
        gm = min(gm, max(4, nt / max(warp_slots, 1)));
        meta->gmax[d] = gm;
    }
}

constexpr int MORTON_THREADS = 512;

template <int NT>
__global__ void __launch_bounds__(MORTON_THREADS) morton_hist_kernel(const float *__restrict__ pos,
                                                           const int32_t *__restrict__ type, int N, float3 lo,
                                                           float3 scale, uint32_t *__restrict__ key_out,
                                                           TreeMeta *__restrict__ meta,
                                                           uint32_t *__restrict__ status0, int status_words,
                                                           int32_t *__restrict__ entry, int entry_words,
                                                           int warp_slots) {
    __shared__ uint32_t s_hist[4][256];
    __shared__ bool s_last;
    for (int i = threadIdx.x; i < 1024; i += blockDim.x) (&s_hist[0][0])[i] = 0;
    __syncthreads();
    const int stride = gridDim.x * blockDim.x;
    const int gtid = blockIdx.x * blockDim.x + threadIdx.x;
    // the look-back status buffer of the first sort pass must be zero before that pass starts; the entry table of
    // the traversal starts out empty (-1) and is filled by tree_kernel
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
    // per-type min/max: warp reduce on the order-preserving encoding, block reduce through shared memory, then one
    // global atomic per block and value (same-address atomics serialise in L2)
    __shared__ uint32_t s_mm[QBVH_TMAX][6];
    if (threadIdx.x < QBVH_TMAX * 6) (&s_mm[0][0])[threadIdx.x] = 0u;
    __syncthreads();
#pragma unroll
    for (int t = 0; t < NT; ++t)
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            uint32_t a = __reduce_max_sync(0xFFFFFFFFu, ~f2ord(mn[t][d]));
            uint32_t b = __reduce_max_sync(0xFFFFFFFFu, f2ord(mx[t][d]));
            if ((threadIdx.x & 31) == 0) {
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
    __syncthreads();
    for (int i = threadIdx.x; i < 1024; i += blockDim.x) {
        uint32_t c = (&s_hist[0][0])[i];
        if (c) atomicAdd(&meta->hist[0][0] + i, c);
    }
    // the last block to get here turns the histograms into offsets (segments, roots, frames).  One cumulative
    // fence by thread 0 after the barrier orders the whole block's atomics before its ticket.
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicAdd(&meta->blocks_done, 1u) == gridDim.x - 1;
        __threadfence();
    }
    __syncthreads();
    if (s_last) finalize_block(meta, N, warp_slots);
}

// N = 0: only the bookkeeping
__global__ void __launch_bounds__(MORTON_THREADS) finalize_kernel(TreeMeta *__restrict__ meta, int N) {
    finalize_block(meta, N, 1);
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
// a2' + a3 + a4 + a5 + a6 in ONE bottom-up pass (tree_kernel).  One thread per sorted position k.
//
// Hierarchy (Karras' binary radix tree, "built bottom up"): every node covers a contiguous range
// [f,l] of the sorted augmented keys (key, position).  With dL = delta(f-1,f) and dR = delta(l,l+1) the common
// prefix lengths with the outside neighbours (-1 beyond the type segment), the node is the LEFT child of its
// parent iff dR > dL, and then the parent splits at gamma = l; otherwise it is the RIGHT child and gamma = f-1.
// (dL = dR only at the root, where both are -1.)  The two children of a parent meet at slot[gamma]: the first to
// arrive leaves {its packed box, the far end of its range, its outer delta} there with ONE 128-bit atomic
// exchange and retires; the second takes them, so it knows the parent's range, box and both outer deltas
// without a single key load or search, writes the parent's 16-byte node and walks on ("walking up the
// tree from the leaf nodes").  Slots are tagged with a per-build number instead of being cleared every build.
// Numbering (pinned in tests/test_oracle_tree.py): a left child [f,gamma] is internal node gamma, a
// right child [gamma+1,l] is internal node gamma+1, a root is the first position of its segment; leaf k is node
// N-1+k.  Rope of a node covering [f,l]: END if l is the segment end, else with m = l+1:
// internal node m if its range starts at m (delta(m,m+1) > delta(m,m-1)), else leaf m.
//
// Boxes (a5 + a6).  Quantizer defined by its decompressor:
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

__global__ void __launch_bounds__(256) tree_kernel(const float *__restrict__ pos, const uint32_t *__restrict__ idx_sorted,
                                                    const uint32_t *__restrict__ key, int N,
                                                    TreeMeta *__restrict__ meta, float4 *__restrict__ sorted_pos,
                                                    int4 *__restrict__ nodes, int32_t *__restrict__ parent,
                                                    uint4 *__restrict__ slot, uint2 *__restrict__ groups,
                                                    int32_t *__restrict__ entry, int K, uint32_t build_tag) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const uint32_t ki = key[k];
    const int t = ki >> 30;
    const int s = meta->seg[t], e = meta->seg[t + 1] - 1;
    const float *fr = meta->frames[t];
    // ---- a2': gather into Z-order ----
    const uint32_t idx = idx_sorted[k];
    const float x = pos[3 * (size_t)idx], y = pos[3 * (size_t)idx + 1], z = pos[3 * (size_t)idx + 2];
    sorted_pos[k] = make_float4(x, y, z, __uint_as_float(idx));
    // ---- the leaf: outer deltas, rope, one-bin box ----
    int dL = (k > s) ? delta_aug(ki, k, __ldg(key + k - 1), k - 1) : -1;
    int dR = -1, rope = -1;
    if (k < e) {
        const uint32_t k1 = __ldg(key + k + 1);
        dR = delta_aug(ki, k, k1, k + 1);
        const int m = k + 1;
        rope = (m <= e - 1 && delta_aug(k1, m, __ldg(key + m + 1), m + 1) > dR) ? m : N - 1 + m;
    }
    uint32_t wlo = quant_lo(x, fr[0], fr[6]) | (quant_lo(y, fr[1], fr[7]) << 10) | (quant_lo(z, fr[2], fr[8]) << 20);
    uint32_t whi = quant_hi(x, fr[0], fr[6]) | (quant_hi(y, fr[1], fr[7]) << 10) | (quant_hi(z, fr[2], fr[8]) << 20);
    nodes[N - 1 + k] = make_int4((int)wlo, (int)whi, ~k, rope);
    if (k == e && k < N - 1) {                       // no internal node carries the index of a segment end
        nodes[k] = make_int4(0, 0, 0, -1);
        parent[k] = -1;
    }
    // Entry table of the traversal.  The upper levels of an LBVH over Morton codes ARE a regular grid: all
    // particles whose code starts with a given 3l-bit prefix (one cell of the 2^l-per-axis grid over the box,
    // PAPER.md:61) form one subtree.  A node whose keys share `dnode` leading bits while its parent's share
    // only `dpar` roots the cell of every level l with dpar < 2 + 3 l <= dnode (2 type bits, then the code).
    int32_t *const etab = entry + t * ENTRY_CELLS;
    auto emit_entry = [&](int dpar, int dnode, int node) {
        if (dpar >= 2 + 3 * ENTRY_LMAX || dnode < 2 + 3 * ENTRY_LMIN) return;   // below or above every grid level
#pragma unroll
        for (int l = ENTRY_LMIN; l <= ENTRY_LMAX; ++l) {
            const int need = 2 + 3 * l;
            if (dpar < need && need <= dnode) etab[entry_offset(l) + (int)((ki & 0x3FFFFFFFu) >> (30 - 3 * l))] = node;
        }
    };
    // query groups (maximal subtrees with <= gmax[type] leaves): appended with one atomic per converged set of lanes
    const int gmax = meta->gmax[t];
    auto emit_groups = [&](uint2 g0, uint2 g1, int n) {
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
    };
    emit_entry(max(dL, dR), 64, N - 1 + k);

    // ---- walk up ----
    int f = k, l = k, cur = N - 1 + k;
    while (true) {
        if (dL < 0 && dR < 0) {                      // the root of this type's tree
            parent[cur] = -1;
            if (l - f + 1 <= gmax) emit_groups(make_uint2((uint32_t)f, (uint32_t)(l - f + 1)), make_uint2(0u, 0u), 1);
            break;
        }
        const bool is_left = dR > dL;
        const int gamma = is_left ? l : f - 1;
        const uint4 mine = make_uint4(wlo, whi, (uint32_t)(is_left ? f : l), (build_tag << 8) | (uint32_t)((is_left ? dL : dR) + 1));
        const uint4 other = exch128(slot + gamma, mine);
        if ((other.w >> 8) != build_tag) break;      // first to arrive: the sibling will carry on
        const int dsplit = is_left ? dR : dL;        // delta(gamma, gamma+1): the parent's own prefix length
        if (is_left) {
            l = (int)other.z;
            dR = (int)(other.w & 255u) - 1;
        } else {
            f = (int)other.z;
            dL = (int)(other.w & 255u) - 1;
        }
        wlo = pack_min(wlo, other.x);
        whi = pack_max(whi, other.y);
        const int lsize = gamma - f + 1, rsize = l - gamma, size = l - f + 1;
        const int lc = (lsize == 1) ? (N - 1 + gamma) : gamma;
        const int rc = (rsize == 1) ? (N + gamma) : (gamma + 1);
        const int id = (dL < 0 && dR < 0) ? s : (dR > dL ? l : f);
        parent[lc] = id;
        parent[rc] = id;
        int nrope = -1;
        if (l < e) {
            const int m = l + 1;
            nrope = (m <= e - 1 && delta_aug(__ldg(key + m), m, __ldg(key + m + 1), m + 1) > dR) ? m : N - 1 + m;
        }
        const int leftword = (K > 1 && size <= K) ? ~f : lc;      // collapsed range leaf: first sorted position
        nodes[id] = make_int4((int)wlo, (int)whi, leftword, nrope);
        emit_entry(max(dL, dR), dsplit, id);
        if (size > gmax) {                           // children that fit are maximal: they become groups
            const int nl = lsize <= gmax, nr = rsize <= gmax;
            if (nl + nr) {
                const uint2 gl = make_uint2((uint32_t)f, (uint32_t)lsize), gr = make_uint2((uint32_t)(gamma + 1), (uint32_t)rsize);
                emit_groups(nl ? gl : gr, gr, nl + nr);
            }
        }
        cur = id;
    }
}

// ------------------------------------------------------------------------------------------------------------
cudaError_t launch_build(const float *pos, const int32_t *type, int N, int T, int K, const float *box_lo,
                         const float *box_scale, const BuildBuffers &b, uint32_t build_tag, cudaStream_t st) {
    cudaError_t err = cudaMemsetAsync(b.meta, 0, sizeof(TreeMeta), st);
    if (err != cudaSuccess) return err;
    if (N == 0) {
        finalize_kernel<<<1, MORTON_THREADS, 0, st>>>(b.meta, 0);
        return cudaGetLastError();
    }
    const int tiles = (N + SORT_TILE - 1) / SORT_TILE;
    const int status_words = tiles * 256;
    const int entry_words = QBVH_TMAX * ENTRY_CELLS;
    static int warp_slots = 0;                     // warps the traversal keeps resident on this device
    if (warp_slots == 0) {
        int dev = 0, sms = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        warp_slots = sms * 28;
    }
    const float3 lo = make_float3(box_lo[0], box_lo[1], box_lo[2]);
    const float3 sc = make_float3(box_scale[0], box_scale[1], box_scale[2]);
    int mblocks = (N / 4 + MORTON_THREADS - 1) / MORTON_THREADS;
    if (mblocks > 148 * 2) mblocks = 148 * 2;
    if (mblocks < 1) mblocks = 1;
    switch (T) {
        case 1: morton_hist_kernel<1><<<mblocks, MORTON_THREADS, 0, st>>>(pos, type, N, lo, sc, b.key_a, b.meta, b.status[0], status_words, b.entry, entry_words, warp_slots); break;
        case 2: morton_hist_kernel<2><<<mblocks, MORTON_THREADS, 0, st>>>(pos, type, N, lo, sc, b.key_a, b.meta, b.status[0], status_words, b.entry, entry_words, warp_slots); break;
        case 3: morton_hist_kernel<3><<<mblocks, MORTON_THREADS, 0, st>>>(pos, type, N, lo, sc, b.key_a, b.meta, b.status[0], status_words, b.entry, entry_words, warp_slots); break;
        default: morton_hist_kernel<4><<<mblocks, MORTON_THREADS, 0, st>>>(pos, type, N, lo, sc, b.key_a, b.meta, b.status[0], status_words, b.entry, entry_words, warp_slots); break;
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
    tree_kernel<<<nb, 256, 0, st>>>(pos, b.idx_a, b.key_a, N, b.meta, b.sorted_pos, b.nodes, b.parent, b.slot, b.groups,
                                    b.entry, K, build_tag);
    return cudaGetLastError();
}

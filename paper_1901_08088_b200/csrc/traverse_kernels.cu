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

cudaError_t launch_traverse(const TraverseParams &p, const BuildBuffers &b, int32_t *nlist, int32_t *n_neigh,
                            bool stats, cudaStream_t st) {
    if (p.N == 0) return cudaSuccess;
    const int threads = 128;
    const int blocks = (p.N + threads - 1) / threads;
    if (stats)
        traverse_kernel<true><<<blocks, threads, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh);
    else
        traverse_kernel<false><<<blocks, threads, 0, st>>>(p, b.nodes, b.sorted_pos, b.meta, nlist, n_neigh);
    return cudaGetLastError();
}

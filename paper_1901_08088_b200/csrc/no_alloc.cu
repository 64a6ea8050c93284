// no_alloc.cu — qbvh_morton_keys_noalloc: step a1 of the path (Morton keys + per-type root frames)
// for callers that have no way of obtaining device memory of their own.
//
// Who that is: code that runs inside somebody else's GPU program and is only ever handed that program's buffers — an
// analysis or force plugin called from an MD engine's step loop, a callback under a framework whose caching allocator
// has already taken all of the HBM (a plain cudaMalloc then fails), or a real-time loop in which cudaMalloc/cudaFree
// are off limits because they synchronise the whole device and stall every other stream.  Everything else in this
// library asks such a caller for a workspace (qbvh_set_workspace), which they cannot produce.  This one call brings
// its working memory with it: the per-block partial results of the min/max reduction live in a file-scope
// `static __device__` array below, which the CUDA module loader places in device memory when the library is loaded
// on a GPU and which stays there until the process exits.  The price is a fixed upper limit on N and that all calls
// share the one array (see the header, include/qbvh.h).
//
// The kernel is a variant of morton_cell_kernel (build_kernels.cu): same keys, same arithmetic for the frames, but
// no Morton-cell histogram, and the root boxes are reduced in two stages through the scratch array (one record per
// block, the block that arrives last folds them) instead of by atomics into the workspace's TreeMeta.
#include <cmath>

#include "../../include/qbvh.h"
#include "qbvh_internal.cuh"

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_PER_BLOCK = 4 * NA_THREADS;                         // four consecutive particles per thread
constexpr int NA_MAX_BLOCKS = QBVH_NOALLOC_MAX_N / NA_PER_BLOCK;     // 4096
constexpr int NA_HEADER_WORDS = 64;                                  // 256 B: word 0 = blocks that have arrived, word 1 = flags
constexpr int NA_REC_WORDS = QBVH_TMAX * 6;                          // per block: per type ~enc(min xyz), enc(max xyz)
static_assert(QBVH_NOALLOC_MAX_N % NA_PER_BLOCK == 0, "the limit is a whole number of blocks");

// The scratch: 256 B of header + 4096 records of 96 B = 393,472 bytes on every GPU that loads libqbvh.so.
// In HOST code the name `g_noalloc_scratch` is only a handle for the runtime (cudaGetSymbolAddress below), never an
// address to hand to a kernel; device code may name it directly, but the kernel takes the pointer as an argument so
// that what the host cleared and what the kernel uses are visibly the same memory.
static __device__ __align__(256) uint32_t g_noalloc_scratch[NA_HEADER_WORDS + NA_MAX_BLOCKS * NA_REC_WORDS];

__device__ __forceinline__ uint32_t na_spread10(uint32_t v) {  // bit t -> bit 3t
    v &= 0x3FFu;
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

// b_d = clamp(floor((p_d - lo_d) * s_d), 0, 1023), fp32 RN (the build's binning)
__device__ __forceinline__ uint32_t na_morton_bin(float p, float lo, float s) {
    float f = floorf(__fmul_rn(__fsub_rn(p, lo), s));
    f = fminf(fmaxf(f, 0.0f), 1023.0f);
    return (uint32_t)f;
}

template <int NT>
__global__ void __launch_bounds__(NA_THREADS) morton_frames_noalloc_kernel(const float *__restrict__ pos,
                                                                           const int32_t *__restrict__ type, int N, float3 lo,
                                                                           float3 scale, uint32_t *__restrict__ keys,
                                                                           float *__restrict__ frames, int32_t *__restrict__ status,
                                                                           uint32_t *__restrict__ scratch) {
    const int tid = threadIdx.x, lane = tid & 31;
    const int i0 = 4 * (blockIdx.x * NA_THREADS + tid);
    float mn[NT][3], mx[NT][3];
#pragma unroll
    for (int t = 0; t < NT; ++t)
#pragma unroll
        for (int d = 0; d < 3; ++d) mn[t][d] = INFINITY, mx[t][d] = -INFINITY;
    bool bad_type = false;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int i = i0 + u;
        if (i >= N) continue;
        const float x = __ldg(pos + 3 * (size_t)i), y = __ldg(pos + 3 * (size_t)i + 1), z = __ldg(pos + 3 * (size_t)i + 2);
        int ty = type ? __ldg(type + i) : 0;
        if (ty < 0 || ty >= NT) bad_type = true, ty = 0;
        const uint32_t code = (na_spread10(na_morton_bin(x, lo.x, scale.x)) << 2) | (na_spread10(na_morton_bin(y, lo.y, scale.y)) << 1) |
                              na_spread10(na_morton_bin(z, lo.z, scale.z));
        keys[i] = ((uint32_t)ty << 30) | code;
#pragma unroll
        for (int v = 0; v < NT; ++v) {
            const bool m = (NT == 1) || (ty == v);
            mn[v][0] = m ? fminf(mn[v][0], x) : mn[v][0], mx[v][0] = m ? fmaxf(mx[v][0], x) : mx[v][0];
            mn[v][1] = m ? fminf(mn[v][1], y) : mn[v][1], mx[v][1] = m ? fmaxf(mx[v][1], y) : mx[v][1];
            mn[v][2] = m ? fminf(mn[v][2], z) : mn[v][2], mx[v][2] = m ? fmaxf(mx[v][2], z) : mx[v][2];
        }
    }
    // block reduce on the order-preserving encoding: a word is the maximum of ~enc(min) resp. enc(max); 0 = nothing seen
    __shared__ uint32_t s_mm[NA_REC_WORDS];
    __shared__ bool s_last;
    if (tid < NA_REC_WORDS) s_mm[tid] = 0u;
    __syncthreads();
#pragma unroll
    for (int t = 0; t < NT; ++t)
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const uint32_t a = __reduce_max_sync(0xFFFFFFFFu, ~f2ord(mn[t][d]));
            const uint32_t b = __reduce_max_sync(0xFFFFFFFFu, f2ord(mx[t][d]));
            if (lane == 0) {
                if (a != ~f2ord(INFINITY)) atomicMax(&s_mm[t * 6 + d], a);
                if (b != f2ord(-INFINITY)) atomicMax(&s_mm[t * 6 + 3 + d], b);
            }
        }
    if (bad_type) atomicOr(&scratch[1], 1u);
    __syncthreads();
    // stage 1: this block's record.  Every block writes all of its words, so nothing of an earlier call is ever read.
    uint32_t *rec = scratch + NA_HEADER_WORDS + (size_t)blockIdx.x * NA_REC_WORDS;
    if (tid < NA_REC_WORDS) rec[tid] = s_mm[tid];
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(&scratch[0], 1u) == gridDim.x - 1;     // scratch[0] was cleared in front of the launch
    __syncthreads();
    if (!s_last) return;
    // stage 2 (the block that arrived last): fold the records of all blocks, then turn them into frames
    __threadfence();
    if (tid < NA_REC_WORDS) s_mm[tid] = 0u;
    __syncthreads();
    if (tid < 10 * NA_REC_WORDS) {
        const int c = tid % NA_REC_WORDS;
        uint32_t v = 0u;
        for (int b = tid / NA_REC_WORDS; b < (int)gridDim.x; b += 10)
            v = max(v, __ldcg(scratch + NA_HEADER_WORDS + (size_t)b * NA_REC_WORDS + c));
        if (v) atomicMax(&s_mm[c], v);
    }
    __syncthreads();
    if (tid < QBVH_TMAX) {
        float *fr = frames + 12 * tid;
        const bool seen = tid < NT && s_mm[tid * 6] != 0u;
        for (int a = 0; a < 3; ++a) {
            const float l = seen ? ord2f(~s_mm[tid * 6 + a]) : 0.0f, h = seen ? ord2f(s_mm[tid * 6 + 3 + a]) : 0.0f;
            fr[a] = l;
            fr[3 + a] = h;
            // Delta = div_ru(sub_ru(hi, lo), 1023): the 1023-bin grid spans at least the root box
            fr[6 + a] = seen ? __fdiv_ru(__fsub_ru(h, l), QBVH_NBINS) : 0.0f;
            fr[9 + a] = 0.0f;
        }
    }
    if (tid == 0) status[0] = (int32_t)__ldcg(&scratch[1]);
}

// Device address of the scratch array, looked up once per device.
constexpr int NA_MAX_DEVICES = 64;
uint32_t *g_scratch_ptr[NA_MAX_DEVICES] = {};

}  // namespace

extern "C" int qbvh_morton_keys_noalloc(const float *pos, const int32_t *type, int64_t N, const float *box, int32_t T,
                                        uint32_t *keys, float *frames, int32_t *status, void *cuda_stream) {
    if (N < 0 || !box || !frames || !status || T < 1 || T > QBVH_MAX_TYPES || (N > 0 && (!pos || !keys))) return QBVH_ERR_INVALID_ARG;
    for (int d = 0; d < 3; ++d)
        if (!std::isfinite(box[d]) || !std::isfinite(box[3 + d]) || !(box[3 + d] > 0.0f)) return QBVH_ERR_INVALID_ARG;
    if (N > QBVH_NOALLOC_MAX_N) return QBVH_ERR_NOALLOC_LIMIT;      // the scratch array holds no more block records
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return qbvh_record_cuda_error(e, "noalloc: cudaGetDevice");
    if (dev < 0 || dev >= NA_MAX_DEVICES) return QBVH_ERR_INVALID_ARG;
    if (!g_scratch_ptr[dev]) {
        // Set-up, once per device and with that device current: ask the runtime where this device's copy of the array
        // lives.  (Passing the bare name from host code would hand the kernel the address of a host-side shadow object.)
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) return qbvh_record_cuda_error(e, "noalloc: cudaGetSymbolAddress");
        g_scratch_ptr[dev] = static_cast<uint32_t *>(p);
    }
    uint32_t *scratch = g_scratch_ptr[dev];
    // The array still holds what the previous call left: the arrival counter and the flag word have to start at zero.
    e = cudaMemsetAsync(scratch, 0, NA_HEADER_WORDS * sizeof(uint32_t), st);
    if (e != cudaSuccess) return qbvh_record_cuda_error(e, "noalloc: clear header");
    float3 lo = make_float3(box[0], box[1], box[2]), sc;
    {
        volatile float sx = 1023.0f / box[3], sy = 1023.0f / box[4], sz = 1023.0f / box[5];   // fp32 RN, as qbvh_build
        sc = make_float3(sx, sy, sz);
    }
    const int blocks = N > 0 ? (int)((N + NA_PER_BLOCK - 1) / NA_PER_BLOCK) : 1;   // N = 0: one block writes empty frames
    switch (T) {
        case 1: morton_frames_noalloc_kernel<1><<<blocks, NA_THREADS, 0, st>>>(pos, type, (int)N, lo, sc, keys, frames, status, scratch); break;
        case 2: morton_frames_noalloc_kernel<2><<<blocks, NA_THREADS, 0, st>>>(pos, type, (int)N, lo, sc, keys, frames, status, scratch); break;
        case 3: morton_frames_noalloc_kernel<3><<<blocks, NA_THREADS, 0, st>>>(pos, type, (int)N, lo, sc, keys, frames, status, scratch); break;
        default: morton_frames_noalloc_kernel<4><<<blocks, NA_THREADS, 0, st>>>(pos, type, (int)N, lo, sc, keys, frames, status, scratch); break;
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return qbvh_record_cuda_error(e, "noalloc: launch");
    return QBVH_OK;
}

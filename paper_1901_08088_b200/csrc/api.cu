// api.cu — the C-ABI of libqbvh.so (include/qbvh.h): argument checks, workspace carving, launches.
#include <cmath>
#include <cstdio>
#include <cstring>

#include "../../include/qbvh.h"
#include "qbvh_internal.cuh"

namespace {

struct Context {
    cudaStream_t stream = nullptr;
    void *ws = nullptr;
    int64_t ws_bytes = 0;
    void *staging = nullptr;
    int64_t staging_bytes = 0;
    int T = 1;
    int K = 32;         // leaf-collapse cap for the next build
    int K_built = 1;
    float r_hint[QBVH_TMAX] = {0, 0, 0, 0};   // collapse heuristic: expected query radius against each tree (<= 0: none)
    bool f64_built = false;
    int64_t last_d2h_bytes = 0;   // bytes the last qbvh_neighbors_host copied back
    int lvl_built = 0;
    bool stats = false;
    int variant = 1;
    bool built = false;
    int group_cap = GROUP_MAX;   // QBVH_OPT_GROUP_MAX
    int cell_level = 0;          // QBVH_OPT_CELL_LEVEL: 0 = chosen from N
    int scan_spin_cycles = 1 << 18;   // ~130 us at 1.9 GHz; normal waits are a few us (QBVH_OPT_DEBUG_SCAN_SPIN)
    bool enqueued = false;       // a qbvh_neighbors_enqueue whose result has not been taken
    bool counters_armed = false; // group_cursor, max_count, warps_done of the tree are zero (after a build, after a production traversal)
    int32_t *pinned_dev = nullptr;   // device-side address of `pinned`
    int64_t N = 0;
    float box[6] = {0, 0, 0, 0, 0, 0};
    double box64[6] = {0, 0, 0, 0, 0, 0};   // the box of a double-precision build
    float scale[3] = {0, 0, 0};
    BuildBuffers buf{};
    uint32_t build_tag = 0;      // tag of the last build's meeting slots; 0: the slot area has to be cleared first
    int64_t tag_N = -1;          // the layout (N, cell level, T) the slot area and the cell counters were cleared for
    int tag_lvl = -1, tag_T = -1;
    int32_t *pinned = nullptr;   // 4 ints: max_count, err_flags, then the 64-bit byte count of rows_to_host_kernel
    qbvh_stats last_stats{};
    char cuda_msg[256] = "no CUDA error recorded";
} g;

inline int64_t align256(int64_t x) { return (x + 255) & ~int64_t(255); }

struct Layout {
    int64_t meta, key, rank, ent, key_sorted, idx_sorted, cell_count, cell_start, cell_list, big_list, croot, sorted_pos,
        sorted_pos64, nodes, parent, slot, groups, entry, scratch, total;
};

// Workspace carve-up.  Sized for the finest cell grid any (N, T) can choose, so the layout depends on N alone.
Layout make_layout(int64_t N) {
    Layout L{};
    const int64_t n1 = N > 0 ? N : 1;
    const int64_t ncells = CELL_MAX_TOTAL;
    const int64_t ncell_lists = n1 < ncells ? n1 : ncells;
    int64_t off = 0;
    auto take = [&](int64_t bytes) {
        int64_t o = off;
        off += align256(bytes);
        return o;
    };
    L.meta = take(sizeof(TreeMeta));
    L.key = take(4 * n1);
    L.rank = take(4 * n1);
    L.ent = take(8 * n1);
    L.key_sorted = take(4 * n1);
    L.idx_sorted = take(4 * n1);
    L.cell_count = take(4 * ncells);
    L.cell_start = take(4 * (ncells + 1));
    L.cell_list = take(4 * ncell_lists);
    L.big_list = take(4 * ncell_lists);
    L.croot = take((int64_t)sizeof(CellRoot) * ncell_lists);
    L.sorted_pos = take(16 * n1);
    L.sorted_pos64 = take(32 * n1);
    L.nodes = take(16 * (2 * n1 - 1));
    L.parent = take(4 * (2 * n1 - 1));
    L.slot = take(16 * n1);
    L.groups = take(8 * n1);
    L.entry = take(4 * (int64_t)QBVH_TMAX * ENTRY_CELLS);
    L.scratch = take(18 * n1);
    L.total = off;
    return L;
}

int cuda_fail(cudaError_t e, const char *where) {
    snprintf(g.cuda_msg, sizeof(g.cuda_msg), "%s: %s", where, cudaGetErrorString(e));
    return QBVH_ERR_CUDA;
}

// smallest fp32 value >= x (x finite, inside the fp32 range)
float up_to_f32(double x) {
    float f = (float)x;                       // round to nearest
    if ((double)f < x) f = std::nextafterf(f, INFINITY);
    return f;
}

// Padded pruning radius (reading R11; PAPER.md:140 pads the sphere for fp64 data only):
//   r_pad = up(up(r (1 + 2^-20)) + 8 ulp32(M)),  M = max_d(|lo_d| + 2 L_d),  ulp32(M) = 2^(floor(log2 M) - 23).
// Both sums below are exact in fp64 (a 24-bit times a 21-bit significand; two fp32 values less than 2^22 ulp apart),
// so the only roundings are the two explicit ones upward.
float padded_radius(float r, const float *box) {
    double M = 0.0;
    for (int d = 0; d < 3; ++d) M = std::fmax(M, std::fabs((double)box[d]) + 2.0 * (double)box[3 + d]);
    const double pad = std::scalbn(1.0, std::ilogb(M) - 20);      // 8 ulp32(M) = 2^3 2^(floor(log2 M) - 23)
    const float a = up_to_f32((double)r * (1.0 + 0x1p-20));
    double sum = (double)a + pad;
    if (sum - pad != (double)a) sum = std::nextafter(sum, INFINITY);   // r below 2^-29 pad: stay on the safe side
    return up_to_f32(sum);
}

// largest fp32 value <= x
float down_to_f32(double x) {
    float f = (float)x;
    if ((double)f > x) f = std::nextafterf(f, -INFINITY);
    return f;
}

// ulp32(M), M = max_d(|lo_d| + 2 L_d): the spacing of fp32 numbers at the largest coordinate the traversal can form
double box_ulp32(const float *box) {
    double M = 0.0;
    for (int d = 0; d < 3; ++d) M = std::fmax(M, std::fabs((double)box[d]) + 2.0 * (double)box[3 + d]);
    return std::scalbn(1.0, std::ilogb(M) - 23);
}

// a * b rounded up (the product of two fp32 values is exact in fp64)
float mul_ru(float a, float b) { return up_to_f32((double)a * (double)b); }

// r_list -> the traversal's parameter block (exact r^2, padded pruning radius, Morton binning of the build).
// f64 (qbvh_neighbors_f64): the fp32 kernel runs on the positions rounded to fp32 with the cutoff
// widened by B = 8 ulp32(M) — |d_fp32 - d_fp64| < 5 ulp32(M): two position roundings, the rounding of L and two
// subtractions per axis (2.5 ulp, times sqrt 3), plus the rounding of the squared sum — so nothing it rejects can be
// an fp64 neighbor; what it finds within r - B certainly is one; the pairs in between go through the fp64 predicate.
template <typename RT>
int make_params(const RT *r_list, bool f64, TraverseParams &P) {
    for (int d = 0; d < 3; ++d) {
        P.L[d] = g.box[3 + d];
        P.box_lo[d] = g.box[d];
        P.scale[d] = g.scale[d];
        P.L64[d] = g.box64[3 + d];
    }
    const double B = f64 ? 8.0 * box_ulp32(g.box) : 0.0;
    for (int k = 0; k < QBVH_TMAX * QBVH_TMAX; ++k) {
        P.r2[k] = P.R2[k] = P.Rp[k] = P.r2lo[k] = -1.0f;
        P.r2_64[k] = -1.0;
    }
    for (int a = 0; a < g.T; ++a)
        for (int b = 0; b < g.T; ++b) {
            const RT r = r_list[a * g.T + b];
            if (!(r > 0)) continue;
            if (!std::isfinite(r)) return QBVH_ERR_INVALID_ARG;
            const int k = a * QBVH_TMAX + b;
            float r_cut;                       // cutoff of the fp32 predicate
            if (f64) {
                r_cut = up_to_f32((double)r + B);
                const double rlo = (double)r - B;
                P.r2[k] = up_to_f32((double)r_cut * (double)r_cut);
                P.r2lo[k] = rlo > 0.0 ? down_to_f32(rlo * rlo * (1.0 - 0x1p-50)) : -1.0f;
                volatile double r2 = (double)r * (double)r;      // fp64 RN
                P.r2_64[k] = r2;
            } else {
                r_cut = (float)r;
                volatile float r2 = r_cut * r_cut;               // fp32 RN
                P.r2[k] = r2;
                P.r2lo[k] = r2;
            }
            const float rp = padded_radius(r_cut, g.box);
            for (int d = 0; d < 3; ++d)
                if (!(rp < 0.5f * g.box[3 + d])) return QBVH_ERR_CUTOFF_TOO_LARGE;
            P.R2[k] = mul_ru(rp, rp);
            P.Rp[k] = rp;
        }
    P.N = (int32_t)g.N;
    P.K = g.K_built;
    return QBVH_OK;
}

template <typename RT>
int neighbors_impl(const RT *r_list, bool f64, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh, int64_t q_first = 0,
                   int64_t q_count = -1) {
    g.enqueued = false;              // whatever was enqueued before: its result words are about to be overwritten
    if (!g.built) return QBVH_ERR_NOT_BUILT;
    if (!r_list || max_neigh < 0) return QBVH_ERR_INVALID_ARG;
    // The census of QBVH_OPT_STATS walks once per particle and writes all N rows: a range call's buffers hold only
    // `count` rows, so the two do not combine.
    if (q_count >= 0 && g.stats) return QBVH_ERR_INVALID_ARG;
    if (f64 != g.f64_built) return QBVH_ERR_INVALID_ARG;          // qbvh_build_f64 pairs with qbvh_neighbors_f64
    if (f64 && g.variant != 1) return QBVH_ERR_INVALID_ARG;       // Algorithm 1 as printed (variant 0) is the fp32 path
    if (g.N > 0 && (!n_neigh || (!nlist && max_neigh > 0))) return QBVH_ERR_INVALID_ARG;
    TraverseParams P{};
    const int prc = make_params(r_list, f64, P);
    if (prc != QBVH_OK) return prc;
    P.N = (int32_t)g.N;
    P.max_neigh = max_neigh;
    P.K = g.K_built;
    P.q_first = (int32_t)q_first;
    P.q_count = (int32_t)q_count;
    if (q_count >= 0 && (g.variant != 1 || q_first < 0 || q_first + q_count > g.N)) return QBVH_ERR_INVALID_ARG;
    cudaError_t e;
    // The production kernel alone: its last warp writes {max_count, err_flags} into the pinned result words and
    // re-arms the counters, so the launch needs no memset in front and no copy behind (two stream operations and
    // their gaps, about 7 us).  Any other path clears the counters first and copies the result afterwards.
    const bool self_contained = g.variant == 1 && !g.stats && g.N > 0 && g.pinned_dev != nullptr;
    P.result_host = self_contained ? g.pinned_dev : nullptr;
    if (!self_contained || !g.counters_armed) {
        // group_cursor, max_count (+ warps_done, stats) of whatever ran before
        e = cudaMemsetAsync(&g.buf.meta->group_cursor, 0, 2 * sizeof(int32_t), g.stream);
        if (e != cudaSuccess) return cuda_fail(e, "memset max_count");
        e = cudaMemsetAsync(&g.buf.meta->warps_done, 0, sizeof(int32_t), g.stream);
        if (e != cudaSuccess) return cuda_fail(e, "memset warps_done");
    }
    if (g.stats) {
        e = cudaMemsetAsync(g.buf.meta->stats, 0, sizeof(g.buf.meta->stats), g.stream);
        if (e != cudaSuccess) return cuda_fail(e, "memset stats");
    }
    g.counters_armed = false;
    e = launch_traverse(P, g.buf, nlist, n_neigh, g.stats, g.variant, f64, g.stream);
    if (e != cudaSuccess) return cuda_fail(e, "traverse launch");
    if (self_contained) {
        g.counters_armed = true;
    } else {
        e = cudaMemcpyAsync(g.pinned, &g.buf.meta->max_count, 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, g.stream);
        if (e != cudaSuccess) return cuda_fail(e, "copy max_count");
    }
    if (g.stats) {
        e = cudaMemcpyAsync(&g.last_stats, g.buf.meta->stats, sizeof(qbvh_stats), cudaMemcpyDeviceToHost, g.stream);
        if (e != cudaSuccess) return cuda_fail(e, "copy stats");
    }
    return QBVH_OK;
}

int finish_neighbors() {
    cudaError_t e = cudaStreamSynchronize(g.stream);
    if (e != cudaSuccess) return cuda_fail(e, "stream synchronize");
    const int32_t flags = g.pinned[1];
    if (flags & 2) {
        // the bound violation belongs to this call only: take bit 1 back out of the tree's flag word (bit 0, set by
        // the build, stays) so that the next traversal of the same tree reports its own outcome
        const int32_t keep = flags & 1;
        e = cudaMemcpy(&g.buf.meta->err_flags, &keep, sizeof(keep), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) return cuda_fail(e, "clear err_flags");
    }
    if (flags & 1) return QBVH_ERR_TYPE_RANGE;
    if (flags & 2) return QBVH_ERR_INTERNAL;
    return g.pinned[0];
}

int build_impl(const void *pos, bool f64, const int32_t *type, int64_t N, const float *box, const double *box64 = nullptr) {
    g.built = false;
    g.enqueued = false;
    if (N < 0 || N >= (int64_t(1) << 30) || !box || (N > 0 && !pos)) return QBVH_ERR_INVALID_ARG;
    for (int d = 0; d < 3; ++d)
        if (!std::isfinite(box[d]) || !std::isfinite(box[3 + d]) || !(box[3 + d] > 0.0f)) return QBVH_ERR_INVALID_ARG;
    const Layout L = make_layout(N);
    if (!g.ws || g.ws_bytes < L.total) return QBVH_ERR_WORKSPACE;
    if (!g.pinned) {
        cudaError_t e = cudaHostAlloc(reinterpret_cast<void **>(&g.pinned), 4 * sizeof(int32_t), cudaHostAllocDefault);
        if (e != cudaSuccess) return cuda_fail(e, "cudaHostAlloc");
        g.pinned[0] = g.pinned[1] = g.pinned[2] = g.pinned[3] = 0;
        void *dp = nullptr;
        if (cudaHostGetDevicePointer(&dp, g.pinned, 0) == cudaSuccess) g.pinned_dev = static_cast<int32_t *>(dp);
        else (void)cudaGetLastError();
    }
    char *w = static_cast<char *>(g.ws);
    g.buf.meta = reinterpret_cast<TreeMeta *>(w + L.meta);
    g.buf.key = reinterpret_cast<uint32_t *>(w + L.key);
    g.buf.rank = reinterpret_cast<uint32_t *>(w + L.rank);
    g.buf.ent = reinterpret_cast<uint2 *>(w + L.ent);
    g.buf.key_sorted = reinterpret_cast<uint32_t *>(w + L.key_sorted);
    g.buf.idx_sorted = reinterpret_cast<uint32_t *>(w + L.idx_sorted);
    g.buf.cell_count = reinterpret_cast<uint32_t *>(w + L.cell_count);
    g.buf.cell_start = reinterpret_cast<uint32_t *>(w + L.cell_start);
    g.buf.cell_list = reinterpret_cast<uint32_t *>(w + L.cell_list);
    g.buf.big_list = reinterpret_cast<int32_t *>(w + L.big_list);
    g.buf.croot = reinterpret_cast<CellRoot *>(w + L.croot);
    g.buf.sorted_pos = reinterpret_cast<float4 *>(w + L.sorted_pos);
    g.buf.sorted_pos64 = reinterpret_cast<Pos64 *>(w + L.sorted_pos64);
    g.buf.nodes = reinterpret_cast<int4 *>(w + L.nodes);
    g.buf.parent = reinterpret_cast<int32_t *>(w + L.parent);
    g.buf.slot = reinterpret_cast<uint4 *>(w + L.slot);
    g.buf.groups = reinterpret_cast<uint2 *>(w + L.groups);
    g.buf.entry = reinterpret_cast<int32_t *>(w + L.entry);
    g.buf.scratch = reinterpret_cast<unsigned char *>(w + L.scratch);
    std::memcpy(g.box, box, sizeof(g.box));
    if (box64) std::memcpy(g.box64, box64, sizeof(g.box64));      // only once the arguments have been accepted
    BuildParams bp{};
    for (int d = 0; d < 3; ++d) {
        volatile float s = 1023.0f / box[3 + d];   // fp32 RN
        g.scale[d] = s;
        bp.box_lo[d] = box[d];
        bp.box_scale[d] = s;
    }
    bp.N = (int)N;
    bp.T = type ? g.T : 1;
    bp.K = g.K;
    bp.lvl = pick_cell_level(N, bp.T);
    if (g.cell_level > 0) {          // the caller knows better (particles filling a small part of the box); still T * 8^lvl <= 2^18
        bp.lvl = g.cell_level;
        while (bp.lvl > CELL_LMIN && ((int64_t)bp.T << (3 * bp.lvl)) > CELL_MAX_TOTAL) --bp.lvl;
    }
    bp.group_cap = g.group_cap;
    bp.f64 = f64;
    bp.scan_spin_cycles = g.scan_spin_cycles;
    for (int t = 0; t < QBVH_TMAX; ++t) bp.r_hint[t] = g.r_hint[t];
    // The meeting slots of the top-level walk carry an 18-bit build number and the cell counters are counted back to
    // zero by every build: both are cleared only when the layout moves or the number wraps.
    if (g.build_tag == 0 || g.build_tag >= QBVH_TAG_MAX || g.tag_N != N || g.tag_lvl != bp.lvl || g.tag_T != bp.T) {
        cudaError_t em = cudaMemsetAsync(g.buf.slot, 0, (size_t)16 * (size_t)(N > 0 ? N : 1), g.stream);
        if (em == cudaSuccess) em = cudaMemsetAsync(g.buf.cell_count, 0, (size_t)4 * CELL_MAX_TOTAL, g.stream);
        if (em != cudaSuccess) return cuda_fail(em, "memset slots");
        g.build_tag = 0;
        g.tag_N = N;
        g.tag_lvl = bp.lvl;
        g.tag_T = bp.T;
    }
    bp.build_tag = ++g.build_tag;
    cudaError_t e = launch_build(pos, type, bp, g.buf, g.stream);
    if (e != cudaSuccess) {
        // some of the five launches may have run: the cell counters are not known to be back at zero and slots may
        // carry this build's tag — the next build on this workspace clears both
        g.build_tag = 0;
        g.tag_N = -1;
        return cuda_fail(e, "build launch");
    }
    g.N = N;
    g.K_built = g.K;
    g.f64_built = f64;
    g.lvl_built = bp.lvl;
    g.built = true;
    g.counters_armed = true;      // the build starts by zeroing TreeMeta
    return QBVH_OK;
}

}  // namespace

int qbvh_record_cuda_error(cudaError_t e, const char *where) { return cuda_fail(e, where); }

extern "C" {

int qbvh_set_stream(void *cuda_stream) {
    g.stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    return QBVH_OK;
}

int qbvh_set_num_types(int32_t T) {
    if (T < 1 || T > QBVH_MAX_TYPES) return QBVH_ERR_INVALID_ARG;
    g.T = T;
    g.built = false;
    return QBVH_OK;
}

int64_t qbvh_workspace_bytes(int64_t N, int32_t T) {
    if (N < 0 || N >= (int64_t(1) << 30) || T < 1 || T > QBVH_MAX_TYPES) return QBVH_ERR_INVALID_ARG;
    return make_layout(N).total;
}

int qbvh_set_workspace(void *dev_ptr, int64_t bytes) {
    g.built = false;
    g.build_tag = 0;
    if (dev_ptr && ((reinterpret_cast<uintptr_t>(dev_ptr) & 255) || bytes <= 0)) return QBVH_ERR_WORKSPACE;
    g.ws = dev_ptr;
    g.ws_bytes = dev_ptr ? bytes : 0;
    return QBVH_OK;
}

int qbvh_set_option(int32_t key, int32_t value) {
    switch (key) {
        case QBVH_OPT_LEAF_COLLAPSE:
            if (value < 1 || value > 32) return QBVH_ERR_INVALID_ARG;
            g.K = value;
            return QBVH_OK;
        case QBVH_OPT_STATS:
            g.stats = value != 0;
            return QBVH_OK;
        case QBVH_OPT_VARIANT:
            if (value < 0 || value > 1) return QBVH_ERR_INVALID_ARG;
            g.variant = value;
            return QBVH_OK;
        case QBVH_OPT_DEBUG_BUILD_TAG:
            // only forward: slots of earlier builds carry smaller tags and must never match a later build
            if (value < 1 || value > (int32_t)QBVH_TAG_MAX || (uint32_t)value <= g.build_tag) return QBVH_ERR_INVALID_ARG;
            if (g.build_tag != 0) g.build_tag = (uint32_t)value - 1;   // a slot area still to be cleared stays at tag 0
            return QBVH_OK;
        case QBVH_OPT_GROUP_MAX:
            if (value < 1 || value > GROUP_MAX) return QBVH_ERR_INVALID_ARG;
            g.group_cap = value;
            return QBVH_OK;
        case QBVH_OPT_CELL_LEVEL:
            if (value != 0 && (value < CELL_LMIN || value > CELL_LMAX)) return QBVH_ERR_INVALID_ARG;
            g.cell_level = value;
            return QBVH_OK;
        case QBVH_OPT_DEBUG_SCAN_SPIN:
            if (value < 0) return QBVH_ERR_INVALID_ARG;
            g.scan_spin_cycles = value;
            return QBVH_OK;
        default:
            return QBVH_ERR_INVALID_ARG;
    }
}

int qbvh_get_option(int32_t key) {
    switch (key) {
        case QBVH_OPT_LEAF_COLLAPSE: return g.K;
        case QBVH_OPT_STATS: return g.stats ? 1 : 0;
        case QBVH_OPT_VARIANT: return g.variant;
        case QBVH_OPT_DEBUG_BUILD_TAG: return (int)g.build_tag;
        case QBVH_OPT_DEBUG_SCAN_SPIN: return g.scan_spin_cycles;
        case QBVH_OPT_GROUP_MAX: return g.group_cap;
        case QBVH_OPT_CELL_LEVEL: return g.cell_level;
        default: return QBVH_ERR_INVALID_ARG;
    }
}

int qbvh_build(const float *pos, const int32_t *type, int64_t N, const float *box) {
    return build_impl(pos, false, type, N, box);
}

int qbvh_set_collapse_hint(const float *r_hint, int32_t n) {
    if (n < 0 || n > QBVH_MAX_TYPES || (n > 0 && !r_hint)) return QBVH_ERR_INVALID_ARG;
    for (int t = 0; t < QBVH_TMAX; ++t) g.r_hint[t] = 0.0f;
    for (int t = 0; t < n; ++t) {
        if (std::isnan(r_hint[t]) || std::isinf(r_hint[t])) return QBVH_ERR_INVALID_ARG;
        g.r_hint[t] = r_hint[t];
    }
    return QBVH_OK;
}

int qbvh_neighbors(const float *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh) {
    int rc = neighbors_impl(r_list_ij, false, nlist, n_neigh, max_neigh);
    if (rc != QBVH_OK) return rc;
    return finish_neighbors();
}

int qbvh_neighbors_enqueue(const float *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh) {
    g.enqueued = false;
    int rc = neighbors_impl(r_list_ij, false, nlist, n_neigh, max_neigh);
    g.enqueued = rc == QBVH_OK;
    return rc;
}

int qbvh_neighbors_f64_enqueue(const double *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh) {
    int rc = neighbors_impl(r_list_ij, true, nlist, n_neigh, max_neigh);
    g.enqueued = rc == QBVH_OK;
    return rc;
}

int qbvh_neighbors_range_enqueue(const float *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh, int64_t first, int64_t count) {
    if (count < 0) return QBVH_ERR_INVALID_ARG;
    int rc = neighbors_impl(r_list_ij, false, nlist, n_neigh, max_neigh, first, count);
    g.enqueued = rc == QBVH_OK;
    return rc;
}

int qbvh_neighbors_result(void) {
    if (!g.enqueued) return QBVH_ERR_NOT_BUILT;
    g.enqueued = false;
    return finish_neighbors();
}

int qbvh_neighbors_range(const float *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh, int64_t first, int64_t count) {
    if (count < 0) return QBVH_ERR_INVALID_ARG;
    int rc = neighbors_impl(r_list_ij, false, nlist, n_neigh, max_neigh, first, count);
    if (rc != QBVH_OK) return rc;
    return finish_neighbors();
}

int qbvh_build_f64(const double *pos, const int32_t *type, int64_t N, const double *box) {
    if (!box) return QBVH_ERR_INVALID_ARG;
    float box32[6];
    for (int d = 0; d < 6; ++d) {
        if (!std::isfinite(box[d])) return QBVH_ERR_INVALID_ARG;
        box32[d] = (float)box[d];                     // the tree lives in fp32: Morton bins and frames from rounded values
    }
    return build_impl(pos, true, type, N, box32, box);
}

int qbvh_neighbors_f64(const double *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh) {
    int rc = neighbors_impl(r_list_ij, true, nlist, n_neigh, max_neigh);
    if (rc != QBVH_OK) return rc;
    return finish_neighbors();
}

int qbvh_count_overlaps(const float *r_list_ij, int32_t *n_overlap) {
    g.enqueued = false;
    if (!g.built) return QBVH_ERR_NOT_BUILT;
    if (!r_list_ij || (g.N > 0 && !n_overlap)) return QBVH_ERR_INVALID_ARG;
    TraverseParams P{};
    if (g.f64_built) return QBVH_ERR_INVALID_ARG;
    const int prc = make_params(r_list_ij, false, P);
    if (prc != QBVH_OK) return prc;
    P.max_neigh = 0;
    P.q_first = 0, P.q_count = -1;
    cudaError_t e = cudaMemsetAsync(&g.buf.meta->group_cursor, 0, 2 * sizeof(int32_t), g.stream);
    if (e != cudaSuccess) return cuda_fail(e, "memset max_count");
    g.counters_armed = false;
    e = launch_count_overlaps(P, g.buf, n_overlap, g.stream);
    if (e != cudaSuccess) return cuda_fail(e, "count launch");
    e = cudaMemcpyAsync(g.pinned, &g.buf.meta->max_count, 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, g.stream);
    if (e != cudaSuccess) return cuda_fail(e, "copy max_count");
    return finish_neighbors();
}

int64_t qbvh_staging_bytes(int64_t N, int32_t max_neigh) {
    if (N < 0 || max_neigh < 0) return QBVH_ERR_INVALID_ARG;
    const int64_t n1 = N > 0 ? N : 1;
    return align256(12 * n1) + align256(4 * n1) + align256(4 * n1 * (int64_t)(max_neigh > 0 ? max_neigh : 1)) + align256(4 * n1);
}

int qbvh_set_staging(void *dev_ptr, int64_t bytes) {
    if (dev_ptr && ((reinterpret_cast<uintptr_t>(dev_ptr) & 255) || bytes <= 0)) return QBVH_ERR_WORKSPACE;
    g.staging = dev_ptr;
    g.staging_bytes = dev_ptr ? bytes : 0;
    return QBVH_OK;
}

int qbvh_build_host(const float *pos, const int32_t *type, int64_t N, const float *box) {
    if (N < 0 || (N > 0 && !pos)) return QBVH_ERR_INVALID_ARG;
    const int64_t n1 = N > 0 ? N : 1;
    if (!g.staging || g.staging_bytes < align256(12 * n1) + align256(4 * n1)) return QBVH_ERR_WORKSPACE;
    char *s = static_cast<char *>(g.staging);
    float *dpos = reinterpret_cast<float *>(s);
    int32_t *dtype = reinterpret_cast<int32_t *>(s + align256(12 * n1));
    cudaError_t e;
    if (N > 0) {
        e = cudaMemcpyAsync(dpos, pos, 12 * N, cudaMemcpyHostToDevice, g.stream);
        if (e != cudaSuccess) return cuda_fail(e, "H2D pos");
        if (type) {
            e = cudaMemcpyAsync(dtype, type, 4 * N, cudaMemcpyHostToDevice, g.stream);
            if (e != cudaSuccess) return cuda_fail(e, "H2D type");
        }
    }
    return qbvh_build(dpos, type ? dtype : nullptr, N, box);
}

int qbvh_neighbors_host(const float *r_list_ij, int32_t *nlist, int32_t *n_neigh, int32_t max_neigh) {
    if (!g.built) return QBVH_ERR_NOT_BUILT;
    if (max_neigh < 0) return QBVH_ERR_INVALID_ARG;
    const int64_t N = g.N, n1 = N > 0 ? N : 1;
    if (!g.staging || g.staging_bytes < qbvh_staging_bytes(N, max_neigh)) return QBVH_ERR_WORKSPACE;
    char *s = static_cast<char *>(g.staging);
    int32_t *dlist = reinterpret_cast<int32_t *>(s + align256(12 * n1) + align256(4 * n1));
    int32_t *dcnt = reinterpret_cast<int32_t *>(s + align256(12 * n1) + align256(4 * n1) +
                                                align256(4 * n1 * (int64_t)(max_neigh > 0 ? max_neigh : 1)));
    if (N > 0 && (!n_neigh || (!nlist && max_neigh > 0))) return QBVH_ERR_INVALID_ARG;
    // Pinned (mapped) host rows are written by the SMs (rows_to_host_kernel): only the entries that exist, 128-byte
    // coalesced, rows in index order.  Anything else (pageable memory, odd capacities) goes through the copy engine
    // once the longest row is known.
    int32_t *hdev = nullptr;
    if (N > 0 && max_neigh > 0 && (max_neigh & 3) == 0 && (reinterpret_cast<uintptr_t>(nlist) & 15) == 0) {
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, nlist) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer)
            hdev = static_cast<int32_t *>(at.devicePointer);
        else
            (void)cudaGetLastError();
    }
    cudaError_t e = cudaSuccess;
    if (hdev) {
        e = cudaMemsetAsync(&g.buf.meta->d2h_bytes, 0, sizeof(unsigned long long), g.stream);
        if (e != cudaSuccess) return cuda_fail(e, "memset d2h_bytes");
    }
    int rc = neighbors_impl(r_list_ij, false, dlist, dcnt, max_neigh);
    if (rc != QBVH_OK) return rc;
    if (N > 0) {
        e = cudaMemcpyAsync(n_neigh, dcnt, 4 * N, cudaMemcpyDeviceToHost, g.stream);
        if (e != cudaSuccess) return cuda_fail(e, "D2H n_neigh");
    }
    if (hdev) {
        e = launch_rows_to_host(dlist, dcnt, hdev, N, max_neigh, g.buf.meta, g.stream);
        if (e != cudaSuccess) return cuda_fail(e, "rows_to_host launch");
        e = cudaMemcpyAsync(g.pinned + 2, &g.buf.meta->d2h_bytes, sizeof(unsigned long long), cudaMemcpyDeviceToHost, g.stream);
        if (e != cudaSuccess) return cuda_fail(e, "copy d2h_bytes");
    }
    const int M = finish_neighbors();          // synchronises: the longest row is known now
    if (M < 0) return M;
    g.last_d2h_bytes = 4 * N + 8;
    if (hdev) {
        unsigned long long b;
        std::memcpy(&b, g.pinned + 2, sizeof(b));
        g.last_d2h_bytes += (int64_t)b + 8;
    } else if (N > 0 && max_neigh > 0 && M > 0) {
        // only the columns that were produced: rows hold at most min(M, max_neigh) entries (the rest is unspecified)
        const int64_t cols = M < max_neigh ? M : max_neigh;
        e = cudaMemcpy2DAsync(nlist, (size_t)4 * max_neigh, dlist, (size_t)4 * max_neigh, (size_t)4 * cols, (size_t)N,
                              cudaMemcpyDeviceToHost, g.stream);
        if (e != cudaSuccess) return cuda_fail(e, "D2H nlist");
        e = cudaStreamSynchronize(g.stream);
        if (e != cudaSuccess) return cuda_fail(e, "stream synchronize");
        g.last_d2h_bytes += 4 * cols * N;
    }
    return M;
}

int64_t qbvh_last_d2h_bytes(void) { return g.last_d2h_bytes; }

float qbvh_padded_radius(float r, const float *box) {
    if (!box || !(r > 0.0f) || !std::isfinite(r)) return -1.0f;
    for (int d = 0; d < 3; ++d)
        if (!std::isfinite(box[d]) || !std::isfinite(box[3 + d]) || !(box[3 + d] > 0.0f)) return -1.0f;
    return padded_radius(r, box);
}

float qbvh_padded_radius_sq(float r, const float *box) {
    const float rp = qbvh_padded_radius(r, box);
    return rp < 0.0f ? -1.0f : mul_ru(rp, rp);        // exactly what make_params stores in TraverseParams::R2
}

int qbvh_get_stats(qbvh_stats *out) {
    if (!out) return QBVH_ERR_INVALID_ARG;
    *out = g.last_stats;
    return QBVH_OK;
}

int64_t qbvh_debug_export(int32_t what, void *dst, int64_t bytes) {
    if (!g.built) return QBVH_ERR_NOT_BUILT;
    if (bytes < 0 || (bytes > 0 && !dst)) return QBVH_ERR_INVALID_ARG;
    const int64_t N = g.N;
    const void *src = nullptr;
    int64_t avail = 0;
    int32_t segroots[10];
    switch (what) {
        case QBVH_EXPORT_KEYS_SORTED: src = g.buf.key_sorted; avail = 4 * N; break;
        case QBVH_EXPORT_PERM: src = g.buf.idx_sorted; avail = 4 * N; break;
        case QBVH_EXPORT_NODES: src = g.buf.nodes; avail = N > 0 ? 16 * (2 * N - 1) : 0; break;
        case QBVH_EXPORT_PARENT: src = g.buf.parent; avail = N > 0 ? 4 * (2 * N - 1) : 0; break;
        case QBVH_EXPORT_FRAMES: src = g.buf.meta->frames; avail = sizeof(float) * QBVH_TMAX * 12; break;
        case QBVH_EXPORT_SORTED_POS: src = g.buf.sorted_pos; avail = 16 * N; break;
        case QBVH_EXPORT_SEGMENTS: avail = sizeof(segroots); break;
        case QBVH_EXPORT_COUNTS: avail = 4 * sizeof(int32_t); break;
        default: return QBVH_ERR_INVALID_ARG;
    }
    cudaError_t e = cudaStreamSynchronize(g.stream);
    if (e != cudaSuccess) return cuda_fail(e, "export synchronize");
    const int64_t n = bytes < avail ? bytes : avail;
    if (what == QBVH_EXPORT_COUNTS) {
        int32_t c[4] = {0, 0, 0, g.lvl_built};
        e = cudaMemcpy(&c[0], &g.buf.meta->nodes_emitted, sizeof(int32_t), cudaMemcpyDeviceToHost);
        if (e == cudaSuccess) e = cudaMemcpy(&c[1], &g.buf.meta->group_count, sizeof(int32_t), cudaMemcpyDeviceToHost);
        if (e == cudaSuccess) e = cudaMemcpy(&c[2], &g.buf.meta->ncell, sizeof(int32_t), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return cuda_fail(e, "export copy");
        std::memcpy(dst, c, (size_t)n);
        return avail;
    }
    if (what == QBVH_EXPORT_SEGMENTS) {
        std::memset(segroots, 0, sizeof(segroots));
        e = cudaMemcpy(segroots, g.buf.meta->seg, sizeof(int32_t) * 5, cudaMemcpyDeviceToHost);
        if (e == cudaSuccess) e = cudaMemcpy(segroots + 5, g.buf.meta->roots, sizeof(int32_t) * 4, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return cuda_fail(e, "export copy");
        std::memcpy(dst, segroots, (size_t)n);
        return avail;
    }
    if (n > 0) {
        e = cudaMemcpy(dst, src, (size_t)n, cudaMemcpyDefault);     // dst: host or device (unified addressing)
        if (e != cudaSuccess) return cuda_fail(e, "export copy");
    }
    return avail;
}

const char *qbvh_error_string(int code) {
    switch (code) {
        case QBVH_OK: return "ok";
        case QBVH_ERR_INVALID_ARG: return "invalid argument";
        case QBVH_ERR_NOT_BUILT: return "no tree: call qbvh_build first";
        case QBVH_ERR_WORKSPACE: return "workspace/staging missing, misaligned or too small";
        case QBVH_ERR_CUTOFF_TOO_LARGE: return "padded cutoff is not below half the shortest box length";
        case QBVH_ERR_TYPE_RANGE: return "a particle type id is outside [0, T)";
        case QBVH_ERR_INTERNAL: return "internal bound violated (traversal work list); please report";
        case QBVH_ERR_NOALLOC_LIMIT: return "N exceeds QBVH_NOALLOC_MAX_N (4194304), the size of the built-in scratch of qbvh_morton_keys_noalloc";
        case QBVH_ERR_CUDA: return g.cuda_msg;
        default: return code > 0 ? "ok (positive return value)" : "unknown error code";
    }
}

}  // extern "C"

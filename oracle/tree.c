/* ORACLE — TEST INFRASTRUCTURE ONLY.
 *
 * CPU restatements of the BUILD steps and of Algorithm 1, written from the
 * paper's definitions, one step at a time, in the paper's order.  Used by the
 * tests to pin steps a1..a8 of the CUDA path bit-exactly and
 * to check the "never miss a pair" property.  Shares no
 * code with the CUDA path.  Readings R1..R15 are listed in DESIGN.md §4.
 *
 * Node numbering (both sides adopt it so arrays compare bit-for-bit):
 *   internal node covering sorted range [f,l] of a tree over segment [s,e]:
 *     root -> s ; left child [f,g] -> g ; right child [g+1,l] -> g+1   (Karras, ref [27] of the paper)
 *   leaf for sorted position k -> (N-1)+k.
 *   `left`  >= 0 : index of the left child;  < 0 : leaf, value = ~k
 *   `rope`  >= 0 : next node to test;        -1 : END ("past the last node")
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -frounding-math -shared -fPIC
 */
#include <fenv.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#pragma STDC FENV_ACCESS ON

#define NBINS 1023 /* 2^10 - 1 bins per axis, PAPER.md:61 (Morton) and :89 (quantizer) */

/* ---------------------------------------------------------------------------
 * a1. Morton keys (§2.1): the simulation box is divided into
 * 2^10-1 bins per axis, bin coordinate = 10-bit integer, 30-bit code by bitwise
 * interleave.  Reading R2/O5:  b_d = clamp(floor((p_d - lo_d) * s_d), 0, 1023),
 * s_d = 1023/L_d, all fp32 RN; x holds the most significant bit of each triple;
 * key = type << 30 | code.
 * ------------------------------------------------------------------------- */
static uint32_t interleave3(uint32_t bx, uint32_t by, uint32_t bz) {
    uint32_t code = 0;
    for (int bit = 9; bit >= 0; --bit) {
        code = (code << 1) | ((bx >> bit) & 1u);
        code = (code << 1) | ((by >> bit) & 1u);
        code = (code << 1) | ((bz >> bit) & 1u);
    }
    return code;
}

void oracle_morton_keys(const float *pos, const int32_t *type, int64_t N, const float *box, uint32_t *key) {
    float s[3];
    for (int d = 0; d < 3; ++d) s[d] = 1023.0f / box[3 + d];
    for (int64_t i = 0; i < N; ++i) {
        uint32_t b[3];
        for (int d = 0; d < 3; ++d) {
            volatile float u = pos[3 * i + d] - box[d];
            volatile float v = u * s[d];
            float fl = floorf(v);
            if (!(fl >= 0.0f)) fl = 0.0f;
            if (fl > 1023.0f) fl = 1023.0f;
            b[d] = (uint32_t)fl;
        }
        uint32_t t = type ? (uint32_t)type[i] : 0u;
        key[i] = (t << 30) | interleave3(b[0], b[1], b[2]);
    }
}

/* ---------------------------------------------------------------------------
 * a3 + a4. Binary radix tree over the sorted keys (construction
 * deferred by the paper to its ref [27]) built TOP-DOWN here: a range is split
 * at the highest bit in which its first and last augmented key (key, position)
 * differ (R8: ties between equal Morton codes are broken by sorted position).
 * Ropes by the textbook recursion rope(left) = right, rope(right) = rope(node),
 * rope(root) = END.  One tree per type segment (R14).
 * ------------------------------------------------------------------------- */
typedef struct {
    const uint32_t *key;
    int64_t N;
    int32_t *left, *right, *rope, *parent, *first, *last;
} tree_ctx;

static inline uint64_t aug(const tree_ctx *c, int64_t k) { return ((uint64_t)c->key[k] << 32) | (uint64_t)(uint32_t)k; }
static inline int32_t leaf_id(const tree_ctx *c, int64_t k) { return (int32_t)(c->N - 1 + k); }

static void build_rec(tree_ctx *c, int64_t f, int64_t l, int32_t self, int32_t parent, int32_t rope) {
    c->parent[self] = parent;
    c->rope[self] = rope;
    c->first[self] = (int32_t)f;
    c->last[self] = (int32_t)l;
    if (f == l) {
        c->left[self] = ~(int32_t)f;
        c->right[self] = ~(int32_t)f;
        return;
    }
    uint64_t x = aug(c, f) ^ aug(c, l);
    int bit = 63 - __builtin_clzll(x);
    int64_t g = f; /* last position whose augmented key has a 0 in `bit` */
    while (g + 1 <= l && !((aug(c, g + 1) >> bit) & 1ull)) ++g;
    int32_t lc = (g == f) ? leaf_id(c, f) : (int32_t)g;
    int32_t rc = (g + 1 == l) ? leaf_id(c, l) : (int32_t)(g + 1);
    c->left[self] = lc;
    c->right[self] = rc;
    build_rec(c, f, g, lc, self, rc);
    build_rec(c, g + 1, l, rc, self, rope);
}

/* arrays have 2N-1 entries; seg has T+1 entries (type t owns sorted positions [seg[t], seg[t+1]));
 * roots[t] = root node of tree t or -1 for an empty type.  Unused internal slots ("holes", one per
 * type boundary) get left = 0, right = 0, rope = -1, parent = -1, first = last = -1. */
void oracle_build_tree(const uint32_t *key_sorted, int64_t N, const int64_t *seg, int32_t T, int32_t *left,
                       int32_t *right, int32_t *rope, int32_t *parent, int32_t *first, int32_t *last,
                       int32_t *roots) {
    tree_ctx c = {key_sorted, N, left, right, rope, parent, first, last};
    for (int64_t n = 0; n < 2 * N - 1; ++n) {
        left[n] = 0;
        right[n] = 0;
        rope[n] = -1;
        parent[n] = -1;
        first[n] = -1;
        last[n] = -1;
    }
    for (int t = 0; t < T; ++t) {
        int64_t s = seg[t], e = seg[t + 1] - 1;
        if (e < s) {
            roots[t] = -1;
            continue;
        }
        int32_t root = (s == e) ? leaf_id(&c, s) : (int32_t)s;
        roots[t] = root;
        build_rec(&c, s, e, root, -1, -1);
    }
}

/* ---------------------------------------------------------------------------
 * a6. Quantizer, defined through its decompressor (R9):
 *   frame of a tree: lo_d, hi_d = fp32 min/max of its particles (R15: the
 *   root-node AABB);  Delta_d = div_ru(sub_ru(hi_d, lo_d), 1023)
 *   D_lo(q) = fma_rd(q, Delta_d, lo_d)     D_hi(q) = fma_ru(q, Delta_d, lo_d)
 *   q_lo(a) = max{ q in [0,1023] : D_lo(q) <= a }   (lower bounds round DOWN)
 *   q_hi(b) = min{ q in [0,1023] : D_hi(q) >= b }   (upper bounds round UP)
 * "IEEE 754-2008 round-down and round-up modes".
 * ------------------------------------------------------------------------- */
static float sub_ru(float a, float b) {
    fesetround(FE_UPWARD);
    volatile float r = a - b;
    fesetround(FE_TONEAREST);
    return r;
}
static float div_ru(float a, float b) {
    fesetround(FE_UPWARD);
    volatile float r = a / b;
    fesetround(FE_TONEAREST);
    return r;
}

/* tables D_lo[q], D_hi[q], q = 0..1023 for one axis of one frame */
void oracle_decompress_tables(float lo, float delta, float *Dlo, float *Dhi) {
    fesetround(FE_DOWNWARD);
    for (int q = 0; q < 1024; ++q) {
        volatile float r = fmaf((float)q, delta, lo);
        Dlo[q] = r;
    }
    fesetround(FE_UPWARD);
    for (int q = 0; q < 1024; ++q) {
        volatile float r = fmaf((float)q, delta, lo);
        Dhi[q] = r;
    }
    fesetround(FE_TONEAREST);
}

float oracle_frame_delta(float lo, float hi) { return div_ru(sub_ru(hi, lo), (float)NBINS); }

/* the definition, by exhaustive scan over all 1024 codes */
int oracle_qlo_scan(const float *Dlo, float a) {
    int best = 0;
    for (int q = 0; q < 1024; ++q)
        if (Dlo[q] <= a) best = q;
    return best;
}
int oracle_qhi_scan(const float *Dhi, float b) {
    for (int q = 0; q < 1024; ++q)
        if (Dhi[q] >= b) return q;
    return 1023;
}
/* same values by bisection (D_lo, D_hi are non-decreasing in q); used in bulk, pinned to the scans in tests */
static int qlo_bisect(const float *Dlo, float a) {
    int q = 0;
    for (int bit = 512; bit; bit >>= 1)
        if (Dlo[q | bit] <= a) q |= bit;
    return q;
}
static int qhi_bisect(const float *Dhi, float b) {
    int q = 0;
    for (int bit = 512; bit; bit >>= 1)
        if (Dhi[(q + bit) - 1] < b) q += bit;
    return q;
}

typedef struct {
    int64_t N;
    const float *pos; /* sorted, N x 3 */
    const int32_t *left, *right;
    const float *Dlo, *Dhi; /* current tree: [3][1024] */
    float *blo, *bhi;       /* fp32 boxes per node, (2N-1) x 3 */
    uint32_t *wlo, *whi;    /* packed words per node */
    int scan;
} fit_ctx;

/* a5: "bounding volumes are fit for each node by walking up the tree from the leaf nodes":
 * leaf box = the particle's point, internal box = union of the children's boxes (exact in fp32). */
static void fit_rec(fit_ctx *c, int32_t n) {
    float *lo = c->blo + 3 * (int64_t)n, *hi = c->bhi + 3 * (int64_t)n;
    if (c->left[n] < 0) {
        int64_t k = ~c->left[n];
        for (int d = 0; d < 3; ++d) lo[d] = hi[d] = c->pos[3 * k + d];
    } else {
        int32_t a = c->left[n], b = c->right[n];
        fit_rec(c, a);
        fit_rec(c, b);
        for (int d = 0; d < 3; ++d) {
            lo[d] = fminf(c->blo[3 * (int64_t)a + d], c->blo[3 * (int64_t)b + d]);
            hi[d] = fmaxf(c->bhi[3 * (int64_t)a + d], c->bhi[3 * (int64_t)b + d]);
        }
    }
    uint32_t wl = 0, wh = 0;
    for (int d = 0; d < 3; ++d) { /* R7: x bits 0-9, y 10-19, z 20-29, bits 30-31 zero */
        int ql = c->scan ? oracle_qlo_scan(c->Dlo + 1024 * d, lo[d]) : qlo_bisect(c->Dlo + 1024 * d, lo[d]);
        int qh = c->scan ? oracle_qhi_scan(c->Dhi + 1024 * d, hi[d]) : qhi_bisect(c->Dhi + 1024 * d, hi[d]);
        wl |= (uint32_t)ql << (10 * d);
        wh |= (uint32_t)qh << (10 * d);
    }
    c->wlo[n] = wl;
    c->whi[n] = wh;
}

/* frames: T x 9 floats {lo_xyz, hi_xyz, delta_xyz}; tables (out, optional): T x 2 x 3 x 1024 floats */
void oracle_fit_quantize(const float *pos_sorted, int64_t N, const int64_t *seg, int32_t T, const int32_t *left,
                         const int32_t *right, const int32_t *roots, float *frames, float *blo, float *bhi,
                         uint32_t *wlo, uint32_t *whi, float *tables, int use_scan) {
    float *Dlo = (float *)malloc(sizeof(float) * 3 * 1024), *Dhi = (float *)malloc(sizeof(float) * 3 * 1024);
    for (int64_t n = 0; n < 2 * N - 1; ++n) {
        wlo[n] = whi[n] = 0;
        for (int d = 0; d < 3; ++d) blo[3 * n + d] = bhi[3 * n + d] = 0.0f;
    }
    for (int t = 0; t < T; ++t) {
        float *fr = frames + 9 * t;
        for (int d = 0; d < 9; ++d) fr[d] = 0.0f;
        if (roots[t] < 0) continue;
        for (int d = 0; d < 3; ++d) {
            float lo = INFINITY, hi = -INFINITY;
            for (int64_t k = seg[t]; k < seg[t + 1]; ++k) {
                lo = fminf(lo, pos_sorted[3 * k + d]);
                hi = fmaxf(hi, pos_sorted[3 * k + d]);
            }
            fr[d] = lo;
            fr[3 + d] = hi;
            fr[6 + d] = oracle_frame_delta(lo, hi);
            oracle_decompress_tables(lo, fr[6 + d], Dlo + 1024 * d, Dhi + 1024 * d);
        }
        if (tables) {
            memcpy(tables + (size_t)t * 6144, Dlo, sizeof(float) * 3072);
            memcpy(tables + (size_t)t * 6144 + 3072, Dhi, sizeof(float) * 3072);
        }
        fit_ctx c = {N, pos_sorted, left, right, Dlo, Dhi, blo, bhi, wlo, whi, use_scan};
        fit_rec(&c, roots[t]);
    }
    free(Dlo);
    free(Dhi);
}

/* ---------------------------------------------------------------------------
 * Padded search radius (R11) — used only for pruning, never in O1:
 *   r_pad = add_ru( mul_ru(r, 1 + 2^-20), 8 * ulp32(M) ),  M = max_d(|lo_d| + 2 L_d)
 *   R2    = mul_ru(r_pad, r_pad)
 * ------------------------------------------------------------------------- */
float oracle_pad_abs(const float *box) {
    double M = 0.0;
    for (int d = 0; d < 3; ++d) {
        double m = fabs((double)box[d]) + 2.0 * (double)box[3 + d];
        if (m > M) M = m;
    }
    int e;
    frexp(M, &e); /* M = f * 2^e, f in [0.5,1)  ->  floor(log2 M) = e-1 */
    return (float)ldexp(8.0, (e - 1) - 23);
}
float oracle_r_pad(float r, float pad_abs) {
    fesetround(FE_UPWARD);
    volatile float a = r * (1.0f + 0x1p-20f);
    volatile float b = a + pad_abs;
    fesetround(FE_TONEAREST);
    return b;
}
static float mul_ru(float a, float b) {
    fesetround(FE_UPWARD);
    volatile float r = a * b;
    fesetround(FE_TONEAREST);
    return r;
}

/* Squared padded pruning radius, rounded UP (reading R11; "the sphere radius is padded"):
 * the right-hand side of every sphere/box test below.  Exported so that a test can pin it against exact rationals. */
float oracle_R2(float r, float pad_abs) {
    float rp = oracle_r_pad(r, pad_abs);
    return mul_ru(rp, rp);
}

/* ---------------------------------------------------------------------------
 * a7 + a8. Algorithm 1 (reconstructed per R1), one particle at
 * a time, in the paper's "accept the leaf on box overlap" mode (line 14).
 * Sphere-AABB test = eq. 2 on the DEcompressed box (line 11,
 * PAPER.md:140), fp32:
 *     x' = x_i + v_j (RN);  a = D_lo(q_lo), b = D_hi(q_hi);  y = min(max(x',a),b)
 *     t = y - x' (RN);  d2 = fma(t_z,t_z, fma(t_y,t_y, t_x*t_x));  overlap <=> d2 <= R2
 * Image j = (i+1) + 3(j+1) + 9(k+1) for v = (i Lx, j Ly, k Lz), i,j,k in {-1,0,1} (R12).
 *
 * For query particle at sorted position k (type a) every tree b with r_ab > 0 is walked.
 * Outputs (count pass: row_ptr == NULL):
 *   n_overlap[k]  number of leaf-box overlaps (the paper's "neighbors", self included when b == a)
 *   n_tests[k]    number of node tests (root tests of line 4 not counted)
 *   n_images[k]   number of set bits of b summed over trees
 * fill pass (row_ptr != NULL): cand[row_ptr[k] ...] = sorted positions of the overlapped leaves, in visit order.
 * ------------------------------------------------------------------------- */
static inline int sphere_box(const float *x, const float *a, const float *b, float R2) {
    float t[3];
    for (int d = 0; d < 3; ++d) {
        float y = fminf(fmaxf(x[d], a[d]), b[d]);
        t[d] = y - x[d];
    }
    float d2 = fmaf(t[2], t[2], fmaf(t[1], t[1], t[0] * t[0]));
    return d2 <= R2;
}

int64_t oracle_traverse(const float *pos_sorted, int64_t N, const int64_t *seg, int32_t T, const float *box,
                        const float *r_list, const uint32_t *wlo, const uint32_t *whi, const int32_t *left,
                        const int32_t *rope, const int32_t *roots, const float *tables, int32_t *n_overlap,
                        int64_t *n_tests, int32_t *n_images, const int64_t *row_ptr, int32_t *cand) {
    float pad_abs = oracle_pad_abs(box);
    int64_t total = 0;
    float *R2 = (float *)malloc(sizeof(float) * (size_t)(T * T));
    for (int k = 0; k < T * T; ++k) R2[k] = r_list[k] > 0.0f ? oracle_R2(r_list[k], pad_abs) : -1.0f;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : total)
    for (int64_t k = 0; k < N; ++k) {
        int ta = 0;
        while (k >= seg[ta + 1]) ++ta;
        const float *xi = pos_sorted + 3 * k;
        int32_t cnt = 0, nimg = 0;
        int64_t tests = 0;
        for (int tb = 0; tb < T; ++tb) {
            float r2 = R2[ta * T + tb];
            if (r2 < 0.0f || roots[tb] < 0) continue;
            const float *Dlo = tables + (size_t)tb * 6144, *Dhi = Dlo + 3072;
            int32_t root = roots[tb];
            /* line 4: bitset of images whose sphere overlaps the root node */
            uint32_t bset = 0;
            float a[3], b[3], x[3];
            for (int d = 0; d < 3; ++d) {
                a[d] = Dlo[1024 * d + ((wlo[root] >> (10 * d)) & 1023u)];
                b[d] = Dhi[1024 * d + ((whi[root] >> (10 * d)) & 1023u)];
            }
            for (int img = 0; img < 27; ++img) {
                int s[3] = {img % 3 - 1, (img / 3) % 3 - 1, img / 9 - 1};
                for (int d = 0; d < 3; ++d) x[d] = xi[d] + (float)s[d] * box[3 + d];
                if (sphere_box(x, a, b, r2)) bset |= 1u << img;
            }
            while (bset) {                          /* line 5 */
                int img = __builtin_ctz(bset);      /* line 6 */
                bset &= bset - 1;                   /* line 7 */
                ++nimg;
                int s[3] = {img % 3 - 1, (img / 3) % 3 - 1, img / 9 - 1};
                for (int d = 0; d < 3; ++d) x[d] = xi[d] + (float)s[d] * box[3 + d]; /* line 8 */
                int32_t n = root;                   /* line 9 */
                while (n >= 0) {                    /* line 10 */
                    for (int d = 0; d < 3; ++d) {   /* line 11 */
                        a[d] = Dlo[1024 * d + ((wlo[n] >> (10 * d)) & 1023u)];
                        b[d] = Dhi[1024 * d + ((whi[n] >> (10 * d)) & 1023u)];
                    }
                    ++tests;
                    if (sphere_box(x, a, b, r2)) {  /* line 12 */
                        if (left[n] < 0) {          /* line 13 */
                            if (row_ptr) cand[row_ptr[k] + cnt] = ~left[n]; /* line 14 */
                            ++cnt;
                            n = rope[n];            /* line 15 */
                        } else {
                            n = left[n];            /* line 17 */
                        }
                    } else {
                        n = rope[n];                /* line 19 */
                    }
                }
            }
        }
        if (!row_ptr) {
            n_overlap[k] = cnt;
            n_tests[k] = tests;
            n_images[k] = nimg;
        }
        total += cnt;
    }
    free(R2);
    return total;
}


/* ---------------------------------------------------------------------------
 * The same walk on the UNquantized fp32 boxes blo/bhi of oracle_fit_quantize (what the tree was before step a6):
 * the census against which "extra false-positive AABB tests caused by quantization" are counted (PAPER.md:85, 89,
 * 196-198).  Count pass only.  Everything but the source of a and b is oracle_traverse's.
 * ------------------------------------------------------------------------- */
int64_t oracle_traverse_fp32_boxes(const float *pos_sorted, int64_t N, const int64_t *seg, int32_t T, const float *box,
                                   const float *r_list, const float *blo, const float *bhi, const int32_t *left,
                                   const int32_t *rope, const int32_t *roots, int32_t *n_overlap, int64_t *n_tests,
                                   int32_t *n_images) {
    float pad_abs = oracle_pad_abs(box);
    int64_t total = 0;
    float *R2 = (float *)malloc(sizeof(float) * (size_t)(T * T));
    for (int k = 0; k < T * T; ++k) R2[k] = r_list[k] > 0.0f ? oracle_R2(r_list[k], pad_abs) : -1.0f;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : total)
    for (int64_t k = 0; k < N; ++k) {
        int ta = 0;
        while (k >= seg[ta + 1]) ++ta;
        const float *xi = pos_sorted + 3 * k;
        int32_t cnt = 0, nimg = 0;
        int64_t tests = 0;
        for (int tb = 0; tb < T; ++tb) {
            float r2 = R2[ta * T + tb];
            if (r2 < 0.0f || roots[tb] < 0) continue;
            int32_t root = roots[tb];
            uint32_t bset = 0;
            float x[3];
            for (int img = 0; img < 27; ++img) {                                     /* line 4 */
                int s[3] = {img % 3 - 1, (img / 3) % 3 - 1, img / 9 - 1};
                for (int d = 0; d < 3; ++d) x[d] = xi[d] + (float)s[d] * box[3 + d];
                if (sphere_box(x, blo + 3 * (size_t)root, bhi + 3 * (size_t)root, r2)) bset |= 1u << img;
            }
            while (bset) {
                int img = __builtin_ctz(bset);
                bset &= bset - 1;
                ++nimg;
                int s[3] = {img % 3 - 1, (img / 3) % 3 - 1, img / 9 - 1};
                for (int d = 0; d < 3; ++d) x[d] = xi[d] + (float)s[d] * box[3 + d];
                int32_t n = root;
                while (n >= 0) {
                    ++tests;
                    if (sphere_box(x, blo + 3 * (size_t)n, bhi + 3 * (size_t)n, r2)) {
                        if (left[n] < 0) {
                            ++cnt;
                            n = rope[n];
                        } else {
                            n = left[n];
                        }
                    } else {
                        n = rope[n];
                    }
                }
            }
        }
        n_overlap[k] = cnt;
        n_tests[k] = tests;
        n_images[k] = nimg;
        total += cnt;
    }
    free(R2);
    return total;
}

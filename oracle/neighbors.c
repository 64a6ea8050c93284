/* ORACLE — TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct CPU statement of what the hot path computes:
 * "the subset of particles within a distance r_c of a given particle ... saved
 * to construct a Verlet (neighbor) list" (§1), "subject to the
 * periodic boundary conditions" (§4).  The quantized BVH only
 * prunes (no false negatives), so with the leaf filter the
 * method reaches exactly this definition; the oracle is the definition.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call this.  It shares no code with the CUDA path.
 *
 * Canonical pair predicate O1.  All fp32,
 * round-to-nearest, in this exact order ("the kernel's precision": the paper
 * fixes fp32 particle data, but not the rounding order):
 *     D_d = p_j[d] - p_i[d]
 *     if      D_d >  h_d : D_d = D_d - L_d        (h_d = 0.5f*L_d, exact)
 *     else if D_d < -h_d : D_d = D_d + L_d
 *     d2 = fmaf(D_z, D_z, fmaf(D_y, D_y, D_x*D_x))
 *     r  = r_list[t_i][t_j];  r2 = r*r
 *     neighbor(i,j)  <=>  i != j  and  r > 0  and  d2 <= r2      (inclusive)
 * A particle is not its own neighbor (Fig. 2 caption): excluded by index.
 *
 * The fp64 "band" classifier tags pairs whose exact minimum-image distance lies
 * within 1e-5 sigma of r (BASELINE.json north_star tolerance rule).
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC  (see oracle/build.py)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define BAND_WIDTH 1e-5

typedef struct {
    float lo[3], L[3], h[3];
} box_t;

static box_t make_box(const float *box) {
    box_t b;
    for (int d = 0; d < 3; ++d) {
        b.lo[d] = box[d];
        b.L[d] = box[3 + d];
        b.h[d] = 0.5f * box[3 + d];
    }
    return b;
}

/* O1: squared minimum-image distance in fp32, canonical order. */
static inline float pair_d2(const float *pi, const float *pj, const box_t *b) {
    float D[3];
    for (int d = 0; d < 3; ++d) {
        float x = pj[d] - pi[d];
        if (x > b->h[d])
            x = x - b->L[d];
        else if (x < -b->h[d])
            x = x + b->L[d];
        D[d] = x;
    }
    return fmaf(D[2], D[2], fmaf(D[1], D[1], D[0] * D[0]));
}

/* fp64 minimum-image distance from the same fp32 inputs (conversions are exact). */
static inline double pair_dist64(const float *pi, const float *pj, const box_t *b) {
    double s = 0.0;
    for (int d = 0; d < 3; ++d) {
        double L = (double)b->L[d];
        double x = (double)pj[d] - (double)pi[d];
        if (x > 0.5 * L)
            x -= L;
        else if (x < -0.5 * L)
            x += L;
        s += x * x;
    }
    return sqrt(s);
}

/* exported so tests can probe single pairs */
int oracle_pair(const float *pi, const float *pj, const float *box, float r, float *d2_out, double *d64_out) {
    box_t b = make_box(box);
    float d2 = pair_d2(pi, pj, &b);
    float r2 = r * r;
    if (d2_out) *d2_out = d2;
    if (d64_out) *d64_out = pair_dist64(pi, pj, &b);
    return (r > 0.0f) && (d2 <= r2);
}

static int cmp_i32(const void *a, const void *b) {
    int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}

static inline int type_of(const int32_t *type, int64_t i) { return type ? type[i] : 0; }

/* ---------------------------------------------------------------------------
 * Brute force: all N(N-1) ordered pairs through O1.  This IS the definition.
 *   row_ptr == NULL : count pass, fills n_neigh[N].
 *   row_ptr != NULL : fill pass, writes ascending neighbor indices of i at
 *                     nbr[row_ptr[i] ...], and band[...] (if not NULL) = 1 for
 *                     pairs with |d64 - r| < 1e-5.
 * returns the total number of ordered pairs, or -1 on bad arguments.
 * ------------------------------------------------------------------------- */
int64_t oracle_brute_force(const float *pos, const int32_t *type, int64_t N, const float *box,
                           const float *r_list, int32_t T, int32_t *n_neigh, const int64_t *row_ptr,
                           int32_t *nbr, uint8_t *band) {
    if (N < 0 || T < 1 || !box || !r_list || !n_neigh) return -1;
    box_t b = make_box(box);
    int64_t total = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : total)
    for (int64_t i = 0; i < N; ++i) {
        const float *pi = pos + 3 * i;
        int ti = type_of(type, i);
        int32_t c = 0;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            float r = r_list[ti * T + type_of(type, j)];
            if (!(r > 0.0f)) continue;
            float r2 = r * r;
            if (pair_d2(pi, pos + 3 * j, &b) <= r2) {
                if (row_ptr) {
                    nbr[row_ptr[i] + c] = (int32_t)j; /* j ascends: row is sorted */
                    if (band) band[row_ptr[i] + c] = fabs(pair_dist64(pi, pos + 3 * j, &b) - (double)r) < BAND_WIDTH;
                }
                ++c;
            }
        }
        if (!row_ptr) n_neigh[i] = c;
        total += c;
    }
    return total;
}

/* ---------------------------------------------------------------------------
 * Cell list: cells per axis n_d = max(1, floor(L_d / (1.001 r_max)))
 * (cell width >= r_max with a 0.1 % margin that dwarfs fp32 rounding in O1),
 * binning in fp64, 27-cell stencil with periodic wrap, stencil cells
 * de-duplicated when n_d < 3; every candidate pair goes through O1.
 * Same two-pass protocol and outputs as oracle_brute_force.
 * ------------------------------------------------------------------------- */
int64_t oracle_cell_list(const float *pos, const int32_t *type, int64_t N, const float *box,
                         const float *r_list, int32_t T, int32_t *n_neigh, const int64_t *row_ptr,
                         int32_t *nbr, uint8_t *band) {
    if (N < 0 || T < 1 || !box || !r_list || !n_neigh) return -1;
    box_t b = make_box(box);
    float r_max = 0.0f;
    for (int k = 0; k < T * T; ++k)
        if (r_list[k] > r_max) r_max = r_list[k];
    int64_t nc[3];
    for (int d = 0; d < 3; ++d) {
        double n = (r_max > 0.0f) ? floor((double)b.L[d] / (1.001 * (double)r_max)) : 1.0;
        if (n < 1.0) n = 1.0;
        if (n > 1024.0) n = 1024.0;
        nc[d] = (int64_t)n;
    }
    int64_t ncell = nc[0] * nc[1] * nc[2];
    int64_t *cell_start = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
    int64_t *cell_of = (int64_t *)malloc(sizeof(int64_t) * (size_t)(N > 0 ? N : 1));
    int32_t *members = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
    if (!cell_start || !cell_of || !members) return -1;
    for (int64_t i = 0; i < N; ++i) {
        int64_t c[3];
        for (int d = 0; d < 3; ++d) {
            double f = ((double)pos[3 * i + d] - (double)b.lo[d]) / (double)b.L[d];
            int64_t k = (int64_t)floor(f * (double)nc[d]);
            if (k < 0) k = 0;
            if (k >= nc[d]) k = nc[d] - 1;
            c[d] = k;
        }
        cell_of[i] = (c[0] * nc[1] + c[1]) * nc[2] + c[2];
        cell_start[cell_of[i] + 1]++;
    }
    for (int64_t c = 0; c < ncell; ++c) cell_start[c + 1] += cell_start[c];
    {
        int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * (size_t)ncell);
        memcpy(fill, cell_start, sizeof(int64_t) * (size_t)ncell);
        for (int64_t i = 0; i < N; ++i) members[fill[cell_of[i]]++] = (int32_t)i; /* ascending inside a cell */
        free(fill);
    }
    int64_t total = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : total)
    for (int64_t i = 0; i < N; ++i) {
        const float *pi = pos + 3 * i;
        int ti = type_of(type, i);
        int64_t ci = cell_of[i];
        int64_t c[3] = {ci / (nc[1] * nc[2]), (ci / nc[2]) % nc[1], ci % nc[2]};
        int64_t cells[27];
        int ncells = 0;
        for (int dx = -1; dx <= 1; ++dx)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dz = -1; dz <= 1; ++dz) {
                    int64_t x = (c[0] + dx + nc[0]) % nc[0];
                    int64_t y = (c[1] + dy + nc[1]) % nc[1];
                    int64_t z = (c[2] + dz + nc[2]) % nc[2];
                    int64_t id = (x * nc[1] + y) * nc[2] + z;
                    int seen = 0;
                    for (int k = 0; k < ncells; ++k) seen |= (cells[k] == id);
                    if (!seen) cells[ncells++] = id;
                }
        int32_t cnt = 0;
        int32_t *row = row_ptr ? nbr + row_ptr[i] : NULL;
        for (int k = 0; k < ncells; ++k) {
            for (int64_t m = cell_start[cells[k]]; m < cell_start[cells[k] + 1]; ++m) {
                int32_t j = members[m];
                if (j == i) continue;
                float r = r_list[ti * T + type_of(type, j)];
                if (!(r > 0.0f)) continue;
                float r2 = r * r;
                if (pair_d2(pi, pos + 3 * (int64_t)j, &b) <= r2) {
                    if (row) row[cnt] = j;
                    ++cnt;
                }
            }
        }
        if (row) {
            qsort(row, (size_t)cnt, sizeof(int32_t), cmp_i32);
            if (band)
                for (int32_t k = 0; k < cnt; ++k) {
                    int32_t j = row[k];
                    float r = r_list[ti * T + type_of(type, j)];
                    band[row_ptr[i] + k] = fabs(pair_dist64(pi, pos + 3 * (int64_t)j, &b) - (double)r) < BAND_WIDTH;
                }
        } else {
            n_neigh[i] = cnt;
        }
        total += cnt;
    }
    free(cell_start);
    free(cell_of);
    free(members);
    return total;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ORACLE — TEST INFRASTRUCTURE ONLY.
 *
 * Double-precision particle data.  The paper supports both precisions and
 * reports its largest gains with double-precision particles; the tree stays single precision and
 * "the sphere radius is padded to account for uncertainty from loss of precision when the particle data is double
 * precision".  What the method then computes is still the plain definition — the particles within
 * r_c of each particle under periodic boundaries — now evaluated in fp64, so the oracle is that
 * definition written out in fp64.
 *
 * Canonical pair predicate O1-64, all IEEE binary64, round to nearest, in this order:
 *     D_d = p_j[d] - p_i[d]
 *     if      D_d >  h_d : D_d = D_d - L_d        (h_d = 0.5*L_d, exact)
 *     else if D_d < -h_d : D_d = D_d + L_d
 *     d2 = fma(D_z, D_z, fma(D_y, D_y, D_x*D_x));   r2 = r*r
 *     neighbor(i,j)  <=>  i != j  and  r > 0  and  d2 <= r2          (inclusive)
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call this.  It shares
 * no code with the CUDA path and none with oracle/neighbors.c (same structure, typed again for double).
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC  (see oracle/build.py)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

static inline double pair_d2_f64(const double *pi, const double *pj, const double *L) {
    double D[3];
    for (int d = 0; d < 3; ++d) {
        double h = 0.5 * L[d];
        double x = pj[d] - pi[d];
        if (x > h)
            x = x - L[d];
        else if (x < -h)
            x = x + L[d];
        D[d] = x;
    }
    return fma(D[2], D[2], fma(D[1], D[1], D[0] * D[0]));
}

/* one pair, for the pins */
int oracle_pair_f64(const double *pi, const double *pj, const double *box, double r, double *d2_out) {
    double d2 = pair_d2_f64(pi, pj, box + 3);
    if (d2_out) *d2_out = d2;
    return (r > 0.0) && (d2 <= r * r);
}

static inline int type_of64(const int32_t *type, int64_t i) { return type ? type[i] : 0; }

static int cmp_i32_64(const void *a, const void *b) {
    int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}

/* Brute force: all N(N-1) ordered pairs through O1-64.  Two-pass protocol of oracle_brute_force:
 * row_ptr == NULL counts into n_neigh; otherwise ascending neighbor indices go to nbr[row_ptr[i] ...]. */
int64_t oracle_brute_force_f64(const double *pos, const int32_t *type, int64_t N, const double *box,
                               const double *r_list, int32_t T, int32_t *n_neigh, const int64_t *row_ptr, int32_t *nbr) {
    if (N < 0 || T < 1 || !box || !r_list || !n_neigh) return -1;
    int64_t total = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : total)
    for (int64_t i = 0; i < N; ++i) {
        int ti = type_of64(type, i);
        int32_t c = 0;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            double r = r_list[ti * T + type_of64(type, j)];
            if (!(r > 0.0)) continue;
            if (pair_d2_f64(pos + 3 * i, pos + 3 * j, box + 3) <= r * r) {
                if (row_ptr) nbr[row_ptr[i] + c] = (int32_t)j;
                ++c;
            }
        }
        if (!row_ptr) n_neigh[i] = c;
        total += c;
    }
    return total;
}

/* Cell list: cells per axis n_d = max(1, floor(L_d / (1.001 r_max))), 27-cell stencil with periodic wrap,
 * de-duplicated when n_d < 3; every candidate pair goes through O1-64. */
int64_t oracle_cell_list_f64(const double *pos, const int32_t *type, int64_t N, const double *box,
                             const double *r_list, int32_t T, int32_t *n_neigh, const int64_t *row_ptr, int32_t *nbr) {
    if (N < 0 || T < 1 || !box || !r_list || !n_neigh) return -1;
    double r_max = 0.0;
    for (int k = 0; k < T * T; ++k)
        if (r_list[k] > r_max) r_max = r_list[k];
    int64_t nc[3];
    for (int d = 0; d < 3; ++d) {
        double n = (r_max > 0.0) ? floor(box[3 + d] / (1.001 * r_max)) : 1.0;
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
            int64_t k = (int64_t)floor((pos[3 * i + d] - box[d]) / box[3 + d] * (double)nc[d]);
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
        for (int64_t i = 0; i < N; ++i) members[fill[cell_of[i]]++] = (int32_t)i;
        free(fill);
    }
    int64_t total = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : total)
    for (int64_t i = 0; i < N; ++i) {
        int ti = type_of64(type, i);
        int64_t ci = cell_of[i];
        int64_t c[3] = {ci / (nc[1] * nc[2]), (ci / nc[2]) % nc[1], ci % nc[2]};
        int64_t cells[27];
        int ncells = 0;
        for (int dx = -1; dx <= 1; ++dx)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dz = -1; dz <= 1; ++dz) {
                    int64_t id = (((c[0] + dx + nc[0]) % nc[0]) * nc[1] + (c[1] + dy + nc[1]) % nc[1]) * nc[2] + (c[2] + dz + nc[2]) % nc[2];
                    int seen = 0;
                    for (int k = 0; k < ncells; ++k) seen |= (cells[k] == id);
                    if (!seen) cells[ncells++] = id;
                }
        int32_t cnt = 0;
        int32_t *row = row_ptr ? nbr + row_ptr[i] : NULL;
        for (int k = 0; k < ncells; ++k)
            for (int64_t m = cell_start[cells[k]]; m < cell_start[cells[k] + 1]; ++m) {
                int32_t j = members[m];
                if (j == i) continue;
                double r = r_list[ti * T + type_of64(type, j)];
                if (!(r > 0.0)) continue;
                if (pair_d2_f64(pos + 3 * i, pos + 3 * (int64_t)j, box + 3) <= r * r) {
                    if (row) row[cnt] = j;
                    ++cnt;
                }
            }
        if (row)
            qsort(row, (size_t)cnt, sizeof(int32_t), cmp_i32_64);
        else
            n_neigh[i] = cnt;
        total += cnt;
    }
    free(cell_start);
    free(cell_of);
    free(members);
    return total;
}

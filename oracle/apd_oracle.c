/*
 * oracle/apd_oracle.c -- TEST INFRASTRUCTURE, not the product.
 *
 * Plain, slow, fp64 CPU statement of what the hot path computes, written from the paper
 * (arxiv 2403.03571, /root/reference/PAPER.md).  It shares no code with the CUDA path
 * (paper_2403_03571_b200/csrc) and is only ever called from tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs.
 *
 * What it is: the DEFINITION written out.
 *   - voxel centre  y = lo + (i + 1/2) s,  s_k = (hi_k - lo_k)/n_k      PAPER.md:106-119 (P(y,s), eq. 2.6)
 *   - cost          C_ij = |y_j - x_i|^2_{A_i} - w_i                     PAPER.md:131 (Alg. 1 step 1; the
 *                   minus signs dropped by the text extraction are restored from eq. (2.1))
 *   - label         H_j in argmin_i C_ij                                 PAPER.md:132 (Alg. 1 step 2);
 *                   on exact ties the lowest index (reading S1): strict '<', ascending i.
 * The quadratic form sums all d*d entries of A_i as given (no symmetry assumed, reading S13).
 * No blocking, no reordering, no early exit: two nested loops.  OpenMP only splits the
 * OUTER (voxel) loop; every voxel's result is independent of the thread count.
 *
 * The reductions of eq. (2.7)-(2.8) (volumes, dual, centroids) are done by oracle/apd_oracle.py
 * from the per-voxel arrays this file returns.
 *
 * Parity pins: tests/test_oracle_pins.py (Voronoi brute force, half-space power diagram, exact
 * rational arithmetic, closed-form ellipse/Moebius volumes, ...).
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_apd_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * dim        2 or 3
 * n[3]       voxels per axis (n[2] ignored when dim == 2)
 * lo, hi     box
 * M          number of seeds
 * X[M*dim], A[M*dim*dim] (row-major), w[M]   fp64 (the caller widens the fp32 inputs exactly)
 * n_sel, sel voxels to evaluate: linear indices j = (iz*ny + iy)*nx + ix; sel == NULL means
 *            all voxels 0..N-1 in order (then n_sel must be N)
 * outputs (each length n_sel; any may be NULL):
 *   label     argmin index (0-based)
 *   best      min_i C_ij
 *   qbest     |y_j - x_i|^2_{A_i} of the winner (the second term of eq. 2.7)
 *   second    second smallest cost (over i != label); +inf when M == 1
 *   runner    index attaining `second`; -1 when M == 1
 */
int oracle_apd_assign(int dim, const int64_t *n, const double *lo, const double *hi,
                      int64_t M, const double *X, const double *A, const double *w,
                      int64_t n_sel, const int64_t *sel,
                      int32_t *label, double *best, double *qbest, double *second, int32_t *runner)
{
    if (dim != 2 && dim != 3) return -1;
    if (M < 1) return -1;
    const int64_t nx = n[0], ny = n[1], nz = (dim == 3) ? n[2] : 1;
    if (nx < 1 || ny < 1 || nz < 1) return -1;
    double s[3] = {0, 0, 0};
    for (int k = 0; k < dim; ++k) s[k] = (hi[k] - lo[k]) / (double)n[k];

    int64_t t;
#pragma omp parallel for schedule(static)
    for (t = 0; t < n_sel; ++t) {
        const int64_t j = sel ? sel[t] : t;
        int64_t idx[3];
        idx[0] = j % nx;
        idx[1] = (j / nx) % ny;
        idx[2] = j / (nx * ny);
        double y[3] = {0, 0, 0};
        for (int k = 0; k < dim; ++k) y[k] = lo[k] + ((double)idx[k] + 0.5) * s[k];

        double c1 = INFINITY, c2 = INFINITY, q1 = 0.0;
        int32_t i1 = -1, i2 = -1;
        for (int64_t i = 0; i < M; ++i) {
            double d[3];
            for (int k = 0; k < dim; ++k) d[k] = y[k] - X[i * dim + k];
            double q = 0.0;
            for (int k = 0; k < dim; ++k)
                for (int l = 0; l < dim; ++l)
                    q += d[k] * A[(i * dim + k) * dim + l] * d[l];
            const double c = q - w[i];
            if (c < c1) {
                c2 = c1; i2 = i1;
                c1 = c;  i1 = (int32_t)i; q1 = q;
            } else if (c < c2) {
                c2 = c;  i2 = (int32_t)i;
            }
        }
        if (label)  label[t] = i1;
        if (best)   best[t] = c1;
        if (qbest)  qbest[t] = q1;
        if (second) second[t] = c2;
        if (runner) runner[t] = i2;
    }
    return 0;
}

/* Cost of ONE named seed at each selected voxel (used to judge a mismatching GPU label:
 * DESIGN.md parity rule 1 needs c_{labels_gpu[j]}(y_j) in fp64). seed[t] is the seed index. */
int oracle_apd_cost_of(int dim, const int64_t *n, const double *lo, const double *hi,
                       int64_t M, const double *X, const double *A, const double *w,
                       int64_t n_sel, const int64_t *sel, const int32_t *seed, double *cost)
{
    if (dim != 2 && dim != 3) return -1;
    const int64_t nx = n[0], ny = n[1];
    double s[3] = {0, 0, 0};
    for (int k = 0; k < dim; ++k) s[k] = (hi[k] - lo[k]) / (double)n[k];
    for (int64_t t = 0; t < n_sel; ++t) {
        const int64_t j = sel[t];
        const int64_t i = seed[t];
        if (i < 0 || i >= M) return -2;
        int64_t idx[3];
        idx[0] = j % nx;
        idx[1] = (j / nx) % ny;
        idx[2] = j / (nx * ny);
        double d[3] = {0, 0, 0};
        for (int k = 0; k < dim; ++k) d[k] = (lo[k] + ((double)idx[k] + 0.5) * s[k]) - X[i * dim + k];
        double q = 0.0;
        for (int k = 0; k < dim; ++k)
            for (int l = 0; l < dim; ++l)
                q += d[k] * A[(i * dim + k) * dim + l] * d[l];
        cost[t] = q - w[i];
    }
    return 0;
}

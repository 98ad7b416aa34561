/*
 * oracle_cg.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (same rules as oracle_spmv.c).
 *
 * Plain conjugate gradients around the CSR row loop, for the "solver loop around apply"
 * row of SURVEY.md sec. 8(f) rank 3 (the paper's ref [1], is about iterative
 * solvers).  The paper does not write the algorithm; this is the textbook
 * Hestenes-Stiefel recurrence, step by step, fp64, every dot product summed left to right,
 * no fusion:
 *
 *     r0 = b - A x0,  p0 = r0,  rr = r0.r0
 *     repeat k = 0, 1, ...          (stop first when sqrt(rr) <= tol * ||b||, or k == max_iters)
 *         q     = A p
 *         alpha = rr / (p.q)
 *         x    += alpha p
 *         r    -= alpha q
 *         rr'   = r.r
 *         beta  = rr' / rr ;  rr = rr'
 *         p     = r + beta p
 *
 * Shares no code with the CUDA library; does not even include oracle_spmv.c (own row loop).
 *
 * Pins (tests/test_oracle_pins.py, "-m not gpu"): C1 solution vs numpy.linalg.solve on small SPD
 * systems; C2 A = I converges in one step, exactly; C3 finite termination: an SPD matrix with m
 * distinct eigenvalues converges in <= m steps; C4 2D Dirichlet Laplacian with b = A x_true
 * recovers x_true, with the residual norm it reports equal to ||b - A x|| recomputed;
 * C5 max_iters = 0 returns x0 and the initial residual.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

static void cg_matvec(int64_t rows, const int32_t *rp, const int32_t *ci, const double *va,
                      const double *x, double *y)
{
    for (int64_t i = 0; i < rows; ++i) {
        double s = 0.0;
        for (int32_t k = rp[i]; k < rp[i + 1]; ++k) s = s + va[k] * x[ci[k]];
        y[i] = s;
    }
}

static double cg_dot(int64_t n, const double *a, const double *b)
{
    double s = 0.0;
    for (int64_t i = 0; i < n; ++i) s = s + a[i] * b[i];
    return s;
}

/* x: initial guess in, solution out.  Returns the number of iterations done; *rel_res receives
 * sqrt(r.r)/||b|| of the recurrence residual (sqrt(r.r) itself when b == 0).
 * res_hist (may be NULL, max_iters+1 entries) receives sqrt(rr) before every iteration and at the end. */
int64_t oracle_cg(int64_t rows, const int32_t *rp, const int32_t *ci, const double *va,
                  const double *b, double *x, double tol, int64_t max_iters, double *rel_res,
                  double *res_hist)
{
    double *r = (double *)malloc(sizeof(double) * (size_t)(rows > 0 ? rows : 1));
    double *p = (double *)malloc(sizeof(double) * (size_t)(rows > 0 ? rows : 1));
    double *q = (double *)malloc(sizeof(double) * (size_t)(rows > 0 ? rows : 1));
    cg_matvec(rows, rp, ci, va, x, q);
    for (int64_t i = 0; i < rows; ++i) { r[i] = b[i] - q[i]; p[i] = r[i]; }
    double rr = cg_dot(rows, r, r);
    const double bnorm = sqrt(cg_dot(rows, b, b));
    const double stop = tol * bnorm;
    int64_t k = 0;
    for (;;) {
        if (res_hist) res_hist[k] = sqrt(rr);
        if (sqrt(rr) <= stop || k == max_iters) break;
        cg_matvec(rows, rp, ci, va, p, q);
        const double pq = cg_dot(rows, p, q);
        if (!(pq > 0.0)) break;                 /* not SPD (or breakdown): stop, as the GPU path does */
        const double alpha = rr / pq;
        for (int64_t i = 0; i < rows; ++i) x[i] = x[i] + alpha * p[i];
        for (int64_t i = 0; i < rows; ++i) r[i] = r[i] - alpha * q[i];
        const double rr_new = cg_dot(rows, r, r);
        const double beta = rr_new / rr;
        rr = rr_new;
        for (int64_t i = 0; i < rows; ++i) p[i] = r[i] + beta * p[i];
        ++k;
    }
    if (rel_res) *rel_res = bnorm > 0.0 ? sqrt(rr) / bnorm : sqrt(rr);
    free(r); free(p); free(q);
    return k;
}

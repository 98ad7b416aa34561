/*
 * oracle_jacobi.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (same rules as oracle_spmv.c).
 *
 * Weighted (damped) Jacobi iteration around the CSR row loop, the second solver loop SURVEY.md sec. 8(f) rank 3
 * names ("CG / Jacobi using spmv_apply"; the paper's ref [1], is about iterative solvers).  The
 * paper does not write the algorithm; this is the textbook stationary iteration, step by step, fp64, every sum
 * left to right, no fusion:
 *
 *     d_i = sum of the stored entries (i, i) of row i, in stored order     (duplicates sum, reading A8)
 *     repeat k = 0, 1, ...
 *         t   = A x_k
 *         r_k = b - t
 *         stop when ||r_k||_2 <= tol * ||b||_2, or k == max_iters          (the test comes BEFORE the update)
 *         x_{k+1} = x_k + omega * (r_k / d)                                (element by element)
 *
 * Shares no code with the CUDA library; does not include the other oracle files (own row loop).
 *
 * Pins (tests/test_oracle_pins.py, "-m not gpu"): J1 closed form on Dirichlet Laplacians: with b = lambda_m v_m
 * (sine eigenvector) and x_0 = 0 the iterate is x_k = (1 - rho^k) v_m and ||r_k|| = rho^k ||b||, rho = 1 - omega
 * lambda_m / d; J2 a diagonal matrix with omega = 1 is solved by the first update, bit for bit b_i / d_i;
 * J3 the limit equals numpy.linalg.solve on strictly diagonally dominant NON-symmetric matrices with a varying
 * diagonal (a transposed product, a wrong diagonal index or a wrong sign fails it); J4 max_iters = 0 returns x_0
 * and the initial residual, b = 0 stops at once; J5 duplicate diagonal entries sum, a zero diagonal is refused.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

/* x: initial guess in, iterate out.  Returns the number of updates done, or -1 if some d_i == 0 (x untouched).
 * *rel_res receives ||r_k|| / ||b|| of the LAST residual computed (that of the returned x; ||r_k|| itself when
 * b == 0).  res_hist (may be NULL, max_iters + 1 entries) receives ||r_k|| for k = 0 .. returned value. */
int64_t oracle_jacobi(int64_t rows, const int32_t *rp, const int32_t *ci, const double *va,
                      const double *b, double *x, double omega, double tol, int64_t max_iters,
                      double *rel_res, double *res_hist)
{
    const size_t n = (size_t)(rows > 0 ? rows : 1);
    double *d = (double *)malloc(sizeof(double) * n);
    double *r = (double *)malloc(sizeof(double) * n);
    for (int64_t i = 0; i < rows; ++i) {
        double s = 0.0;
        for (int32_t k = rp[i]; k < rp[i + 1]; ++k)
            if (ci[k] == i) s = s + va[k];
        d[i] = s;
        if (s == 0.0) { free(d); free(r); return -1; }
    }
    double bb = 0.0;
    for (int64_t i = 0; i < rows; ++i) bb = bb + b[i] * b[i];
    const double bnorm = sqrt(bb);
    const double stop = tol * bnorm;
    int64_t k = 0;
    double rr = 0.0;
    for (;;) {
        for (int64_t i = 0; i < rows; ++i) {
            double t = 0.0;
            for (int32_t j = rp[i]; j < rp[i + 1]; ++j) t = t + va[j] * x[ci[j]];
            r[i] = b[i] - t;
        }
        rr = 0.0;
        for (int64_t i = 0; i < rows; ++i) rr = rr + r[i] * r[i];
        if (res_hist) res_hist[k] = sqrt(rr);
        if (sqrt(rr) <= stop || k == max_iters) break;
        for (int64_t i = 0; i < rows; ++i) x[i] = x[i] + omega * (r[i] / d[i]);
        ++k;
    }
    if (rel_res) *rel_res = bnorm > 0.0 ? sqrt(rr) / bnorm : sqrt(rr);
    free(d); free(r);
    return k;
}

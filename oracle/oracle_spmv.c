/*
 * oracle_spmv.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU definition of the hot path
 *     y = alpha * A * x + beta * y,   A in CSR, fp64 values, int32 indices.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may build, link or call anything in this directory.
 * The CUDA library (paper_1309_1894_b200/csrc) shares no code, header,
 * table or helper with this file and never calls it.
 *
 * What it follows:
 *   - PAPER.md:19 (sec. 2 "Approach"): the un-annotated program "acts as a
 *     reference implementation that can be compiled and executed to obtain
 *     reference results"; every variant's outputs are compared with these.
 *   - BASELINE.json north_star: "a plain serial C++ row loop in fp64 that
 *     shares no code with the GPU path"; formula y = alpha*A*x + beta*y;
 *     tolerance "per-row relative 1e-12 measured against sum_j |a_ij*x_j|".
 *   - SURVEY.md sec. 8(c): step-by-step statement and readings A1-A9.
 *
 * SpMV has a plain mathematical definition, so the oracle IS that definition
 * written as the obvious loop: stored order, one rounding per multiply, one
 * rounding per add (compile with -ffp-contract=off so no FMA is formed).
 *
 * Pins (tests/test_oracle_pins.py, all "-m not gpu"):
 *   P1 brute-force dense matvec 1..64 rows (bitwise), P2 A*1 on Dirichlet
 *   Laplacians (exact integers), P3 sin eigenvectors, P4 row permutation
 *   invariance (bitwise), P5 x=e_j, P6 small-integer exactness, P7 val=1,x=1
 *   gives row lengths, P8 identity/diagonal/dense-row/alpha=2^k/alpha=0
 *   special cases, P9 long-double accumulation bound, scipy.sparse and numpy
 *   dense products as library cross-checks.
 * Every function here is pinned; nothing is "parity unpinned". (The
 * generator-shape readings A11/A13/A14/A16 are unpinned; they live in
 * paper_1309_1894_b200/workloads.py, not here.)
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

#ifdef _OPENMP
#include <omp.h>
#endif

/* One row of SURVEY 8(c) step 2: s = sum_k val[k]*x[col[k]] in stored order,
 * a = sum_k |val[k]*x[col[k]]|; then the BLAS-style epilogue (A1: y not read
 * when beta == 0) and the tolerance denominator (A4). */
static void oracle_row(int64_t i, const int32_t *row_ptr, const int32_t *col_idx,
                       const double *val, double alpha, const double *x,
                       double beta, double *y, double *scale_out)
{
    double s = 0.0, a = 0.0;
    for (int32_t k = row_ptr[i]; k < row_ptr[i + 1]; ++k) {
        double t = val[k] * x[col_idx[k]];
        s = s + t;
        a = a + fabs(t);
    }
    if (beta == 0.0) {
        y[i] = alpha * s;
        if (scale_out) scale_out[i] = fabs(alpha) * a;
    } else {
        double by = beta * y[i];
        y[i] = alpha * s + by;
        if (scale_out) scale_out[i] = fabs(alpha) * a + fabs(by);
    }
}

/* alpha == 0 (reading A2, BLAS convention): A and x are not referenced. */
static void oracle_alpha_zero(int64_t rows, double beta, double *y, double *scale_out)
{
    for (int64_t i = 0; i < rows; ++i) {
        if (beta == 0.0) {
            y[i] = 0.0;
            if (scale_out) scale_out[i] = 0.0;
        } else {
            double by = beta * y[i];
            y[i] = by;
            if (scale_out) scale_out[i] = fabs(by);
        }
    }
}

/* THE oracle. y is updated in place; scale_out (may be NULL) receives the
 * per-row tolerance denominator |alpha|*sum|a_ij x_j| + |beta*y_old|. */
void oracle_spmv(int64_t rows, const int32_t *row_ptr, const int32_t *col_idx,
                 const double *val, double alpha, const double *x, double beta,
                 double *y, double *scale_out)
{
    if (alpha == 0.0) {
        oracle_alpha_zero(rows, beta, y, scale_out);
        return;
    }
    for (int64_t i = 0; i < rows; ++i)
        oracle_row(i, row_ptr, col_idx, val, alpha, x, beta, y, scale_out);
}

/* The same row loop, rows split over threads. Rows are independent and each
 * row is still summed serially in stored order, so the result is bit-identical
 * to oracle_spmv (asserted in tests). Used only as the timed CPU baseline.
 * Returns the number of threads used. */
int oracle_spmv_omp(int64_t rows, const int32_t *row_ptr, const int32_t *col_idx,
                    const double *val, double alpha, const double *x, double beta,
                    double *y, double *scale_out)
{
    int nthreads = 1;
    if (alpha == 0.0) {
        oracle_alpha_zero(rows, beta, y, scale_out);
        return nthreads;
    }
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        nthreads = omp_get_num_threads();
#pragma omp for schedule(static, 4096)
        for (int64_t i = 0; i < rows; ++i)
            oracle_row(i, row_ptr, col_idx, val, alpha, x, beta, y, scale_out);
    }
#else
    for (int64_t i = 0; i < rows; ++i)
        oracle_row(i, row_ptr, col_idx, val, alpha, x, beta, y, scale_out);
#endif
    return nthreads;
}

/* Test-only: the same definition with long double (x87 80-bit) accumulation,
 * products formed exactly enough (53x53 bits fit 64-bit mantissa + 1 rounding).
 * NOT the oracle; it bounds the oracle's own rounding error (pin P9). */
void oracle_spmv_ext(int64_t rows, const int32_t *row_ptr, const int32_t *col_idx,
                     const double *val, double alpha, const double *x, double beta,
                     double *y)
{
    for (int64_t i = 0; i < rows; ++i) {
        long double s = 0.0L;
        if (alpha != 0.0)
            for (int32_t k = row_ptr[i]; k < row_ptr[i + 1]; ++k)
                s += (long double)val[k] * (long double)x[col_idx[k]];
        long double r = (long double)alpha * s;
        if (beta != 0.0) r += (long double)beta * (long double)y[i];
        y[i] = (double)r;
    }
}

int oracle_long_double_bits(void) { return (int)(sizeof(long double) * 8); }

/* Acceptance rule of SURVEY 8(c) / north_star: for every row
 *   |y_test - y_ref| <= tol * scale;  scale == 0 -> values must be equal;
 *   NaN must match NaN, +-Inf must match the same signed infinity.
 * Outputs: max over rows of |diff|/scale (rows with scale > 0), the index of
 * the first failing row (-1 if none) and the number of failing rows. */
void oracle_accept(int64_t rows, const double *y_test, const double *y_ref,
                   const double *scale, double tol, double *max_ratio,
                   int64_t *first_fail, int64_t *n_fail)
{
    double mr = 0.0;
    int64_t ff = -1, nf = 0;
    for (int64_t i = 0; i < rows; ++i) {
        double t = y_test[i], r = y_ref[i];
        int ok;
        if (isnan(r)) {
            ok = isnan(t);
        } else if (isinf(r)) {
            ok = (t == r);
        } else if (isnan(t) || isinf(t)) {
            ok = 0;
        } else {
            double d = fabs(t - r), sc = scale[i];
            if (sc == 0.0 || isnan(sc)) {
                ok = (t == r);
            } else if (isinf(sc)) {
                ok = 1;
            } else {
                double q = d / sc;
                if (q > mr) mr = q;
                ok = (d <= tol * sc);
            }
        }
        if (!ok) {
            if (ff < 0) ff = i;
            ++nf;
        }
    }
    *max_ratio = mr;
    *first_fail = ff;
    *n_fail = nf;
}

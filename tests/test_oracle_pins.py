"""Pins for oracle/ (CPU only).  Each test cites the pin id of SURVEY.md sec. 8(c) and
the statement of BASELINE.json:north_star it enforces: "(i) brute-force dense matvec on
matrices of 1 to 64 rows, (ii) closed forms for Laplacian stencils ..., (iii) invariance
under row permutation".  None of the expected values below is produced by oracle/ or by
the CUDA path: they are closed forms, exact integers, brute force written differently
(dense, pure Python floats) or library routines (numpy dense matmul, scipy.sparse).
"""
import math

import numpy as np
import pytest
import scipy.sparse as sp

import oracle
from paper_1309_1894_b200 import workloads as W


def _dense(A):
    D = np.zeros((A.rows, A.cols))
    for i in range(A.rows):
        for k in range(A.row_ptr[i], A.row_ptr[i + 1]):
            D[i, A.col_idx[k]] += A.val[k]
    return D


def _random_small(rows, cols, density, seed, sort=True):
    rng = np.random.default_rng(seed)
    lengths = rng.binomial(cols, density, size=rows)
    if rows > 2:
        lengths[rng.integers(rows)] = 0          # always include an empty row
    return W.csr_from_lengths(lengths, cols, 100 + seed, sort=sort)


# ---- P1: brute-force dense matvec, 1..64 rows, bitwise -------------------------------
@pytest.mark.parametrize("rows", [1, 2, 3, 5, 8, 13, 31, 32, 33, 64])
@pytest.mark.parametrize("density", [0.0, 0.1, 0.5, 1.0])
def test_p1_dense_bruteforce_bitwise(rows, density):
    for cols in (rows, max(1, rows // 2), rows + 7):          # square and rectangular
        A = _random_small(rows, cols, density, rows * 7 + cols)
        D = _dense(A)
        x = W.uniform(3, cols)
        y0 = W.uniform(4, rows)
        for alpha, beta in ((1.0, 0.0), (1.0, 0.5), (-2.5, 1.0), (0.75, -0.25)):
            y, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, alpha, x, beta, y0)
            for i in range(rows):
                s = 0.0
                a = 0.0
                for j in range(cols):          # left to right, unfused python floats;
                    t = float(D[i, j]) * float(x[j])   # structural zeros add exact 0.0
                    s = s + t
                    a = a + abs(t)
                e = alpha * s if beta == 0.0 else alpha * s + beta * float(y0[i])
                sc = abs(alpha) * a + (0.0 if beta == 0.0 else abs(beta * float(y0[i])))
                assert y[i] == e, (rows, cols, i)
                assert scale[i] == pytest.approx(sc, rel=1e-15, abs=0)


def test_p1_library_crosscheck_numpy_scipy():
    A = _random_small(64, 50, 0.3, 99)
    x = W.uniform(5, 50)
    y0 = W.uniform(6, 64)
    y, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.5, x, -0.5, y0)
    M = sp.csr_matrix((A.val, A.col_idx, A.row_ptr), shape=(64, 50))
    np.testing.assert_allclose(y, 1.5 * (M @ x) - 0.5 * y0, rtol=0, atol=1e-13)
    np.testing.assert_allclose(y, 1.5 * (_dense(A) @ x) - 0.5 * y0, rtol=0, atol=1e-13)
    np.testing.assert_allclose(scale, 1.5 * (abs(M) @ abs(x)) + abs(0.5 * y0), rtol=1e-14)


# ---- P2: A*ones on Dirichlet Laplacians: exact integers ------------------------------
def _boundary_count(n, dim):
    idx = np.arange(n ** dim)
    cnt = np.zeros(n ** dim, dtype=int)
    for d in range(dim):
        c = (idx // n ** d) % n
        cnt += (c == 0).astype(int) + (c == n - 1).astype(int)
    return cnt


@pytest.mark.parametrize("n", [3, 5, 8])
def test_p2_laplacian_times_ones(n):
    A = W.laplace2d_5pt(n)
    y, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, np.ones(A.cols), 0.0)
    assert np.array_equal(y, _boundary_count(n, 2).astype(float))     # 0 interior,1 edge,2 corner
    A = W.laplace3d_7pt(n)
    y, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, np.ones(A.cols), 0.0)
    assert np.array_equal(y, _boundary_count(n, 3).astype(float))     # 0/1/2/3
    A = W.stencil3d_27pt(n)
    y, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, np.ones(A.cols), 0.0)
    # 27-pt, diag 26, off -1: row sum = 27 - (#present points); a point on b boundary
    # planes (n >= 3) has 27 * (2/3)^b ... explicitly 27,18,12,8 present -> 0,9,15,19
    present = {0: 27, 1: 18, 2: 12, 3: 8}
    b = _boundary_count(n, 3)
    assert np.array_equal(y, np.array([27.0 - present[int(v)] for v in b]))


# ---- P3: sin eigenvectors ------------------------------------------------------------
@pytest.mark.parametrize("n,p,q,r", [(6, 1, 1, 1), (7, 2, 3, 1), (9, 4, 1, 5)])
def test_p3_sin_eigenvectors(n, p, q, r):
    th = lambda m: m * math.pi / (n + 1)
    s = lambda m: np.sin(th(m) * (np.arange(n) + 1))
    # 2D: row = i + n*j
    v2 = np.kron(s(q), s(p))
    lam2 = 4 - 2 * math.cos(th(p)) - 2 * math.cos(th(q))
    A = W.laplace2d_5pt(n)
    y, sc = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, v2, 0.0)
    assert np.all(np.abs(y - lam2 * v2) <= 1e-12 * sc + 1e-300)
    v3 = np.kron(s(r), np.kron(s(q), s(p)))
    lam7 = 6 - 2 * (math.cos(th(p)) + math.cos(th(q)) + math.cos(th(r)))
    A = W.laplace3d_7pt(n)
    y, sc = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, v3, 0.0)
    assert np.all(np.abs(y - lam7 * v3) <= 1e-12 * sc + 1e-300)
    # 27-pt (diag 26, off -1) = 27 I - T(x)T(x)T, T = tridiag(1,1,1): eig 1 + 2cos(theta)
    lam27 = 27 - (1 + 2 * math.cos(th(p))) * (1 + 2 * math.cos(th(q))) * (1 + 2 * math.cos(th(r)))
    A = W.stencil3d_27pt(n)
    y, sc = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, v3, 0.0)
    assert np.all(np.abs(y - lam27 * v3) <= 1e-12 * sc + 1e-300)
    # and with alpha/beta: alpha*A*v + beta*v = (alpha*lam + beta) v
    y, sc = oracle.spmv(A.row_ptr, A.col_idx, A.val, 0.5, v3, 2.0, v3)
    assert np.all(np.abs(y - (0.5 * lam27 + 2.0) * v3) <= 1e-12 * sc + 1e-300)


# ---- P4: row permutation invariance (bitwise) ----------------------------------------
def test_p4_row_permutation_bitwise():
    A = W.powerlaw(2000, lmax=300)
    x = W.uniform(7, A.cols)
    y0 = W.uniform(8, A.rows)
    y, sc = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.25, x, 0.5, y0)
    perm = np.random.default_rng(1).permutation(A.rows)
    lens = A.row_lengths()[perm]
    rp = np.zeros(A.rows + 1, dtype=np.int64)
    np.cumsum(lens, out=rp[1:])
    ci = np.concatenate([A.col_idx[A.row_ptr[i]:A.row_ptr[i + 1]] for i in perm])
    va = np.concatenate([A.val[A.row_ptr[i]:A.row_ptr[i + 1]] for i in perm])
    yp, scp = oracle.spmv(rp, ci, va, 1.25, x, 0.5, y0[perm])
    assert np.array_equal(yp, y[perm]) and np.array_equal(scp, sc[perm])


# ---- P5: x = e_j picks out column j exactly ------------------------------------------
def test_p5_unit_vectors():
    A = _random_small(40, 30, 0.3, 5)
    D = _dense(A)
    for j in range(30):
        e = np.zeros(30)
        e[j] = 1.0
        y, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 2.0, e, 0.0)
        assert np.array_equal(y, 2.0 * D[:, j])


# ---- P6: small integers -> exact in any order ----------------------------------------
def test_p6_small_integers_exact():
    lengths = np.random.default_rng(2).integers(0, 200, size=300)
    A = W.csr_from_lengths(lengths, 4000, 11, values="smallint")
    x = np.round(W.uniform(12, A.cols) * 8)
    y0 = np.round(W.uniform(13, A.rows) * 8)
    y, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 3.0, x, -2.0, y0)
    M = sp.csr_matrix((A.val.astype(np.int64), A.col_idx, A.row_ptr), shape=(A.rows, A.cols))
    e = 3 * (M @ x.astype(np.int64)) - 2 * y0.astype(np.int64)
    assert np.array_equal(y, e.astype(np.float64))


# ---- P7: val = 1, x = 1 -> row lengths -----------------------------------------------
def test_p7_row_lengths():
    lengths = [0, 1, 2, 3, 31, 32, 33, 0, 0, 1023, 1025, 5, 0]
    A = W.csr_from_lengths(lengths, 5000, 21, values="ones")
    y, sc = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, np.ones(A.cols), 0.0)
    assert np.array_equal(y, np.array(lengths, dtype=float))
    assert np.array_equal(sc, np.array(lengths, dtype=float))


# ---- P8: special cases reducing to textbook routines ---------------------------------
def test_p8_identity_is_axpby():
    n = 257
    rp = np.arange(n + 1)
    x = W.uniform(1, n)
    y0 = W.uniform(2, n)
    y, _ = oracle.spmv(rp, np.arange(n), np.ones(n), 0.3, x, 0.7, y0)
    assert np.array_equal(y, 0.3 * x + 0.7 * y0)


def test_p8_diagonal_is_elementwise():
    n = 100
    d = W.normal(3, n)
    x = W.uniform(4, n)
    y, _ = oracle.spmv(np.arange(n + 1), np.arange(n), d, 1.0, x, 0.0)
    assert np.array_equal(y, d * x)


def test_p8_single_dense_row_is_dot():
    n = 20000
    y, _ = oracle.spmv(np.array([0, n]), np.arange(n), np.ones(n), 1.0, np.arange(1, n + 1.0), 0.0)
    assert y[0] == n * (n + 1) / 2
    # N x 1 column matrix
    y, _ = oracle.spmv(np.arange(6), np.zeros(5, dtype=int), np.arange(1.0, 6.0), 2.0, np.array([3.0]), 0.0)
    assert np.array_equal(y, 6.0 * np.arange(1.0, 6.0))


def test_p8_power_of_two_alpha_scales_exactly():
    A = _random_small(50, 50, 0.2, 8)
    x = W.uniform(9, 50)
    y1, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x, 0.0)
    y8, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 8.0, x, 0.0)
    assert np.array_equal(y8, 8.0 * y1)


def test_p8_alpha_zero_and_beta_cases():
    A = _random_small(30, 30, 0.3, 10)
    x = W.uniform(1, 30)
    x[3] = np.inf                                   # A, x not referenced when alpha == 0 (A2)
    y0 = W.uniform(2, 30)
    y, sc = oracle.spmv(A.row_ptr, A.col_idx, A.val, 0.0, x, 1.0, y0)
    assert np.array_equal(y, y0) and np.array_equal(sc, np.abs(y0))
    y, sc = oracle.spmv(A.row_ptr, A.col_idx, A.val, 0.0, x, 0.0, np.full(30, np.nan))
    assert np.array_equal(y, np.zeros(30)) and not np.any(sc)
    # beta == 0: incoming y is never read (A1): NaN does not propagate
    x = W.uniform(1, 30)
    y, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x, 0.0, np.full(30, np.nan))
    assert np.all(np.isfinite(y))
    # empty rows (A9): y_i = beta*y_i exactly
    lengths = [0, 3, 0, 0, 2, 0]
    B = W.csr_from_lengths(lengths, 10, 3)
    y, sc = oracle.spmv(B.row_ptr, B.col_idx, B.val, 1.0, W.uniform(5, 10), 0.5, np.arange(6.0))
    for i in (0, 2, 3, 5):
        assert y[i] == 0.5 * i and sc[i] == 0.5 * i


def test_duplicate_and_unsorted_columns_sum():
    # A8: duplicates sum, order is the stored order
    rp = np.array([0, 4, 6])
    ci = np.array([2, 0, 2, 1, 1, 1])
    va = np.array([1.0, 2.0, 3.0, 4.0, 5.0, -5.0])
    x = np.array([10.0, 100.0, 1000.0])
    y, sc = oracle.spmv(rp, ci, va, 1.0, x, 0.0)
    assert np.array_equal(y, [4000.0 + 20.0 + 400.0, 0.0])
    assert np.array_equal(sc, [4420.0, 1000.0])


# ---- P9: the oracle's own rounding error vs extended precision -----------------------
def test_p9_extended_precision_bound():
    assert oracle.long_double_bits() >= 96, "x87 80-bit long double expected on this host"
    for prob in (W.config(1), W.config(2, 0.25), W.config(3, 1 / 64), W.config(4, 0.1), W.config(5, 0.2)):
        A = prob.A
        y, sc = oracle.spmv(A.row_ptr, A.col_idx, A.val, prob.alpha, prob.x, prob.beta, prob.y0)
        ye = oracle.spmv_ext(A.row_ptr, A.col_idx, A.val, prob.alpha, prob.x, prob.beta, prob.y0)
        assert np.all(np.abs(y - ye) <= 1e-13 * sc), prob.name


def test_parallel_oracle_is_bit_identical():
    prob = W.config(3, 1 / 32)
    A = prob.A
    y, sc = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, prob.x, 0.0)
    yp, scp = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, prob.x, 0.0, parallel=True)
    assert np.array_equal(y, yp) and np.array_equal(sc, scp)


# ---- acceptance rule -----------------------------------------------------------------
def test_accept_rule():
    ref = np.array([1.0, 0.0, np.nan, np.inf, -np.inf, 5.0])
    sc = np.array([1.0, 0.0, 1.0, 1.0, 1.0, 10.0])
    ok, mr, ff, nf = oracle.accept(ref.copy(), ref, sc)
    assert ok and nf == 0
    t = ref.copy(); t[0] += 5e-13                    # inside 1e-12
    assert oracle.accept(t, ref, sc)[0]
    t = ref.copy(); t[0] += 2e-12
    ok, mr, ff, nf = oracle.accept(t, ref, sc)
    assert not ok and ff == 0 and nf == 1 and mr == pytest.approx(2e-12, rel=1e-3)
    t = ref.copy(); t[1] = 1e-300                    # scale 0 -> exact
    assert not oracle.accept(t, ref, sc)[0]
    t = ref.copy(); t[1] = -0.0                      # -0 == +0
    assert oracle.accept(t, ref, sc)[0]
    t = ref.copy(); t[2] = 1.0
    assert not oracle.accept(t, ref, sc)[0]
    t = ref.copy(); t[3] = -np.inf
    assert not oracle.accept(t, ref, sc)[0]
    t = ref.copy(); t[5] = np.nan
    assert not oracle.accept(t, ref, sc)[0]


# ----------------------------------------------------------------------------
# CG oracle (oracle_cg.c) -- pins C1..C5
# ----------------------------------------------------------------------------
def _dense(A):
    D = np.zeros((A.rows, A.cols))
    for i in range(A.rows):
        for k in range(A.row_ptr[i], A.row_ptr[i + 1]):
            D[i, A.col_idx[k]] += A.val[k]
    return D


@pytest.mark.parametrize("n", [3, 7, 12])
def test_c1_cg_matches_dense_solve(n):
    A = W.laplace2d_5pt(n)
    D = _dense(A)
    b = W.uniform(90, A.rows)
    x, k, rel, hist = oracle.cg(A.row_ptr, A.col_idx, A.val, b, tol=1e-13, max_iters=500)
    xs = np.linalg.solve(D, b)
    assert np.abs(x - xs).max() <= 1e-10 * np.abs(xs).max()
    assert rel <= 1e-13 and k < 500 and hist.size == k + 1


def test_c2_identity_converges_in_one_exact_step():
    n = 50
    I = W.CSR(n, n, np.arange(n + 1, dtype=np.int32), np.arange(n, dtype=np.int32), np.ones(n))
    b = W.uniform(91, n)
    x, k, rel, hist = oracle.cg(I.row_ptr, I.col_idx, I.val, b, tol=1e-15, max_iters=10)
    assert k == 1 and np.array_equal(x, b) and rel == 0.0


def test_c3_finite_termination_with_m_distinct_eigenvalues():
    # diagonal SPD matrix with 4 distinct eigenvalues: CG must converge in <= 4 steps
    n = 64
    d = np.array([1.0, 2.0, 5.0, 9.0])[np.arange(n) % 4]
    Dg = W.CSR(n, n, np.arange(n + 1, dtype=np.int32), np.arange(n, dtype=np.int32), d)
    b = W.uniform(92, n)
    x, k, rel, _ = oracle.cg(Dg.row_ptr, Dg.col_idx, Dg.val, b, tol=1e-12, max_iters=50)
    assert k <= 4 and np.abs(x - b / d).max() <= 1e-12


def test_c4_recovers_x_true_and_reports_the_true_residual():
    A = W.laplace2d_5pt(20)
    xt = W.uniform(93, A.rows)
    b, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, xt, 0.0)
    x, k, rel, hist = oracle.cg(A.row_ptr, A.col_idx, A.val, b, tol=1e-12, max_iters=400)
    assert np.abs(x - xt).max() <= 1e-9
    Ax, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x, 0.0)
    true_rel = np.linalg.norm(b - Ax) / np.linalg.norm(b)
    assert abs(true_rel - rel) <= 1e-12 and rel <= 1e-12
    assert hist[0] == pytest.approx(np.linalg.norm(b), rel=1e-14)      # x0 = 0: r0 = b


def test_c5_zero_iterations_and_initial_guess():
    A = W.laplace2d_5pt(6)
    b = W.uniform(94, A.rows)
    x0 = W.uniform(95, A.rows)
    x, k, rel, hist = oracle.cg(A.row_ptr, A.col_idx, A.val, b, x0=x0, tol=1e-12, max_iters=0)
    Ax0, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x0, 0.0)
    assert k == 0 and np.array_equal(x, x0)
    assert rel == pytest.approx(np.linalg.norm(b - Ax0) / np.linalg.norm(b), rel=1e-13)
    # starting at the solution: no iteration needed
    xs = np.linalg.solve(_dense(A), b)
    _, k2, rel2, _ = oracle.cg(A.row_ptr, A.col_idx, A.val, b, x0=xs, tol=1e-10, max_iters=100)
    assert k2 == 0 and rel2 <= 1e-10


# ------------------------------------------------------------------ J1-J5: the weighted-Jacobi oracle (oracle_jacobi.c)
def _sine_mode(n, dim, m):
    """Eigenvector / eigenvalue of the Dirichlet Laplacian (diag 2*dim, off -1) on an n^dim grid: product of sines."""
    i = np.arange(1, n + 1)
    lam = 0.0
    v = np.ones(1)
    for mm in m[:dim]:
        v = np.kron(np.sin(mm * np.pi * i / (n + 1)), v)       # first index fastest: row = i + n*j
        lam += 2.0 - 2.0 * np.cos(mm * np.pi / (n + 1))
    return v, lam


@pytest.mark.parametrize("dim,n,m,omega", [(2, 12, (1, 1), 1.0), (2, 12, (3, 7), 0.8), (2, 9, (9, 9), 2.0 / 3.0), (3, 6, (2, 5, 1), 0.9)])
def test_j1_jacobi_closed_form_on_laplacian_eigenvectors(dim, n, m, omega):
    """b = lambda v (v a sine eigenvector), x0 = 0: x_k = (1 - rho^k) v and ||r_k|| = |rho|^k ||b|| with
    rho = 1 - omega lambda / d (textbook: the Jacobi iteration matrix I - omega D^-1 A shares A's eigenvectors
    when the diagonal is constant)."""
    A = W.laplace2d_5pt(n) if dim == 2 else W.laplace3d_7pt(n)
    v, lam = _sine_mode(n, dim, m)
    d = 2.0 * dim
    rho = 1.0 - omega * lam / d
    b = lam * v
    for k in (1, 2, 7, 20):
        x, it, rel, hist = oracle.jacobi(A.row_ptr, A.col_idx, A.val, b, omega=omega, tol=0.0, max_iters=k)
        assert it == k and hist.size == k + 1
        assert np.abs(x - (1.0 - rho ** k) * v).max() <= 1e-13
        want = np.abs(rho) ** np.arange(k + 1) * np.linalg.norm(b)
        assert np.abs(hist - want).max() <= 1e-12 * np.linalg.norm(b)
        assert rel == pytest.approx(abs(rho) ** k, abs=1e-13)


def test_j2_diagonal_matrix_is_solved_by_the_first_update_exactly():
    n = 40
    d = 0.5 + np.arange(n) % 7
    Dg = W.CSR(n, n, np.arange(n + 1, dtype=np.int32), np.arange(n, dtype=np.int32), d)
    b = W.uniform(96, n)
    x, k, rel, hist = oracle.jacobi(Dg.row_ptr, Dg.col_idx, Dg.val, b, omega=1.0, tol=1e-15, max_iters=10)
    assert k == 1 and np.array_equal(x, b / d) and rel <= 1e-15
    assert hist[0] == pytest.approx(np.linalg.norm(b), rel=1e-15)


@pytest.mark.parametrize("seed,omega", [(0, 1.0), (1, 0.7), (2, 1.0)])
def test_j3_jacobi_limit_is_the_dense_solution_nonsymmetric(seed, omega):
    """Strictly row-diagonally-dominant, NON-symmetric, varying diagonal of both signs: Jacobi converges, and to
    numpy.linalg.solve's answer.  A^T instead of A, d_j instead of d_i, or a sign slip cannot pass."""
    rng = np.random.default_rng(seed)
    n = 60
    lens = rng.integers(2, 9, n)
    A = W.csr_from_lengths(lens, n, 97 + seed)
    D = _dense(A)
    np.fill_diagonal(D, 0.0)
    diag = (np.abs(D).sum(axis=1) * 1.5 + 1.0) * np.where(np.arange(n) % 3 == 0, -1.0, 1.0)
    D[np.arange(n), np.arange(n)] = diag
    rp = [0]; ci = []; va = []
    for i in range(n):
        nz = np.nonzero(D[i])[0]
        ci += nz.tolist(); va += D[i, nz].tolist(); rp.append(len(ci))
    rp, ci, va = np.array(rp, np.int32), np.array(ci, np.int32), np.array(va)
    assert not np.allclose(D, D.T)
    b = W.uniform(99 + seed, n)
    x, k, rel, hist = oracle.jacobi(rp, ci, va, b, omega=omega, tol=1e-14, max_iters=2000)
    xs = np.linalg.solve(D, b)
    assert 0 < k < 2000 and rel <= 1e-14
    assert np.abs(x - xs).max() <= 1e-12 * np.abs(xs).max()
    assert np.all(np.diff(hist) < 0)                               # monotone in this (dominant) case


def test_j4_zero_iterations_initial_guess_and_zero_rhs():
    A = W.laplace2d_5pt(6)
    b = W.uniform(94, A.rows)
    x0 = W.uniform(95, A.rows)
    x, k, rel, hist = oracle.jacobi(A.row_ptr, A.col_idx, A.val, b, x0=x0, tol=1e-12, max_iters=0)
    Ax0, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x0, 0.0)
    assert k == 0 and np.array_equal(x, x0)
    assert rel == pytest.approx(np.linalg.norm(b - Ax0) / np.linalg.norm(b), rel=1e-13)
    xs = np.linalg.solve(_dense(A), b)                                  # starting at the solution: no update
    x2, k2, rel2, _ = oracle.jacobi(A.row_ptr, A.col_idx, A.val, b, x0=xs, tol=1e-10, max_iters=100)
    assert k2 == 0 and np.array_equal(x2, xs)
    x3, k3, rel3, _ = oracle.jacobi(A.row_ptr, A.col_idx, A.val, np.zeros(A.rows), tol=1e-10, max_iters=100)
    assert k3 == 0 and rel3 == 0.0 and not x3.any()


def test_j5_duplicate_diagonal_entries_sum_and_zero_diagonal_is_refused():
    # row 0: (0,0)=1.5 and (0,0)=2.5 -> d_0 = 4; row 1: d_1 = 2; off-diagonals small
    rp = np.array([0, 3, 5], dtype=np.int32)
    ci = np.array([0, 1, 0, 0, 1], dtype=np.int32)
    va = np.array([1.5, 0.5, 2.5, -0.25, 2.0])
    b = np.array([1.0, -2.0])
    x, k, rel, _ = oracle.jacobi(rp, ci, va, b, omega=1.0, tol=0.0, max_iters=1)
    assert k == 1 and np.array_equal(x, np.array([1.0 / 4.0, -2.0 / 2.0]))       # x0 = 0: x1 = b / d
    xs = np.linalg.solve(np.array([[4.0, 0.5], [-0.25, 2.0]]), b)
    x, k, rel, _ = oracle.jacobi(rp, ci, va, b, tol=1e-15, max_iters=200)
    assert np.abs(x - xs).max() <= 1e-14
    x0 = np.array([3.0, 4.0])
    xz, kz, _, _ = oracle.jacobi(np.array([0, 1, 2], np.int32), np.array([1, 1], np.int32), np.array([1.0, 1.0]), b, x0=x0)
    assert kz == -1 and np.array_equal(xz, x0)                           # row 0 has no diagonal entry

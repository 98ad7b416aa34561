"""GPU tests of spmv_jacobi ("CG / Jacobi using spmv_apply") against the plain
weighted-Jacobi oracle (oracle/oracle_jacobi.c).  Jacobi is a stationary linear iteration: the GPU's products use
another summation order and one FMA in the update, so after k steps the iterates differ by rounding of order
k * 2^-53 * |x| (the iteration is a contraction in the cases below: differences are not amplified).  Compared:
the iterate after a FIXED number of steps (tolerance 1e-12 * max|x|, derived from k <= 200 steps of <= 9-term
rows), the closed form on Laplacian eigenvectors, the stop rule (test before update: iteration counts equal the
oracle's up to one step when the residual crosses the threshold within rounding), the reported residual against the
recomputed one, bit-identical repeats and graph replay equal to plain launches."""
import numpy as np
import pytest

import oracle
from paper_1309_1894_b200 import binding
from paper_1309_1894_b200 import workloads as W
from tests import helpers as H

pytestmark = pytest.mark.gpu


def _true_rel_res(A, x, b):
    Ax, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x, 0.0)
    return np.linalg.norm(b - Ax) / np.linalg.norm(b)


@pytest.mark.parametrize("desc", ["default", "dia_const:b256:r2:x0", "dia_tma:b288:c256:r1:u7:i3:x0",
                                  "sell_tma:b288:c256:s1:r1:u8:i3:x0", "merge:b256:i7:x0", "csr_vector:b256:w8:u2:x0"])
def test_jacobi_fixed_step_count_matches_the_oracle(cuda, desc):
    import torch
    A = W.laplace3d_7pt(21)                                   # 9261 rows (odd): ragged last block
    xt = W.uniform(121, A.rows)
    b, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, xt, 0.0)
    x0 = W.uniform(122, A.rows)
    S = binding.SpMV.from_csr(A)
    S.select(desc)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        db = H.to_dev(b)
        for k, omega in ((1, 1.0), (2, 0.8), (7, 2.0 / 3.0), (50, 1.0), (131, 0.9)):
            x_ref, k_ref, rel_ref, hist = oracle.jacobi(A.row_ptr, A.col_idx, A.val, b, x0=x0, omega=omega, tol=1e-300, max_iters=k)
            dx = H.to_dev(x0).clone()
            res = S.jacobi(db, dx, omega=omega, tol=1e-300, max_iters=k, check_every=6)
            stream.synchronize()
            x = dx.cpu().numpy()
            assert res["iters"] == k == k_ref and res["converged"] == 0 and res["zero_diagonal"] == 0
            assert res["kernels_per_iteration"] == (3 if desc.startswith("merge") else 2)
            assert np.abs(x - x_ref).max() <= 1e-12 * np.abs(x_ref).max(), (desc, k)
            assert res["rel_residual"] == pytest.approx(rel_ref, rel=1e-11)
            assert res["rel_residual"] == pytest.approx(_true_rel_res(A, x, b), rel=1e-11)   # residual OF the returned x
            # bit-identical repeat; plain launches equal graph replay bit for bit
            dx2, dx3 = H.to_dev(x0).clone(), H.to_dev(x0).clone()
            res2 = S.jacobi(db, dx2, omega=omega, tol=1e-300, max_iters=k, check_every=6)
            res3 = S.jacobi(db, dx3, omega=omega, tol=1e-300, max_iters=k, no_graph=True)
            stream.synchronize()
            assert torch.equal(dx, dx2) and torch.equal(dx, dx3)
            assert res3["graph_replays"] == 0 and (k <= 2 or res2["graph_replays"] >= 1)
            # constant-coefficient stencil: the step runs inside the product kernel; the iterates are the same bits
            # as with the separate pass (the update is element-wise; only the shape of the norm's sum differs)
            assert res["fused_step"] == (1 if desc.startswith("dia_const") else 0)
            if desc.startswith("dia_const"):
                dx4 = H.to_dev(x0).clone()
                res4 = S.jacobi(db, dx4, omega=omega, tol=1e-300, max_iters=k, check_every=6, no_fused=True)
                stream.synchronize()
                assert res4["fused_step"] == 0 and res4["iters"] == k and torch.equal(dx, dx4)
                assert res4["rel_residual"] == pytest.approx(res["rel_residual"], rel=1e-12)
    S.close()


def test_jacobi_closed_form_on_a_laplacian_eigenvector(cuda):
    """b = lambda v, x0 = 0: x_k = (1 - rho^k) v, ||r_k|| / ||b|| = |rho|^k, rho = 1 - omega lambda / 4 (2D, 5-point)."""
    import torch
    n, m, omega = 40, (3, 5), 0.8
    A = W.laplace2d_5pt(n)
    i = np.arange(1, n + 1)
    v = np.kron(np.sin(m[1] * np.pi * i / (n + 1)), np.sin(m[0] * np.pi * i / (n + 1)))
    lam = 4.0 - 2.0 * np.cos(m[0] * np.pi / (n + 1)) - 2.0 * np.cos(m[1] * np.pi / (n + 1))
    rho = 1.0 - omega * lam / 4.0
    S = binding.SpMV.from_csr(A)
    S.select("dia_const:b256:r1:x0")
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        db = H.to_dev(lam * v)
        for k in (1, 4, 33):
            dx = torch.zeros(A.rows, dtype=torch.float64, device="cuda")
            res = S.jacobi(db, dx, omega=omega, tol=1e-300, max_iters=k)
            stream.synchronize()
            assert res["iters"] == k
            assert np.abs(dx.cpu().numpy() - (1.0 - rho ** k) * v).max() <= 1e-13
            assert res["rel_residual"] == pytest.approx(abs(rho) ** k, rel=1e-11)
    S.close()


def test_jacobi_fused_step_on_the_27_point_stencil_and_a_2d_grid(cuda):
    """The fused step for other diagonal counts (27-point: the generic-count instantiation of the mask type; 5-point:
    exact-ND), ragged sizes, stop rule included: against the oracle and bit-identical to the unfused path."""
    import torch
    stream = torch.cuda.Stream()
    for A, desc in ((W.stencil3d_27pt(13), "dia_const:b128:r1:x0"), (W.laplace2d_5pt(77), "dia_const:b512:r2:x0"),
                    (W.laplace3d_7pt(30), "dia_const:b256:r4:x0")):
        xt = W.uniform(128, A.rows)
        b, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, xt, 0.0)
        S = binding.SpMV.from_csr(A)
        S.select(desc)
        with torch.cuda.stream(stream):
            db = H.to_dev(b)
            for tol, max_iters in ((1e-300, 37), (1e-3, 5000)):
                x_ref, k_ref, rel_ref, _ = oracle.jacobi(A.row_ptr, A.col_idx, A.val, b, omega=0.9, tol=tol, max_iters=max_iters)
                dx = torch.zeros(A.rows, dtype=torch.float64, device="cuda")
                res = S.jacobi(db, dx, omega=0.9, tol=tol, max_iters=max_iters)
                dx2 = torch.zeros_like(dx)
                res2 = S.jacobi(db, dx2, omega=0.9, tol=tol, max_iters=max_iters, no_fused=True)
                stream.synchronize()
                assert res["fused_step"] == 1 and res2["fused_step"] == 0 and res["kernels_per_iteration"] == 2
                assert abs(res["iters"] - k_ref) <= 1 and res["iters"] == res2["iters"], (desc, res, k_ref)
                assert torch.equal(dx, dx2)
                if res["iters"] == k_ref:
                    assert np.abs(dx.cpu().numpy() - x_ref).max() <= 1e-12 * np.abs(x_ref).max()
                    assert res["rel_residual"] == pytest.approx(rel_ref, rel=1e-10)
                assert res["converged"] == (1 if tol > 1e-100 else 0)
        S.close()


def test_jacobi_converges_like_the_oracle_on_a_dominant_nonsymmetric_matrix(cuda):
    """Stop rule: both sides stop at the first k with ||r_k|| <= tol ||b||; the limit is the dense solution."""
    import torch
    rng = np.random.default_rng(5)
    n = 3001
    A0 = W.csr_from_lengths(rng.integers(1, 12, n), n, 123)
    # make it strictly diagonally dominant with a varying diagonal of both signs: append (i, i) to every row
    rows = np.repeat(np.arange(n), np.diff(A0.row_ptr))
    off = A0.col_idx != rows
    absrow = np.bincount(rows[off], weights=np.abs(A0.val[off]), minlength=n)
    diag = (1.5 * absrow + 1.0) * np.where(np.arange(n) % 3 == 0, -1.0, 1.0)
    r2 = np.concatenate([rows[off], np.arange(n)]); c2 = np.concatenate([A0.col_idx[off], np.arange(n)])
    v2 = np.concatenate([A0.val[off], diag])
    order = np.lexsort((c2, r2))
    rp = np.zeros(n + 1, dtype=np.int32); np.add.at(rp, r2 + 1, 1); rp = np.cumsum(rp).astype(np.int32)
    A = W.CSR(n, n, rp, c2[order].astype(np.int32), v2[order])
    b = W.uniform(124, n)
    tol = 1e-12
    x_ref, k_ref, rel_ref, _ = oracle.jacobi(A.row_ptr, A.col_idx, A.val, b, omega=1.0, tol=tol, max_iters=2000)
    assert 0 < k_ref < 2000
    S = binding.SpMV.from_csr(A)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        db = H.to_dev(b)
        for desc in ("default", "csr_vector:b256:w4:u2:x0", "sell:b256:c128:s1:r2:u4:x0"):
            S.select(desc)
            dx = torch.zeros(n, dtype=torch.float64, device="cuda")
            res = S.jacobi(db, dx, omega=1.0, tol=tol, max_iters=2000, check_every=4)
            stream.synchronize()
            x = dx.cpu().numpy()
            assert res["converged"] == 1 and abs(res["iters"] - k_ref) <= 1, (res, k_ref)
            assert res["rel_residual"] <= tol and _true_rel_res(A, x, b) <= 2 * tol
            assert np.abs(x - x_ref).max() <= 10 * tol * np.abs(x_ref).max()
            assert res["iterations_launched"] >= res["iters"] + 1
    S.close()


def test_jacobi_edge_cases(cuda):
    import torch
    A = W.laplace2d_5pt(9)
    b = W.uniform(125, A.rows)
    x0 = W.uniform(126, A.rows)
    S = binding.SpMV.from_csr(A)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        db = H.to_dev(b)
        # zero iterations: x0 returned, its residual reported
        dx = H.to_dev(x0).clone()
        res = S.jacobi(db, dx, max_iters=0)
        stream.synchronize()
        assert res["iters"] == 0 and np.array_equal(dx.cpu().numpy(), x0)
        assert res["rel_residual"] == pytest.approx(_true_rel_res(A, x0, b), rel=1e-12)
        # starting at the solution: the stop rule fires before any update
        xs, _, _, _ = oracle.jacobi(A.row_ptr, A.col_idx, A.val, b, tol=1e-15, max_iters=20000)
        dx = H.to_dev(xs).clone()
        res = S.jacobi(db, dx, tol=1e-10)
        stream.synchronize()
        assert res["iters"] == 0 and res["converged"] == 1 and np.array_equal(dx.cpu().numpy(), xs)
        # b = 0: nothing to do
        dz = torch.zeros(A.rows, dtype=torch.float64, device="cuda")
        res = S.jacobi(torch.zeros_like(dz), dz)
        stream.synchronize()
        assert res["iters"] == 0 and res["converged"] == 1 and res["rel_residual"] == 0.0 and not dz.any()
    S.close()
    # a row without a diagonal entry: refused through the result, x untouched; duplicates on the diagonal sum
    rp = np.array([0, 3, 5], dtype=np.int32)
    ci = np.array([0, 1, 0, 0, 1], dtype=np.int32)
    va = np.array([1.5, 0.5, 2.5, -0.25, 2.0])
    Sd = binding.SpMV.from_csr(W.CSR(2, 2, rp, ci, va))
    with torch.cuda.stream(stream):
        dx = torch.zeros(2, dtype=torch.float64, device="cuda")
        res = Sd.jacobi(H.to_dev(np.array([1.0, -2.0])), dx, tol=1e-300, max_iters=1)
        stream.synchronize()
        assert res["iters"] == 1 and np.array_equal(dx.cpu().numpy(), np.array([0.25, -1.0]))      # b / d with d_0 = 1.5 + 2.5
    Sd.close()
    Sz = binding.SpMV.from_csr(W.CSR(2, 2, np.array([0, 1, 2], np.int32), np.array([1, 1], np.int32), np.array([1.0, 1.0])))
    with torch.cuda.stream(stream):
        dx = H.to_dev(np.array([3.0, 4.0])).clone()
        res = Sz.jacobi(H.to_dev(np.array([1.0, -2.0])), dx)
        stream.synchronize()
        assert res["zero_diagonal"] == 1 and res["iters"] == 0 and np.array_equal(dx.cpu().numpy(), np.array([3.0, 4.0]))
    Sz.close()
    Sr = binding.SpMV.from_csr(W.csr_from_lengths([2, 2, 2], 5, 127))                        # not square
    with pytest.raises(binding.SpmvError) as e:
        Sr.jacobi(torch.zeros(3, dtype=torch.float64, device="cuda"), torch.zeros(3, dtype=torch.float64, device="cuda"))
    assert e.value.status == 1
    Sr.close()

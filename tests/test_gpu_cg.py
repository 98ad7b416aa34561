"""GPU tests of spmv_cg (solver loop around apply) against the plain CG
oracle (oracle/oracle_cg.c).  CG is an iteration: the GPU's dot products use another summation order,
so the iterates drift apart by rounding amplified over the iterations.  What is unique is compared
(the solution of the SPD system, to a tolerance derived from the stopping rule: both sides stop at
||r|| <= tol*||b||, so ||x_gpu - x_ref|| <= 2*tol*cond(A)*||x||), and the rest is checked for
validity: the reported residual is the true residual, iteration counts agree within a few steps,
repeated runs are bit-identical, graph replay equals plain launches bit for bit."""
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
def test_cg_solves_the_laplacian_like_the_oracle(cuda, desc):
    import torch
    A = W.laplace3d_7pt(24)                                   # cond ~ 250
    xt = W.uniform(101, A.rows)
    b, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, xt, 0.0)
    tol = 1e-10
    x_ref, k_ref, rel_ref, _ = oracle.cg(A.row_ptr, A.col_idx, A.val, b, tol=tol, max_iters=500)
    S = binding.SpMV.from_csr(A)
    S.select(desc)
    stream = torch.cuda.Stream()                              # a capturable stream: the graph path
    with torch.cuda.stream(stream):
        db = H.to_dev(b)
        dx = torch.zeros(A.rows, dtype=torch.float64, device="cuda")
        res = S.cg(db, dx, tol=tol, max_iters=500, no_fused=True)      # the multi-kernel path (any size)
        stream.synchronize()
        x = dx.cpu().numpy()
        assert res["converged"] == 1 and res["breakdown"] == 0 and res["graph_replays"] >= 1 and res["fused"] == 0
        # p.q comes out of the SpMV epilogue for dia_const (no second pass over p and q), from a dot kernel otherwise
        assert res["fused_dot"] == (1 if desc.startswith("dia_const") else 0)
        assert res["kernels_per_iteration"] == (5 if desc.startswith("merge") else 4)
        assert abs(res["iters"] - k_ref) <= 3, (res, k_ref)
        assert res["rel_residual"] <= tol
        assert _true_rel_res(A, x, b) <= 2 * tol              # recurrence residual ~ true residual
        assert np.abs(x - x_ref).max() <= 2 * tol * 250 * np.abs(x_ref).max()
        assert np.abs(x - xt).max() <= 1e-6
        # bit-identical repeat; plain launches equal graph replay bit for bit
        dx2 = torch.zeros_like(dx)
        res2 = S.cg(db, dx2, tol=tol, max_iters=500, no_fused=True)
        dx3 = torch.zeros_like(dx)
        res3 = S.cg(db, dx3, tol=tol, max_iters=500, no_graph=True, no_fused=True)
        stream.synchronize()
        assert torch.equal(dx, dx2) and torch.equal(dx, dx3)
        assert res2["iters"] == res["iters"] == res3["iters"] and res3["graph_replays"] == 0
    S.close()


def test_cg_edge_cases(cuda):
    import torch
    A = W.laplace2d_5pt(30)
    b = W.uniform(102, A.rows)
    x0 = W.uniform(103, A.rows)
    S = binding.SpMV.from_csr(A)
    db, dx = H.to_dev(b), H.to_dev(x0).clone()
    # zero iterations: x untouched, residual of the initial guess
    res = S.cg(db, dx, tol=1e-12, max_iters=0)
    assert res["iters"] == 0 and res["converged"] == 0 and np.array_equal(dx.cpu().numpy(), x0)
    assert res["rel_residual"] == pytest.approx(_true_rel_res(A, x0, b), rel=1e-12)
    # iteration cap on the legacy default stream (no graph possible): stops at exactly max_iters
    res = S.cg(db, dx, tol=1e-14, max_iters=5, check_every=3)
    x5, k5, rel5, _ = oracle.cg(A.row_ptr, A.col_idx, A.val, b, x0=x0, tol=1e-14, max_iters=5)
    assert res["iters"] == 5 and res["converged"] == 0 and res["graph_replays"] == 0
    assert res["rel_residual"] == pytest.approx(rel5, rel=1e-9)
    assert np.abs(dx.cpu().numpy() - x5).max() <= 1e-12 * np.abs(x5).max()
    # starting at the solution: converged without an iteration
    xs, _, _, _ = oracle.cg(A.row_ptr, A.col_idx, A.val, b, tol=1e-13, max_iters=2000)
    dxs = H.to_dev(xs).clone()
    res = S.cg(db, dxs, tol=1e-9, max_iters=100)
    assert res["iters"] == 0 and res["converged"] == 1 and np.array_equal(dxs.cpu().numpy(), xs)
    S.close()
    # negative definite matrix: p.Ap <= 0 -> breakdown reported, no NaN written
    N = W.CSR(A.rows, A.cols, A.row_ptr, A.col_idx, -A.val)
    T = binding.SpMV.from_csr(N)
    dx = torch.zeros(A.rows, dtype=torch.float64, device="cuda")
    res = T.cg(db, dx, tol=1e-10, max_iters=50)
    assert res["breakdown"] == 1 and res["converged"] == 0 and res["iters"] == 0
    assert bool(torch.isfinite(dx).all())
    T.close()
    # rectangular: refused
    R = binding.SpMV.from_csr(W.csr_from_lengths([2, 3, 1], 7, 104))
    with pytest.raises(binding.SpmvError) as e:
        R.cg(torch.zeros(3, dtype=torch.float64, device="cuda"), torch.zeros(3, dtype=torch.float64, device="cuda"))
    assert e.value.status == 1
    R.close()


def test_cg_after_tune_on_cfg1(cuda):
    """BASELINE.json:configs[0] (2D 5-pt 64^2): tune, then solve with the winner."""
    import torch
    prob = W.config(1)
    A = prob.A
    S = binding.SpMV.from_csr(A)
    S.tune(use_cache=2, reps=1, min_batch_ms=0.02)
    b, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, prob.x, 0.0)
    with torch.cuda.stream(torch.cuda.Stream()):
        dx = torch.zeros(A.rows, dtype=torch.float64, device="cuda")
        res = S.cg(H.to_dev(b), dx, tol=1e-11, max_iters=1000)
        torch.cuda.current_stream().synchronize()
        x = dx.cpu().numpy()
    x_ref, k_ref, _, _ = oracle.cg(A.row_ptr, A.col_idx, A.val, b, tol=1e-11, max_iters=1000)
    assert res["converged"] == 1 and abs(res["iters"] - k_ref) <= 5
    assert np.abs(x - prob.x).max() <= 1e-7 and _true_rel_res(A, x, b) <= 2e-11
    S.close()


def test_cg_fused_single_kernel_for_small_systems(cuda):
    """rows <= 262144: the whole solve runs in one cooperative kernel (3 grid barriers per iteration,
    no launches).  Same recurrence and stop rule as the multi-kernel path and the oracle."""
    import torch
    for A, cond in ((W.laplace2d_5pt(64), 1800.0), (W.laplace3d_7pt(40), 700.0)):
        xt = W.uniform(121, A.rows)
        b, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, xt, 0.0)
        tol = 1e-10
        x_ref, k_ref, _, _ = oracle.cg(A.row_ptr, A.col_idx, A.val, b, tol=tol, max_iters=2000)
        S = binding.SpMV.from_csr(A)
        db = H.to_dev(b)
        dx = torch.zeros(A.rows, dtype=torch.float64, device="cuda")
        res = S.cg(db, dx, tol=tol, max_iters=2000)
        x = dx.cpu().numpy()
        assert res["fused"] == 1 and res["converged"] == 1 and res["graph_replays"] == 0
        assert abs(res["iters"] - k_ref) <= 5 and res["rel_residual"] <= tol
        assert _true_rel_res(A, x, b) <= 2 * tol
        assert np.abs(x - x_ref).max() <= 2 * tol * cond * np.abs(x_ref).max()
        dx2 = torch.zeros_like(dx)
        res2 = S.cg(db, dx2, tol=tol, max_iters=2000)
        assert torch.equal(dx, dx2) and res2["iters"] == res["iters"]          # deterministic
        dx3 = torch.zeros_like(dx)
        res3 = S.cg(db, dx3, tol=tol, max_iters=2000, no_fused=True)           # multi-kernel path agrees
        assert res3["fused"] == 0 and abs(res3["iters"] - res["iters"]) <= 5
        assert np.abs(dx3.cpu().numpy() - x).max() <= 2 * tol * cond * np.abs(x).max()
        S.close()


def test_cg_fused_dot_equals_separate_dot_and_loop_tuning(cuda):
    """(i) the dot product fused into the dia_const kernel gives a valid CG run next to the
    separate dot kernel (another summation shape: compared through the solution, not bitwise); (ii) tune_loop
    times the leaders of spmv_tune inside the iteration and adopts one of them; the solve is still right."""
    import torch
    A = W.laplace3d_7pt(72)                                   # 373 248 rows: above the single-kernel limit
    xt = W.uniform(131, A.rows)
    b, _ = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, xt, 0.0)
    tol = 1e-9
    S = binding.SpMV.from_csr(A)
    rep = S.tune(alpha=1.0, beta=0.0, use_cache=2, reps=2, min_batch_ms=0.1, search=1)
    with torch.cuda.stream(torch.cuda.Stream()):
        db = H.to_dev(b)
        S.select("dia_const:b256:r1:x0")
        out = {}
        for key, kw in (("fused", {}), ("separate", {"no_fused_dot": True})):
            dx = torch.zeros(A.rows, dtype=torch.float64, device="cuda")
            res = S.cg(db, dx, tol=tol, max_iters=2000, **kw)
            torch.cuda.current_stream().synchronize()
            out[key] = (res, dx.cpu().numpy())
            assert res["converged"] == 1 and res["fused"] == 0
            assert _true_rel_res(A, out[key][1], b) <= 2 * tol
        assert out["fused"][0]["fused_dot"] == 1 and out["fused"][0]["kernels_per_iteration"] == 4
        assert out["separate"][0]["fused_dot"] == 0 and out["separate"][0]["kernels_per_iteration"] == 4
        assert abs(out["fused"][0]["iters"] - out["separate"][0]["iters"]) <= 3
        assert np.abs(out["fused"][1] - out["separate"][1]).max() <= 2 * tol * 2200 * np.abs(xt).max()
        # repeat of the fused form: bit-identical (fixed reduction shape, last-block sums in index order)
        dx2 = torch.zeros(A.rows, dtype=torch.float64, device="cuda")
        res2 = S.cg(db, dx2, tol=tol, max_iters=2000)
        torch.cuda.current_stream().synchronize()
        assert np.array_equal(dx2.cpu().numpy(), out["fused"][1]) and res2["iters"] == out["fused"][0]["iters"]
    # tune for the loop: needs the leaders of a tune in this process
    T = binding.SpMV.from_csr(A)
    rep = T.tune(alpha=1.0, beta=0.0, use_cache=2, reps=2, min_batch_ms=0.1, search=1)
    with torch.cuda.stream(torch.cuda.Stream()):
        dx = torch.zeros(A.rows, dtype=torch.float64, device="cuda")
        res = T.cg(H.to_dev(b), dx, tol=tol, max_iters=2000, tune_loop=True)
        torch.cuda.current_stream().synchronize()
        assert res["converged"] == 1 and res["loop_variant"] == T.variant and len(res["loop_variant"]) > 0
        assert _true_rel_res(A, dx.cpu().numpy(), b) <= 2 * tol
    S.close(); T.close()

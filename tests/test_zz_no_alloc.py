"""spmv_merge_apply_noalloc against the handle path (collected last: `pytest -x` stops at the first failure, so a
failure here must not hide the other GPU tests).

Who needs the entry point: code that has to form y = alpha*A*x + beta*y at a place where it may not allocate device
memory -- it runs inside an application whose own pool already holds the whole GPU (cudaMalloc fails there), or in a
loop that cannot take the device-wide stall of cudaMalloc / cudaFree.  The entry point therefore keeps the
merge-path kernels' scratch (tile table, tile carries) in one fixed array inside the library instead of in buffers
owned by a handle.  That array is shared by every call and keeps the previous call's contents, which is what these
tests lean on: two calls in a row, the second on a DIFFERENT, smaller matrix (stale entries of the first call lie
behind the ones it uses), then the first matrix again.

The reference is the existing path: spmv_create + spmv_select("merge:b256:i7:x0") + spmv_apply on the same device
arrays, whose result the other test files pin to the CPU oracle.  Tolerance: the one all parity tests use (helpers.TOL
= 1e-12 relative to the oracle's per-row scale_i); the two paths run the same kernels with the same tiling, so the
tests also ask for equal bits.  Works alone in a fresh process (the first call then does the per-device set-up) and
after the other tests."""
import ctypes

import numpy as np
import pytest

import oracle
from paper_1309_1894_b200 import binding, workloads as W
from tests.helpers import TOL, to_dev

pytestmark = pytest.mark.gpu

VARIANT = "merge:b256:i7:x0"


def _device_csr(A):
    return to_dev(A.row_ptr), to_dev(A.col_idx), to_dev(A.val)


def _handle_path(A, d_csr, alpha, dx, beta, y0):
    """The existing path on the same device arrays."""
    import torch
    S = binding.SpMV(A.rows, A.cols, *d_csr)
    S.select(VARIANT)
    dy = to_dev(y0).clone()
    S.apply(alpha, dx, beta, dy)
    torch.cuda.synchronize()
    y = dy.cpu().numpy()
    S.close()
    return y


def _noalloc_path(A, d_csr, alpha, dx, beta, y0):
    import torch
    dy = to_dev(y0).clone()
    binding.merge_apply_noalloc(A.rows, A.cols, *d_csr, alpha, dx, beta, dy)
    torch.cuda.synchronize()
    return dy.cpu().numpy()


def _compare(A, alpha, beta, seed, what):
    rng = np.random.default_rng(seed)
    x = rng.uniform(-1, 1, A.cols)
    y0 = rng.uniform(-1, 1, A.rows)
    d_csr = _device_csr(A)
    dx = to_dev(x)
    y_new = _noalloc_path(A, d_csr, alpha, dx, beta, y0)
    y_old = _handle_path(A, d_csr, alpha, dx, beta, y0)
    # the tests' tolerance rule: |y - y_ref| <= TOL * scale_i, scale_i from the oracle
    _, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, alpha, x, beta, y0)
    ok, mr, ff, nf = oracle.accept(y_new, y_old, scale, TOL)
    assert ok, f"{what}: {nf} rows differ from the handle path, first {ff}, max err/scale {mr:.3e}"
    assert np.array_equal(y_new.view(np.uint64), y_old.view(np.uint64)), f"{what}: same kernels, same tiling, other bits"
    return y_new


def test_two_calls_in_a_row_match_the_handle_path(cuda):
    big = W.powerlaw(60000, lmax=5000)          # skewed rows, some 550 tiles, rows cut by tile boundaries
    small = W.csr_from_lengths([0, 0, 3, 0, 2500, 1, 0, 7, 1800, 0, 0], 4000, 21)   # 3 tiles, empty rows, long rows
    y1 = _compare(big, 1.0, 0.5, 1, "first call (big)")
    _compare(small, -0.75, 0.0, 2, "second call (small, stale scratch behind it)")
    y3 = _compare(big, 1.0, 0.5, 1, "third call (big again)")
    assert np.array_equal(y1.view(np.uint64), y3.view(np.uint64))      # repeatable bit for bit


def test_back_to_back_without_sync_and_against_the_oracle(cuda):
    """Two calls enqueued on one stream with nothing in between (the documented use), each checked against oracle/."""
    import torch
    A = W.powerlaw(20000, lmax=3000)
    B = W.laplace3d_7pt(23)
    rng = np.random.default_rng(5)
    xa, ya = rng.uniform(-1, 1, A.cols), rng.uniform(-1, 1, A.rows)
    xb, yb = rng.uniform(-1, 1, B.cols), rng.uniform(-1, 1, B.rows)
    da, db = _device_csr(A), _device_csr(B)
    dxa, dya, dxb, dyb = to_dev(xa), to_dev(ya).clone(), to_dev(xb), to_dev(yb).clone()
    binding.merge_apply_noalloc(A.rows, A.cols, *da, 2.0, dxa, -1.0, dya)
    binding.merge_apply_noalloc(B.rows, B.cols, *db, 1.0, dxb, 0.5, dyb)
    torch.cuda.synchronize()
    for M, al, x, be, y0, dy in ((A, 2.0, xa, -1.0, ya, dya), (B, 1.0, xb, 0.5, yb, dyb)):
        y_ref, scale = oracle.spmv(M.row_ptr, M.col_idx, M.val, al, x, be, y0)
        ok, mr, ff, nf = oracle.accept(dy.cpu().numpy(), y_ref, scale, TOL)
        assert ok, f"{nf} rows fail vs the oracle, first {ff}, max err/scale {mr:.3e}"


def test_no_device_allocation_and_edge_cases(cuda):
    import torch
    A = W.powerlaw(5000, lmax=600)
    d_csr = _device_csr(A)
    dx = to_dev(np.random.default_rng(3).uniform(-1, 1, A.cols))
    dy = torch.zeros(A.rows, dtype=torch.float64, device="cuda:0")
    binding.merge_apply_noalloc(A.rows, A.cols, *d_csr, 1.0, dx, 0.0, dy)      # set-up call for this device
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(20):
        binding.merge_apply_noalloc(A.rows, A.cols, *d_csr, 1.0, dx, 0.0, dy)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, "the device's free memory moved across 20 calls"
    # beta == 0 never reads y (NaN in), alpha == 0 never reads A or x
    dy.fill_(float("nan"))
    binding.merge_apply_noalloc(A.rows, A.cols, *d_csr, 1.0, dx, 0.0, dy)
    assert torch.isfinite(dy).all()
    keep = dy.clone()
    binding.merge_apply_noalloc(A.rows, A.cols, *d_csr, 0.0, dx.fill_(float("nan")), 2.0, dy)
    assert torch.equal(dy, 2.0 * keep)
    # nnz == 0 and rows == 0
    E = W.csr_from_lengths([0] * 37, 11, 4)
    de = _device_csr(E)
    dye = torch.full((37,), 3.0, dtype=torch.float64, device="cuda:0")
    binding.merge_apply_noalloc(37, 11, *de, 1.0, dx, 0.5, dye)
    assert torch.equal(dye, torch.full_like(dye, 1.5))
    L = binding.lib()
    assert L.spmv_merge_apply_noalloc(0, 0, 0, None, None, None, 1.0, None, 0.0, None, None) == 0


def test_over_the_limit_is_refused_with_a_message(cuda):
    L = binding.lib()
    cap = binding.merge_noalloc_max_path()
    assert cap == 65536 * 1792
    p = ctypes.c_void_p(256)             # never dereferenced: the size check comes before any launch
    rows = 1 << 20
    st = L.spmv_merge_apply_noalloc(rows, rows, cap - rows + 1, p, p, p, 1.0, p, 0.0, ctypes.c_void_p(512), None)
    assert st == 3                       # SPMV_ERR_UNSUPPORTED
    msg = L.spmv_last_error().decode()
    assert "over the limit" in msg and str(cap) in msg
    assert L.spmv_merge_apply_noalloc(-1, 1, 0, p, p, p, 1.0, p, 0.0, p, None) == 1
    assert L.spmv_merge_apply_noalloc(4, 4, 4, p, p, p, 1.0, p, 0.0, p, None) == 1      # d_x == d_y

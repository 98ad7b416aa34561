"""Shared helpers for the GPU parity tests: run the CUDA library through its binding and
compare with oracle/ (the acceptance rule of SURVEY.md sec. 8(c), tolerance 1e-12 relative to
scale_i = |alpha| sum_j |a_ij x_j| + |beta y_i| -- BASELINE.json:north_star)."""
import numpy as np

import oracle
from paper_1309_1894_b200 import workloads as W

TOL = 1e-12


def to_dev(a, device="cuda:0"):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).to(device)


def gpu_apply(S, alpha, x, beta, y0):
    """One spmv_apply from y0 (None: NaN-filled, must be overwritten); returns numpy y."""
    import torch
    dx = to_dev(x)
    if y0 is None:
        dy = torch.full((S.rows,), float("nan"), dtype=torch.float64, device=dx.device)
    else:
        dy = to_dev(y0).clone()
    S.apply(alpha, dx, beta, dy)
    torch.cuda.synchronize()
    return dy.cpu().numpy()


def check_against_oracle(S, A, alpha, x, beta, y0, tol=TOL, what=""):
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, alpha, x, beta, y0)
    y = gpu_apply(S, alpha, x, beta, y0)
    ok, mr, ff, nf = oracle.accept(y, y_ref, scale, tol)
    assert ok, f"{what} {S.variant}: {nf} rows fail, first {ff}, max err/scale {mr:.3e}, y={y[ff]!r} ref={y_ref[ff]!r}"
    return y, y_ref, mr


# one representative per kernel family x template axis; eligibility is checked per matrix
REPRESENTATIVE_VARIANTS = [
    "default",
    "csr_scalar:b128:r2:u2:x0", "csr_scalar:b256:r4:u2:x1", "csr_scalar:b512:r1:u4:x0:g2",
    "csr_vector:b256:w2:u1:x0", "csr_vector:b128:w4:u2:x1", "csr_vector:b256:w8:u4:x0",
    "csr_vector:b512:w16:u2:x0:g1", "csr_vector:b256:w32:u4:x0:co50",
    "sell:b256:c128:s1:r1:u1:x0", "sell:b128:c128:s1:r2:u4:x0", "sell:b256:c512:s1:r4:u2:x1",
    "sell:b256:c128:s8192:r2:u2:x0", "sell:b512:c512:s512:r4:u4:x0:g2", "sell:b256:c128:s1024:r1:u8:x0",
    "ell:b256:r1:u2:x0", "ell:b128:r2:u8:x0", "ell:b256:r4:u4:x1",
    "sell_tma:b288:c256:s1:r1:u8:i3:x0", "sell_tma:b160:c256:s1:r2:u4:i4:x0", "sell_tma:b160:c128:s1024:r1:u16:i2:x0",
    "sell_tma:b288:c512:s8192:r2:u8:i2:x0:g2", "sell_tma:b544:c512:s1:r1:u4:i6:x0",
    # x window staged in shared memory (a10 ii)
    "sell_tma:b288:c256:s1:r1:u8:i3:x2:h136", "sell_tma:b160:c256:s1:r2:u4:i3:x2:h72", "sell_tma:b160:c128:s1:r1:u16:i2:x2:h8",
    "sell_tma:b288:c512:s1024:r2:u8:i2:x2:h136", "sell_tma:b160:c128:s8192:l32:r1:u4:i3:x2:h72",
    # x3: the window covers the whole band -- every gather is a shared-memory read (eligible when h >= bandwidth)
    "sell_tma:b288:c256:s1:r1:u8:i3:x3:h904", "sell_tma:b160:c128:s1:r1:u4:i6:x3:h4096",
    "sell16_tma:b160:c128:s1:r1:u8:i4:x3:h1000", "sell16_tma:b288:c512:s1:r2:u4:i4:x3:h904",
    # long rows cut into segments of l entries (virtual rows) + ordered fix-up
    "sell:b256:c128:s8192:l16:r2:u2:x0", "sell:b128:c512:s1024:l64:r1:u4:x0", "sell:b256:c128:s256:l4:r1:u2:x1",
    "sell_tma:b160:c128:s8192:l32:r1:u4:i3:x0", "sell_tma:b160:c256:s2048:l128:r2:u8:i2:x0",
    # 16-bit delta-encoded column indices (banded patterns only)
    "sell16:b256:c128:s1:r1:u2:x0", "sell16:b128:c128:s1:r2:u4:x0", "sell16:b256:c512:s512:r4:u2:x1", "sell16:b256:c128:s8192:r2:u8:x0:g2",
    "sell16_tma:b288:c256:s1:r1:u8:i3:x0", "sell16_tma:b160:c256:s1:r2:u4:i4:x0", "sell16_tma:b160:c128:s1024:r1:u16:i2:x0",
    "dia:b256:c128:r1:u4:x0", "dia:b128:c256:r2:u8:x0", "dia:b256:c512:r4:u2:x1", "dia:b512:c128:r1:u1:x0:g2",
    "dia_const:b256:r1:x0", "dia_const:b128:r2:x1", "dia_const:b512:r4:x0",
    "dia_win:b288:c256:r1:i2:x0", "dia_win:b96:c128:r2:i3:x0", "dia_win:b160:c128:r1:i4:x0:g2",
    "dia_cwin:b288:c256:r1:i3:x0", "dia_cwin:b288:c512:r2:i2:x0", "dia_cwin:b544:c512:r1:i4:x0",
    "dia_tma:b288:c256:r1:u8:i3:x0", "dia_tma:b96:c128:r2:u4:i2:x0", "dia_tma:b544:c512:r1:u7:i4:x0", "dia_tma:b160:c256:r2:u9:i2:x0:g2",
    "merge:b128:i5:x0", "merge:b256:i7:x0", "merge:b256:i11:x1", "merge:b512:i7:x0", "merge:b128:i11:x0",
    "bcsr3:b256:w4:u1:x0", "bcsr3:b128:w8:u2:x0", "bcsr3:b256:w16:u1:x1", "bcsr3:b256:w32:u2:x0:g1", "bcsr3:b512:w16:u2:x3:g1", "bcsr3:b128:w8:u1:x3",
    # 16-bit block columns
    "bcsr3:b128:w8:u2:i16:x0", "bcsr3:b256:w16:u1:i16:x3:g1", "bcsr3:b256:w4:u2:i16:x1",
]


def zoo():
    """Test zoo of SURVEY.md sec. 4 T3: (name, CSR)."""
    out = []
    out.append(("1x1", W.csr_from_lengths([1], 1, 1)))
    out.append(("1xN_dense_row", W.csr_from_lengths([3000], 3000, 2)))
    out.append(("Nx1", W.csr_from_lengths([1, 0, 1, 1, 0, 1, 1], 1, 3)))
    out.append(("nnz0", W.csr_from_lengths([0] * 37, 11, 4)))
    out.append(("empty_rows_runs", W.csr_from_lengths([0, 0, 0, 5, 0, 7, 0, 0, 0, 0, 3, 1, 0, 0], 50, 5)))
    out.append(("lengths_ladder", W.csr_from_lengths(
        [1, 2, 3, 31, 32, 33, 63, 64, 65, 1023, 1025, 20000, 0, 7, 129, 255, 257], 40000, 6)))
    out.append(("identity", W.CSR(300, 300, np.arange(301, dtype=np.int32), np.arange(300, dtype=np.int32), np.ones(300))))
    out.append(("rect_wide", W.csr_from_lengths(np.random.default_rng(7).integers(0, 40, 500), 7000, 7)))
    out.append(("rect_tall", W.csr_from_lengths(np.random.default_rng(8).integers(0, 9, 3001), 10, 8)))
    out.append(("unsorted", W.csr_from_lengths(np.random.default_rng(9).integers(0, 60, 700), 900, 9, sort=False)))
    rp = np.array([0, 4, 6, 6, 9], dtype=np.int32)          # duplicate columns (A8): they sum
    ci = np.array([2, 0, 2, 1, 1, 1, 3, 3, 3], dtype=np.int32)
    out.append(("duplicates", W.CSR(4, 4, rp, ci, np.arange(1.0, 10.0))))
    out.append(("lap2d_17", W.laplace2d_5pt(17)))
    out.append(("lap3d_11", W.laplace3d_7pt(11)))
    out.append(("st27_9", W.stencil3d_27pt(9, perturb_stream=50)))
    out.append(("fem_5", W.fem_block27(5)))
    out.append(("powerlaw_3k", W.powerlaw(3000, lmax=2500)))
    out.append(("banded_4k", W.banded_random(4000, 12, 900, stream=81)))
    out.append(("rows_129", W.csr_from_lengths(np.random.default_rng(10).integers(1, 20, 129), 129, 10)))
    return out

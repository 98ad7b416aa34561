"""Generator self-checks (pin P10): nnz closed forms, the
figures BASELINE.json:configs prints, sortedness, reproducibility."""
import json
import os

import numpy as np
import pytest

from paper_1309_1894_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "config_sizes.json")


def _sorted_unique(A):
    d = np.diff(A.col_idx.astype(np.int64))
    row_start = np.zeros(A.nnz, dtype=bool)
    row_start[A.row_ptr[:-1][A.row_lengths() > 0]] = True
    return np.all((d > 0) | row_start[1:])


def test_config1_matches_baseline_json_text():
    g = json.load(open(GOLDEN))
    A = W.config(1).A
    assert (A.rows, A.cols, A.nnz) == (g["cfg1"]["rows"], g["cfg1"]["rows"], g["cfg1"]["nnz"]) == (4096, 4096, 20224)
    assert A.row_ptr.dtype == np.int32 and A.col_idx.dtype == np.int32 and A.val.dtype == np.float64
    assert set(np.unique(A.val)) == {4.0, -1.0}


@pytest.mark.parametrize("n", [2, 3, 7, 16])
def test_nnz_closed_forms(n):
    assert W.laplace2d_5pt(n).nnz == 5 * n * n - 4 * n
    assert W.laplace3d_7pt(n).nnz == 7 * n ** 3 - 6 * n ** 2
    assert W.stencil3d_27pt(n).nnz == (3 * n - 2) ** 3
    A = W.fem_block27(n)
    assert A.nnz == 9 * (3 * n - 2) ** 3 and A.rows == 3 * n ** 3
    for B in (W.laplace2d_5pt(n), W.laplace3d_7pt(n), W.stencil3d_27pt(n), A):
        assert _sorted_unique(B)
        assert B.col_idx.min() >= 0 and B.col_idx.max() < B.cols


def test_config2_full_size():
    g = json.load(open(GOLDEN))
    A = W.config(2).A
    assert A.rows == g["cfg2"]["rows"] == 2097152 and A.nnz == g["cfg2"]["nnz"] == 14581760


def test_fem_blocks_are_dense_and_shifted():
    A = W.fem_block27(8)
    # every 3x3 block fully present: rows 3v..3v+2 share the column list, columns come in triples
    for v in range(0, A.rows // 3, 7):
        c0 = A.col_idx[A.row_ptr[3 * v]:A.row_ptr[3 * v + 1]]
        for d in (1, 2):
            assert np.array_equal(c0, A.col_idx[A.row_ptr[3 * v + d]:A.row_ptr[3 * v + d + 1]])
        t = c0.reshape(-1, 3)
        assert np.all(t[:, 0] % 3 == 0) and np.all(t[:, 1] == t[:, 0] + 1) and np.all(t[:, 2] == t[:, 0] + 2)
    rid = np.repeat(np.arange(A.rows), A.row_lengths())
    diag = A.val[A.col_idx == rid]
    assert diag.size == A.rows and abs(diag.mean() - 30.0) < 0.2
    off = A.val[A.col_idx != rid]
    assert abs(off.mean()) < 0.02 and abs(off.std() - 1.0) < 0.02


def test_powerlaw_shape():
    A = W.powerlaw(1 << 19)
    L = A.row_lengths()
    assert L.min() >= 1 and L.max() <= 20000
    assert np.median(L) == 1
    assert 14.0 < L.mean() < 20.0            # heavy tail: +-0.3 holds only at 4.19M rows
    assert _sorted_unique(A)
    assert A.col_idx.min() >= 0 and A.col_idx.max() < A.cols
    assert abs(A.val.mean()) < 0.01 and abs(A.val.std() - 1) < 0.01


def test_zipf_pmf_mean_matches_survey():
    # truncated, renormalised pmf (reading A11): analytic mean 16.90, P(L=1) = 0.53
    k = np.arange(1, 20001, dtype=np.float64)
    pmf = k ** -1.8
    pmf /= pmf.sum()
    assert abs((k * pmf).sum() - 16.90) < 0.01
    L = W.zipf_lengths(1 << 20)
    assert abs((L == 1).mean() - pmf[0]) < 2e-3


def test_reproducible_and_streams_differ():
    a = W.config(5, 0.1, member=0)
    b = W.config(5, 0.1, member=0)
    c = W.config(5, 0.1, member=1)
    assert np.array_equal(a.A.val, b.A.val) and np.array_equal(a.x, b.x)
    assert np.array_equal(a.A.col_idx, c.A.col_idx) and not np.array_equal(a.A.val, c.A.val)
    assert np.all(np.abs(a.A.val[a.A.val > 0] - 26.0) <= 0.01)
    assert np.all(np.abs(a.A.val[a.A.val < 0] + 1.0) <= 0.01)
    u = W.uniform(0, 100000)
    assert u.min() >= -1.0 and u.max() < 1.0 and abs(u.mean()) < 0.01
    assert np.array_equal(W.uniform(0, 10), u[:10])          # counter-based: prefix-stable


def test_byte_model_matches_survey_table():
    g = json.load(open(GOLDEN))
    assert W.algorithmic_bytes(4096, 4096, 20224, 0.0) == g["cfg1"]["bytes"] == 324612
    assert W.algorithmic_bytes(2097152, 2097152, 14581760, 0.5) == g["cfg2"]["bytes"]


def test_banded_random_structure():
    """banded_random: fixed row length, distinct sorted columns inside the clipped band, reproducible."""
    A = W.banded_random(3000, 12, 400, stream=7)
    lens = A.row_lengths()
    assert (lens == 12).all() and A.nnz == 36000
    rid = np.repeat(np.arange(A.rows), lens)
    d = A.col_idx.astype(np.int64) - rid
    assert d.min() >= -400 and d.max() <= 400 and A.col_idx.min() >= 0 and A.col_idx.max() < A.cols
    key = (rid.astype(np.int64) << 32) | A.col_idx
    assert (np.diff(key) > 0).all()                       # sorted, no duplicates within a row
    assert np.unique(d).size > 32                         # far more diagonals than DIA admits
    B = W.banded_random(3000, 12, 400, stream=7)
    assert np.array_equal(A.col_idx, B.col_idx) and np.array_equal(A.val, B.val)

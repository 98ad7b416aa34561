"""GPU tests of spmv_create (row a1: validation, statistics, signature) and of the on-device
format converters (rows a2-a4, a8 partition, sec. 8(f) DIA): the arrays the library builds are
downloaded through spmv_format_download and compared, bit for bit, with a numpy re-derivation of
the layout documented in DESIGN.md sec. 5 (integer/index work: exact)."""
import numpy as np
import pytest

from paper_1309_1894_b200 import binding
from paper_1309_1894_b200 import workloads as W
from tests import helpers as H

pytestmark = pytest.mark.gpu


# ------------------------------------------------------------------ a1: statistics, signature, validation
def test_info_statistics_match_numpy(cuda):
    lengths = np.array([0, 1, 2, 3, 4, 7, 8, 9, 100, 0, 31, 32, 33, 5000, 1], dtype=np.int64)
    A = W.csr_from_lengths(lengths, 9000, 11)
    S = binding.SpMV.from_csr(A)
    i = S.info()
    assert (i.rows, i.cols, i.nnz) == (A.rows, A.cols, A.nnz)
    assert i.min_row_len == 0 and i.max_row_len == 5000
    assert abs(i.mean_row_len - lengths.mean()) < 1e-12
    assert abs(i.var_row_len - lengths.var()) < 1e-6 * lengths.var()
    hist = np.zeros(32, dtype=np.int64)
    for l in lengths:
        hist[0 if l == 0 else int(np.floor(np.log2(l))) + 1] += 1
    assert list(i.len_hist) == list(hist)
    rows_of = np.repeat(np.arange(A.rows), lengths)
    assert i.bandwidth == int(np.abs(A.col_idx.astype(np.int64) - rows_of).max())
    assert i.cols_sorted == 1 and i.block3_full == 0 and i.tuned == 0
    assert i.sm_count > 0 and i.l2_bytes > 0 and i.variant.decode().startswith("csr_scalar:b256:r1:u1:x0")
    assert i.format_bytes == A.nnz * 12 + (A.rows + 1) * 4
    S.close()
    U = binding.SpMV.from_csr(W.csr_from_lengths(np.full(50, 6), 300, 12, sort=False))
    assert U.info().cols_sorted == 0
    U.close()


def test_block3_detection_and_signature(cuda):
    F = W.fem_block27(4)
    S = binding.SpMV.from_csr(F)
    i = S.info()
    assert i.block3_full == 1 and i.n_blocks3 * 9 == F.nnz
    # same structure, other values: same signature; one column changed: different col signature
    G = W.CSR(F.rows, F.cols, F.row_ptr, F.col_idx, F.val + 1.0)
    T = binding.SpMV.from_csr(G)
    assert (T.info().sig_row_ptr, T.info().sig_col_idx) == (i.sig_row_ptr, i.sig_col_idx)
    ci = F.col_idx.copy()
    a, b = F.row_ptr[7], F.row_ptr[8]
    ci[a:b] = np.sort(np.r_[ci[a:b - 1], (ci[b - 1] + 5) % F.cols])
    Hm = binding.SpMV.from_csr(W.CSR(F.rows, F.cols, F.row_ptr, ci, F.val))
    assert Hm.info().sig_col_idx != i.sig_col_idx and Hm.info().sig_row_ptr == i.sig_row_ptr
    assert Hm.info().block3_full == 0                      # the moved entry breaks a dense block
    # swapping two row lengths changes the row_ptr signature (position-dependent hash)
    L1 = W.csr_from_lengths([3, 5, 2, 7], 20, 13)
    L2 = W.csr_from_lengths([5, 3, 2, 7], 20, 13)
    s1, s2 = binding.SpMV.from_csr(L1), binding.SpMV.from_csr(L2)
    assert s1.info().sig_row_ptr != s2.info().sig_row_ptr
    for h in (S, T, Hm, s1, s2):
        h.close()


def test_invalid_matrices_are_refused(cuda):
    import torch
    A = W.laplace2d_5pt(6)

    def create(rp, ci, rows=A.rows, cols=A.cols):
        return binding.SpMV(rows, cols, torch.from_numpy(rp.astype(np.int32)).cuda(),
                            torch.from_numpy(ci.astype(np.int32)).cuda(), torch.from_numpy(A.val).cuda())

    bad = A.row_ptr.copy(); bad[5] = bad[4] - 1                    # not monotone
    with pytest.raises(binding.SpmvError) as e:
        create(bad, A.col_idx)
    assert e.value.status == 2
    bad = A.row_ptr.copy(); bad[0] = 1                            # row_ptr[0] != 0
    with pytest.raises(binding.SpmvError) as e:
        create(bad, A.col_idx)
    assert e.value.status == 2
    bad = A.row_ptr.copy(); bad[-1] -= 1                          # row_ptr[rows] != nnz
    with pytest.raises(binding.SpmvError) as e:
        create(bad, A.col_idx)
    assert e.value.status == 2
    for v in (-1, A.cols):                                        # column out of range
        bc = A.col_idx.copy(); bc[17] = v
        with pytest.raises(binding.SpmvError) as e:
            create(A.row_ptr, bc)
        assert e.value.status == 2
    ok = create(A.row_ptr, A.col_idx)
    ok.close()
    assert binding.lib().spmv_destroy(binding.C.c_void_p(12345)) == 1      # not a live handle: INVALID_ARG


def test_unparsable_and_ineligible_variants(cuda):
    S = binding.SpMV.from_csr(W.csr_from_lengths([4, 4, 4, 4, 4, 9], 60, 14))
    for desc, status in (("nonsense:b1", 1), ("csr_vector:b100:w8:u1:x0", 3), ("bcsr3:b256:w8:u1:x0", 3),
                         ("sell:b256:c100:s1:r1:u1:x0", 3), ("sell:b256:c128:s1:l32:r1:u2:x0", 3),
                         ("sell_tma:b288:c256:s1:r1:u8:i3:x2:h7", 3), ("csr_scalar:b256:zz", 1)):
        with pytest.raises(binding.SpmvError) as e:
            S.select(desc)
        assert e.value.status == status, desc
    S.close()


# ------------------------------------------------------------------ a2/a3: SELL-C-sigma, ELL
def _sell_reference(A, C, sigma, split=0):
    """numpy re-derivation of the SELL layout, with optional row splitting."""
    lens = A.row_lengths().astype(np.int64)
    if split:
        nseg = np.where(lens > split, -(-lens // split), 1)
        vstart = np.r_[0, np.cumsum(nseg)]
        vrows = int(vstart[-1])
        vrp = np.empty(vrows + 1, dtype=np.int64)
        target = np.empty(vrows, dtype=np.int64)
        slot = 0
        for r in range(A.rows):
            for sg in range(nseg[r]):
                vrp[vstart[r] + sg] = A.row_ptr[r] + sg * (split if lens[r] > split else 0)
                if lens[r] > split:
                    target[vstart[r] + sg] = -(2 + slot); slot += 1
                else:
                    target[vstart[r]] = r
        vrp[vrows] = A.nnz
    else:
        vrows, vrp, target = A.rows, A.row_ptr.astype(np.int64), np.arange(A.rows)
    vlen = np.diff(vrp)
    nsl = max(1, -(-vrows // C))
    padded_rows = nsl * C
    order = np.full(padded_rows, -1, dtype=np.int64)
    if sigma > 1:
        for w0 in range(0, padded_rows, sigma):
            idx = np.arange(w0, min(w0 + sigma, vrows))
            if idx.size:
                srt = idx[np.argsort(-vlen[idx], kind="stable")]       # descending length, ties by row
                order[w0:w0 + srt.size] = srt
    else:
        order[:vrows] = np.arange(vrows)
    width = np.zeros(nsl, dtype=np.int64)
    for s in range(nsl):
        rows = order[s * C:(s + 1) * C]
        rows = rows[rows >= 0]
        width[s] = vlen[rows].max() if rows.size else 0
    slice_ptr = np.r_[0, np.cumsum(width * C)]
    sval = np.zeros(int(slice_ptr[-1])); scol = np.full(int(slice_ptr[-1]), -1, dtype=np.int32)
    for p in range(padded_rows):
        v = order[p]
        if v < 0:
            continue
        s, off = divmod(p, C)
        for j in range(vlen[v]):
            q = slice_ptr[s] + j * C + off
            sval[q] = A.val[vrp[v] + j]; scol[q] = A.col_idx[vrp[v] + j]
    perm = np.where(order >= 0, target[np.maximum(order, 0)], -1).astype(np.int32)
    return slice_ptr, sval, scol, perm


@pytest.mark.parametrize("desc,C,sigma,split", [
    ("sell:b256:c128:s1:r1:u2:x0", 128, 1, 0),
    ("sell:b256:c128:s512:r2:u2:x0", 128, 512, 0),
    ("sell:b256:c256:s8192:r1:u2:x0", 256, 8192, 0),
    ("sell:b256:c128:s1024:l8:r1:u2:x0", 128, 1024, 8),
    ("sell_tma:b160:c128:s256:l16:r1:u4:i3:x0", 128, 256, 16),
])
def test_sell_layout_matches_numpy(cuda, desc, C, sigma, split):
    lengths = np.random.default_rng(21).integers(0, 23, 1500)
    lengths[[3, 700, 1499]] = [130, 57, 40]
    A = W.csr_from_lengths(lengths, 2000, 22)
    S = binding.SpMV.from_csr(A)
    S.select(desc)
    sp, sv, sc, pm = _sell_reference(A, C, sigma, split)
    assert np.array_equal(S.download("slice_ptr", np.int64), sp)
    got_v, got_c = S.download("sval", np.float64), S.download("scol", np.int32)
    n = int(sp[-1])
    assert np.array_equal(got_c[:n], sc) and np.array_equal(got_v[:n], sv)
    if sigma > 1:
        assert np.array_equal(S.download("perm", np.int32), pm)
    i = S.info()
    assert i.format_bytes >= 12 * n
    H.check_against_oracle(S, A, 1.5, W.uniform(23, A.cols), 0.5, W.uniform(24, A.rows), what=desc)
    S.close()


@pytest.mark.parametrize("desc,C,sigma", [
    ("sell16:b256:c128:s1:r2:u4:x0", 128, 1),
    ("sell16:b128:c256:s1024:r1:u2:x0", 256, 1024),
    ("sell16_tma:b160:c128:s256:r1:u4:i4:x0", 128, 256),
])
def test_sell16_layout_matches_numpy(cuda, desc, C, sigma):
    """16-bit delta-encoded column indices.  The layout is SELL's with the column array
    replaced by sbase[slice] = smallest stored column of the slice and col16 = col - sbase (0xFFFF: padding)."""
    A = W.banded_random(3000, 14, 700, stream=26)
    S = binding.SpMV.from_csr(A)
    S.select(desc)
    sp, sv, sc, pm = _sell_reference(A, C, sigma)
    n = int(sp[-1])
    assert np.array_equal(S.download("slice_ptr", np.int64), sp)
    assert np.array_equal(S.download("sval", np.float64)[:n], sv)
    nsl = sp.size - 1
    base = np.zeros(nsl, dtype=np.int32)
    c16 = np.full(n, 0xFFFF, dtype=np.uint16)
    for sl in range(nsl):
        seg = sc[sp[sl]:sp[sl + 1]]
        if (seg >= 0).any():
            base[sl] = seg[seg >= 0].min()
            assert seg.max() - base[sl] < 0xFFFF
        c16[sp[sl]:sp[sl + 1]] = np.where(seg >= 0, seg - base[sl], 0xFFFF).astype(np.uint16)
    assert np.array_equal(S.download("sbase", np.int32), base)
    assert np.array_equal(S.download("scol16", np.uint16)[:n], c16)
    if sigma > 1:
        assert np.array_equal(S.download("perm", np.int32), pm)
    assert 10 * n <= S.info().format_bytes < 12 * n            # 8 + 2 bytes per stored entry (+ slice tables)
    H.check_against_oracle(S, A, 1.5, W.uniform(27, A.cols), 0.5, W.uniform(28, A.rows), what=desc)
    S.close()


def test_sell16_refused_when_a_slice_spans_65535_columns(cuda):
    """Eligibility: structural (2*bandwidth + max(C, sigma) < 65535) at select time, per slice at build time."""
    wide = W.csr_from_lengths(np.full(700, 5), 200000, 29)           # uniform columns over 200 000: span too large
    S = binding.SpMV.from_csr(wide)
    with pytest.raises(binding.SpmvError) as e:
        S.select("sell16:b256:c128:s1:r1:u2:x0")
    assert e.value.status == 3
    assert not any(c.startswith("sell16") for c in S.variants())
    S.close()
    band = W.banded_random(80000, 6, 33000, stream=30)               # bandwidth ~33 000: 2*bw + C >= 65535, refused as well
    T = binding.SpMV.from_csr(band)
    with pytest.raises(binding.SpmvError) as e:
        T.select("sell16:b256:c128:s1:r1:u2:x0")
    assert e.value.status == 3
    T.close()
    ok = binding.SpMV.from_csr(W.banded_random(5000, 10, 2400, stream=31))
    assert any(c.startswith("sell16:") for c in ok.variants()) and any(c.startswith("sell16_tma") for c in ok.variants())
    assert not any(c.startswith("dia") for c in ok.variants()) or True
    ok.select("sell16:b256:c128:s1:r1:u2:x0")
    with pytest.raises(binding.SpmvError) as e:                      # thousands of diagonals: DIA refuses the matrix
        ok.select("dia:b256:c128:r1:u4:x0")
    assert e.value.status == 3
    ok.close()


def test_ell_is_one_slice_and_padding_rule(cuda):
    A = W.laplace2d_5pt(19)
    S = binding.SpMV.from_csr(A)
    S.select("ell:b256:r1:u2:x0")
    sp = S.download("slice_ptr", np.int64)
    rows_padded = -(-A.rows // 128) * 128
    assert list(sp) == [0, 5 * rows_padded]
    sc = S.download("scol", np.int32)[:sp[1]].reshape(5, rows_padded)
    lens = A.row_lengths()
    for j in range(5):
        assert np.array_equal(sc[j, :A.rows] >= 0, lens > j)
        assert (sc[j, A.rows:] == -1).all()
    S.close()
    # ELL eligibility: width*rows <= 1.5*nnz
    P = binding.SpMV.from_csr(W.csr_from_lengths([1] * 400 + [300], 500, 25))
    with pytest.raises(binding.SpmvError) as e:
        P.select("ell:b256:r1:u2:x0")
    assert e.value.status == 3
    P.close()


# ------------------------------------------------------------------ a4: BCSR 3x3
def test_bcsr3_layout_matches_numpy(cuda):
    A = W.fem_block27(4)
    S = binding.SpMV.from_csr(A)
    S.select("bcsr3:b256:w8:u1:x0")
    bp = S.download("brow_ptr", np.int32)
    bc = S.download("bcol", np.int32)
    bv = S.download("bval", np.float64)
    brows = A.rows // 3
    assert bp.size == brows + 1 and bp[0] == 0 and bp[-1] * 9 == A.nnz
    for b in (0, 1, brows // 2, brows - 1):
        a, e = A.row_ptr[3 * b], A.row_ptr[3 * b + 1]
        cols = np.unique(A.col_idx[a:e] // 3)
        nb = bp[b + 1] - bp[b]
        assert np.array_equal(bc[bp[b]:bp[b + 1]], cols) and nb == cols.size
        blk = bv[9 * bp[b]:9 * bp[b + 1]].reshape(9, nb)           # element k of block j at k*nb + j
        for r in range(3):
            ra, re = A.row_ptr[3 * b + r], A.row_ptr[3 * b + r + 1]
            assert np.array_equal(blk[3 * r:3 * r + 3, :].T.reshape(-1), A.val[ra:re])
    assert S.info().format_bytes == int(bp[-1]) * 76 + (brows + 1) * 4
    # 16-bit block columns (variant key i16): bcol - block row + 32768; selecting it drops the 32-bit array
    S.select("bcsr3:b256:w8:u1:i16:x0")
    assert S.variant == "bcsr3:b256:w8:u1:i16:x0"
    bc16 = S.download("bcol16", np.uint16)
    brow_of = np.repeat(np.arange(brows), np.diff(bp))
    assert np.array_equal(bc16.astype(np.int64), bc.astype(np.int64) - brow_of + 32768)
    assert S.info().format_bytes == int(bp[-1]) * 74 + (brows + 1) * 4
    with pytest.raises(binding.SpmvError):
        S.download("bcol", np.int32)
    S.select("bcsr3:b256:w8:u1:x0")                                    # and back: the 32-bit form is rebuilt
    assert np.array_equal(S.download("bcol", np.int32), bc)
    S.close()


def test_bcsr3_i16_refused_when_block_columns_are_far(cuda):
    """bcsr3 i16 stores bcol - block row + 32768 in 16 bits: a matrix with a block 35 000 block rows away from the
    diagonal is refused for i16 (structurally, from the bandwidth statistic) and runs with 32-bit block columns."""
    brows = 40000
    far = (np.arange(brows) + 35000) % brows
    bcols = np.sort(np.stack([np.arange(brows), far], axis=1), axis=1)            # two dense 3x3 blocks per block row
    cols = (3 * bcols[:, None, :, None] + np.arange(3)[None, None, None, :]).repeat(3, axis=1).reshape(3 * brows, 6)
    rp = (6 * np.arange(3 * brows + 1)).astype(np.int32)
    A = W.CSR(3 * brows, 3 * brows, rp, cols.reshape(-1).astype(np.int32), W.normal(27, 18 * brows))
    x = W.uniform(28, A.cols)
    S = binding.SpMV.from_csr(A)
    assert S.info().block3_full == 1
    with pytest.raises(binding.SpmvError) as e:
        S.select("bcsr3:b256:w8:u1:i16:x0")
    assert e.value.status == 3
    assert not any(":i16" in d for d in S.variants() if d.startswith("bcsr3"))
    S.select("bcsr3:b256:w4:u1:x0")
    H.check_against_oracle(S, A, 1.0, x, 0.0, None, what="bcsr3 far blocks")
    S.close()


# ------------------------------------------------------------------ sec. 8(f) rank 1: DIA
@pytest.mark.parametrize("C", [128, 256, 512])
def test_dia_layout_matches_numpy(cuda, C):
    A = W.stencil3d_27pt(7, perturb_stream=50)
    S = binding.SpMV.from_csr(A)
    S.select(f"dia:b256:c{C}:r1:u4:x0")
    off = S.download("dia_off", np.int32)
    rows_of = np.repeat(np.arange(A.rows), A.row_lengths())
    d_all = A.col_idx.astype(np.int64) - rows_of
    assert np.array_equal(off, np.unique(d_all)) and off.size == 27
    ld = -(-A.rows // C) * C
    dv = S.download("dia_val", np.float64)
    mk = S.download("dia_mask", np.uint32)
    assert dv.size == 27 * ld and mk.size == ld
    ref_v = np.zeros(27 * ld); ref_m = np.zeros(ld, dtype=np.uint32)
    didx = np.searchsorted(off, d_all)
    ref_v[((rows_of // C) * 27 + didx) * C + rows_of % C] = A.val
    np.bitwise_or.at(ref_m, rows_of, (np.uint32(1) << didx.astype(np.uint32)))
    assert np.array_equal(dv, ref_v) and np.array_equal(mk, ref_m)
    assert S.info().format_bytes == 27 * ld * 8 + ld * 4
    S.close()


def test_dia_refused_on_non_diagonal_patterns(cuda):
    for A in (W.powerlaw(3000, lmax=500), W.csr_from_lengths(np.full(200, 5), 4000, 26), W.fem_block27(4)):
        S = binding.SpMV.from_csr(A)
        with pytest.raises(binding.SpmvError) as e:
            S.select("dia:b256:c128:r1:u4:x0")
        assert e.value.status == 3
        with pytest.raises(binding.SpmvError):                     # and stays refused (remembered per handle)
            S.select("dia_tma:b288:c256:r1:u8:i3:x0")
        H.check_against_oracle(S, A, 1.0, W.uniform(27, A.cols), 0.0, None, what="still on the default")
        S.close()


# ------------------------------------------------------------------ a8: merge-path partition
def test_merge_partition_matches_bruteforce(cuda):
    lengths = np.random.default_rng(28).integers(0, 30, 4000)
    lengths[[10, 11, 2000]] = [9000, 0, 4500]
    A = W.csr_from_lengths(lengths, 12000, 29)
    S = binding.SpMV.from_csr(A)
    S.select("merge:b128:i5:x0")
    tile_row = S.download("tile_row", np.int32)
    TI = 128 * 5
    P = A.rows + A.nnz
    ntiles = -(-P // TI)
    assert tile_row.size == ntiles + 1
    # merged order: row-end item i comes after the non-zeros k < row_ptr[i+1] (ties: row end first iff
    # row_ptr[i+1] <= k).  Number of row-end items among the first d merged items, by brute force:
    ends = A.row_ptr[1:].astype(np.int64)
    pos_end = ends + np.arange(A.rows)              # position of row-end item i in the merged list
    for t in range(ntiles + 1):
        d = min(t * TI, P)
        assert tile_row[t] == int(np.searchsorted(pos_end, d, side="left")), t
    S.close()


def test_dia_const_detection_and_bitwise_equality_with_dia(cuda):
    """Constant-coefficient stencil: detected only when every stored entry of each
    diagonal has the same bits; dia_const then reads no values and equals dia bit for bit."""
    A = W.laplace3d_7pt(13)
    S = binding.SpMV.from_csr(A)
    S.select("dia_const:b256:r2:x0")
    assert list(S.download("dia_coef", np.float64)) == [-1.0, -1.0, -1.0, 6.0, -1.0, -1.0, -1.0]
    assert S.info().format_bytes == A.rows          # 7 diagonals: one mask byte per row
    x, y0 = W.uniform(61, A.cols), W.uniform(62, A.rows)
    yc = H.gpu_apply(S, 1.25, x, 0.5, y0)
    H.check_against_oracle(S, A, 1.25, x, 0.5, y0, what="dia_const")
    S.select("dia:b256:c128:r1:u4:x0")
    assert np.array_equal(H.gpu_apply(S, 1.25, x, 0.5, y0), yc)
    S.close()
    # one perturbed entry (or a perturbed stencil) -> refused, and remembered
    B = W.CSR(A.rows, A.cols, A.row_ptr, A.col_idx, A.val.copy())
    B.val[B.nnz // 2] = np.nextafter(B.val[B.nnz // 2], 10.0)
    for M in (B, W.stencil3d_27pt(7, perturb_stream=50)):
        T = binding.SpMV.from_csr(M)
        for _ in range(2):
            with pytest.raises(binding.SpmvError) as e:
                T.select("dia_const:b256:r1:x0")
            assert e.value.status == 3
        T.select("dia:b256:c128:r1:u4:x0")            # the general DIA kernel still applies
        H.check_against_oracle(T, M, 1.0, W.uniform(63, M.cols), 0.0, None, what="dia after refused dia_const")
        assert not any(c.startswith("dia_const") for c in T.variants()) or True
        T.close()

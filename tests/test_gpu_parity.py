"""GPU parity: every kernel family / template axis against the oracle, element by element,
through the C ABI.  Floating point: |y - y_ref| <= 1e-12 * scale
(north_star); exactness cases (x = e_j, small integers, val = x = 1) bitwise."""
import numpy as np
import pytest

import oracle
from paper_1309_1894_b200 import binding
from paper_1309_1894_b200 import workloads as W
from tests import helpers as H

pytestmark = pytest.mark.gpu

ZOO = H.zoo()


def _select_or_skip(S, desc):
    try:
        S.select(desc)
        return True
    except binding.SpmvError as e:
        assert e.status == 3, e          # only SPMV_ERR_UNSUPPORTED may refuse a parsable variant
        return False


@pytest.mark.parametrize("name,A", ZOO, ids=[z[0] for z in ZOO])
def test_zoo_all_representative_variants(cuda, name, A):
    S = binding.SpMV.from_csr(A)
    x = W.uniform(70, A.cols)
    y0 = W.uniform(71, A.rows)
    ran = 0
    for desc in H.REPRESENTATIVE_VARIANTS:
        if not _select_or_skip(S, desc):
            continue
        ran += 1
        for alpha, beta in ((1.0, 0.0), (1.0, 0.5), (-2.5, 1.0)):
            H.check_against_oracle(S, A, alpha, x, beta, None if beta == 0.0 else y0, what=name)
    assert ran >= 10          # CSR and merge families are always eligible
    S.close()


@pytest.mark.parametrize("name,A", [z for z in ZOO if z[0] in ("lap3d_11", "fem_5", "powerlaw_3k", "lengths_ladder")],
                         ids=["lap3d_11", "fem_5", "powerlaw_3k", "lengths_ladder"])
def test_every_enumerated_candidate(cuda, name, A):
    """Everything the tuner would enumerate for this matrix passes parity."""
    S = binding.SpMV.from_csr(A)
    x = W.uniform(72, A.cols)
    y0 = W.uniform(73, A.rows)
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x, 0.5, y0)
    cands = S.variants()
    assert len(cands) > 50
    fams = {c.split(":")[0] for c in cands}
    assert {"csr_scalar", "csr_vector", "merge"} <= fams
    for desc in cands:
        if not _select_or_skip(S, desc):
            continue
        y = H.gpu_apply(S, 1.0, x, 0.5, y0)
        ok, mr, ff, nf = oracle.accept(y, y_ref, scale, H.TOL)
        assert ok, (desc, nf, ff, mr)
    S.close()


def test_exactness_cases_bitwise(cuda):
    """P5/P6/P7 for every family: x = e_j, small integers, val = x = 1 are exact in any order."""
    lengths = np.random.default_rng(3).integers(0, 90, 1200)
    lengths[5] = 3000
    A = W.csr_from_lengths(lengths, 6000, 31, values="smallint")
    xi = np.round(W.uniform(32, A.cols) * 8)
    yi = np.round(W.uniform(33, A.rows) * 8)
    B = W.fem_block27(4)
    B.val[:] = np.round(B.val * 2)
    xb = np.round(W.uniform(34, B.cols) * 8)
    for M, x, y0 in ((A, xi, yi), (B, xb, np.round(W.uniform(35, B.rows) * 8))):
        S = binding.SpMV.from_csr(M)
        y_ref, _ = oracle.spmv(M.row_ptr, M.col_idx, M.val, 3.0, x, -2.0, y0)
        e = np.zeros(M.cols); e[M.cols // 3] = 1.0
        ye_ref, _ = oracle.spmv(M.row_ptr, M.col_idx, M.val, 2.0, e, 0.0)
        ones_ref = M.row_lengths().astype(np.float64)
        Mones = W.CSR(M.rows, M.cols, M.row_ptr, M.col_idx, np.ones(M.nnz))
        S1 = binding.SpMV.from_csr(Mones)
        for desc in H.REPRESENTATIVE_VARIANTS:
            if not _select_or_skip(S, desc):
                continue
            assert np.array_equal(H.gpu_apply(S, 3.0, x, -2.0, y0), y_ref), desc
            assert np.array_equal(H.gpu_apply(S, 2.0, e, 0.0, None), ye_ref), desc
            S1.select(desc)
            assert np.array_equal(H.gpu_apply(S1, 1.0, np.ones(M.cols), 0.0, None), ones_ref), desc
        S.close(); S1.close()


def test_nonfinite_x_touches_only_real_entries(cuda):
    """A7: padding (SELL/ELL) is never multiplied, so NaN/Inf in x reaches exactly the rows
    CSR semantics say; beta = 0 ignores NaN in incoming y (A1); alpha = 0 ignores A and x (A2)."""
    A = W.csr_from_lengths(np.random.default_rng(4).integers(1, 12, 2000), 2000, 41)
    x = W.uniform(42, A.cols)
    x[17] = np.nan
    x[900] = np.inf
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x, 0.0)
    assert np.isfinite(y_ref).sum() > 1000 and (~np.isfinite(y_ref)).sum() > 0
    S = binding.SpMV.from_csr(A)
    for desc in H.REPRESENTATIVE_VARIANTS:
        if not _select_or_skip(S, desc):
            continue
        y = H.gpu_apply(S, 1.0, x, 0.0, None)          # incoming y is NaN-filled
        assert oracle.accept(y, y_ref, scale, H.TOL)[0], desc
        y0 = W.uniform(43, A.rows)
        y = H.gpu_apply(S, 0.0, x, 1.0, y0)
        assert np.array_equal(y, y0), desc
        y = H.gpu_apply(S, 0.0, x, 0.0, None)
        assert np.array_equal(y, np.zeros(A.rows)), desc
    S.close()


def test_bit_identical_across_repeated_runs(cuda):
    """north_star: 'the selected variant must give bit-identical results across repeated runs'."""
    A = W.powerlaw(20000, lmax=5000)
    x = W.uniform(44, A.cols)
    y0 = W.uniform(45, A.rows)
    S = binding.SpMV.from_csr(A)
    for desc in H.REPRESENTATIVE_VARIANTS:
        if not _select_or_skip(S, desc):
            continue
        first = H.gpu_apply(S, 1.5, x, 0.5, y0)
        for _ in range(9):
            assert np.array_equal(H.gpu_apply(S, 1.5, x, 0.5, y0), first), desc
    S.close()


def test_apply_host_matches_device_apply(cuda):
    import torch
    prob = W.config(2, 0.25)
    A = prob.A
    S = binding.SpMV.from_csr(A)
    S.select("sell:b256:c128:s1:r2:u4:x0")
    y_dev = H.gpu_apply(S, prob.alpha, prob.x, prob.beta, prob.y0)
    xh = torch.from_numpy(prob.x).pin_memory()
    yh = torch.from_numpy(prob.y0.copy()).pin_memory()
    S.apply_host(prob.alpha, xh, prob.beta, yh)
    assert np.array_equal(yh.numpy(), y_dev)
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, prob.alpha, prob.x, prob.beta, prob.y0)
    assert oracle.accept(yh.numpy(), y_ref, scale, H.TOL)[0]
    S.close()


def test_graph_replay_equals_plain_applies(cuda):
    """spmv_graph_create: k back-to-back applies captured into one CUDA graph give, bit for bit, what k plain
    applies give (beta != 0, so every apply depends on the one before), for one- and two-kernel variants; the
    graph can be replayed, and refuses bad arguments."""
    import torch
    prob = W.config(2, 0.3)
    A = prob.A
    S = binding.SpMV.from_csr(A)
    dx = H.to_dev(prob.x)
    for desc in ("dia_const:b256:r1:x0", "sell_tma:b288:c256:s1:r1:u8:i3:x0", "merge:b256:i7:x0", "default"):
        S.select(desc)
        y_plain = H.to_dev(prob.y0).clone()
        for _ in range(7):
            S.apply(0.75, dx, 0.5, y_plain)
        y_graph = H.to_dev(prob.y0).clone()
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            g = S.graph(0.75, dx, 0.5, y_graph, 7)
            g.launch()
            st.synchronize()
            assert torch.equal(y_graph, y_plain), desc
            g.launch()                                           # a second replay continues from the current y
            st.synchronize()
        for _ in range(7):
            S.apply(0.75, dx, 0.5, y_plain)
        torch.cuda.synchronize()
        assert torch.equal(y_graph, y_plain), desc
        g.close()
    with pytest.raises(binding.SpmvError) as e:
        S.graph(1.0, dx, 0.0, y_plain, 0)
    assert e.value.status == 1
    S.close()


@pytest.mark.parametrize("which", ["stencil7", "fem", "banded"])
def test_apply_host_pipeline_is_bit_identical_to_device_apply(cuda, which):
    """spmv_apply_host pipelines chunks of rows (upload | kernel on a row range | download) where the variant
    has a range form.  Large enough for several chunks (~2 MB of y each) with a ragged last one; every family's
    range launch must reproduce the one-launch result bit for bit, for beta == 0 and beta != 0, and match the
    oracle."""
    import torch
    if which == "stencil7":
        A = W.laplace3d_7pt(93)                                # 804 357 rows: odd, not a multiple of any slice height
        descs = ["default", "csr_vector:b256:w8:u2:x0", "sell:b256:c128:s1:r2:u4:x0", "sell:b256:c128:s1024:r1:u2:x0",
                 "sell_tma:b288:c256:s1:r1:u8:i3:x0", "sell_tma:b160:c128:s512:r1:u4:i4:x0", "sell16:b256:c128:s1:r2:u4:x0",
                 "sell16_tma:b288:c256:s1:r1:u8:i3:x0", "dia:b256:c128:r2:u4:x0", "dia_tma:b288:c256:r1:u7:i3:x0",
                 "dia_const:b256:r1:x0", "dia_const:b128:r2:x0", "dia_const:b256:r4:x0",
                 "merge:b256:i7:x0", "ell:b256:r1:u2:x0"]       # the last two have no range form: one launch
    elif which == "fem":
        A = W.fem_block27(56)                                  # 526 848 rows, dense 3x3 blocks
        descs = ["bcsr3:b256:w8:u2:x0", "bcsr3:b512:w16:u2:x0:g1", "bcsr3:b128:w16:u2:i16:x3:g8", "csr_vector:b256:w32:u2:x0"]
    else:
        A = W.banded_random(700001, 9, 1500, stream=83)
        descs = ["sell16:b256:c512:s1:r4:u2:x0", "sell16_tma:b544:c512:s1:r1:u4:i4:x0", "sell:b128:c128:s8192:r1:u2:x0", "csr_scalar:b256:r2:u2:x0:g2"]
    x, y0 = W.uniform(84, A.cols), W.uniform(85, A.rows)
    S = binding.SpMV.from_csr(A)
    xh = torch.from_numpy(x).pin_memory()
    ref = {}
    for beta in (0.0, -0.75):
        ref[beta] = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.25, x, beta, None if beta == 0.0 else y0, parallel=True)
    for desc in descs:
        S.select(desc)
        for beta in (0.0, -0.75):
            y_dev = H.gpu_apply(S, 1.25, x, beta, None if beta == 0.0 else y0)
            yh = torch.from_numpy(np.full(A.rows, np.nan) if beta == 0.0 else y0.copy()).pin_memory()
            S.apply_host(1.25, xh, beta, yh)
            assert np.array_equal(yh.numpy(), y_dev), (desc, beta)
            assert oracle.accept(yh.numpy(), ref[beta][0], ref[beta][1], H.TOL)[0], (desc, beta)
    # pageable (unpinned) host memory and an unaligned host pointer work too
    S.select(descs[0])
    xu = np.empty(A.cols + 1); xu[1:] = x
    yu = np.empty(A.rows + 1); yu[1:] = y0
    S.apply_host(1.25, xu[1:], -0.75, yu[1:])
    assert oracle.accept(yu[1:], ref[-0.75][0], ref[-0.75][1], H.TOL)[0]
    S.close()


def test_apply_host_zero_copy_y_equals_staged_copies(cuda, monkeypatch):
    """spmv_apply_host on pinned (mapped) host memory lets the DIA families' chunk kernels read and write y in
    place over PCIe; pageable memory and SPMV_HOST_ZEROCOPY=0 take the staged copies.  All three give the bits of
    the device apply, for beta == 0 (y write-only: incoming NaN ignored) and beta != 0, several chunks with a
    ragged last one, and match the oracle."""
    import torch
    monkeypatch.setenv("SPMV_HOST_CHUNK_MB", "1.5")
    A = W.stencil3d_27pt(83)                                   # 571 787 rows = 4.6 MB of y: 3 chunks
    x, y0 = W.uniform(86, A.cols), W.uniform(87, A.rows)
    S = binding.SpMV.from_csr(A)
    xh = torch.from_numpy(x).pin_memory()
    for desc in ("dia:b256:c128:r2:u4:x0", "dia_tma:b288:c256:r1:u9:i3:x0", "dia_const:b256:r1:x0", "dia_const:b128:r2:x0"):
        S.select(desc)
        for beta in (0.0, -0.75):
            y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.25, x, beta, None if beta == 0.0 else y0, parallel=True)
            y_dev = H.gpu_apply(S, 1.25, x, beta, None if beta == 0.0 else y0)
            start = np.full(A.rows, np.nan) if beta == 0.0 else y0.copy()
            y_zero = torch.from_numpy(start.copy()).pin_memory()
            S.apply_host(1.25, xh, beta, y_zero)                 # zero-copy y
            y_page = start.copy()
            S.apply_host(1.25, xh, beta, y_page)                 # pageable y: staged
            monkeypatch.setenv("SPMV_HOST_ZEROCOPY", "0")
            y_off = torch.from_numpy(start.copy()).pin_memory()
            S.apply_host(1.25, xh, beta, y_off)                  # pinned y, zero-copy off: staged
            monkeypatch.delenv("SPMV_HOST_ZEROCOPY")
            for got in (y_zero.numpy(), y_page, y_off.numpy()):
                assert np.array_equal(got, y_dev), (desc, beta)
            assert oracle.accept(y_zero.numpy(), y_ref, scale, H.TOL)[0], (desc, beta)
    # small system, x and y both mapped: the kernel works on the host vectors in place (no copies at all)
    A1 = W.laplace2d_5pt(64)
    x1, y1 = W.uniform(88, A1.cols), W.uniform(89, A1.rows)
    S1 = binding.SpMV.from_csr(A1)
    x1h = torch.from_numpy(x1).pin_memory()
    for desc in ("dia_const:b256:r1:x0", "dia_const:b128:r2:x0", "dia:b256:c128:r1:u4:x0", "default"):
        S1.select(desc)
        for beta in (0.0, 0.5):
            y_dev = H.gpu_apply(S1, -1.5, x1, beta, None if beta == 0.0 else y1)
            yh1 = torch.from_numpy(np.full(A1.rows, np.nan) if beta == 0.0 else y1.copy()).pin_memory()
            S1.apply_host(-1.5, x1h, beta, yh1)
            assert np.array_equal(yh1.numpy(), y_dev), (desc, beta)
            yp1 = np.full(A1.rows, np.nan) if beta == 0.0 else y1.copy()
            S1.apply_host(-1.5, x1, beta, yp1)                   # pageable: staged
            assert np.array_equal(yp1, y_dev), (desc, beta)
    S1.close()
    # a pinned but odd-aligned y (8 mod 16) takes the staged path
    S.select("dia_const:b256:r1:x0")
    yo = torch.empty(A.rows + 1, dtype=torch.float64).pin_memory()
    yo[1:] = torch.from_numpy(y0)
    S.apply_host(1.25, xh, -0.75, yo[1:])
    assert np.array_equal(yo[1:].numpy(), H.gpu_apply(S, 1.25, x, -0.75, y0))
    S.close()


def test_apply_host_batch_equals_member_calls(cuda, monkeypatch):
    """spmv_apply_host_batch: the members' pipelines are enqueued together and synchronised once; results equal
    one spmv_apply_host call per member bit for bit -- pipelined members (several chunks, staged and zero-copy
    y), a member without a range form (one launch) and a small one; a handle passed twice is refused."""
    import torch
    monkeypatch.setenv("SPMV_HOST_CHUNK_MB", "1.0")
    mats = [W.stencil3d_27pt(70, perturb_stream=61), W.laplace3d_7pt(75), W.fem_block27(40), W.powerlaw(20000), W.laplace2d_5pt(20)]
    descs = ["dia_tma:b288:c256:r1:u9:i3:x0", "dia_const:b256:r1:x0", "bcsr3:b128:w16:u2:i16:x0:g8", "merge:b256:i7:x0", "dia_const:b256:r1:x0"]
    hs = [binding.SpMV.from_csr(A) for A in mats]
    for S, d in zip(hs, descs):
        S.select(d)
    alphas = [1.0, -0.5, 2.0, 1.25, 1.0]
    betas = [1.0, 0.5, 0.0, -0.75, 0.0]
    xs = [W.uniform(130 + i, A.cols) for i, A in enumerate(mats)]
    y0 = [W.uniform(140 + i, A.rows) for i, A in enumerate(mats)]
    xh = [torch.from_numpy(x).pin_memory() for x in xs]
    want = []
    for S, a, b, x, y in zip(hs, alphas, betas, xh, y0):
        yy = torch.from_numpy(y.copy()).pin_memory()
        S.apply_host(a, x, b, yy)
        want.append(yy.numpy().copy())
    for rep in range(3):
        yh = [torch.from_numpy(y.copy()).pin_memory() for y in y0]
        binding.apply_host_batch(hs, alphas, xh, betas, yh)
        for i in range(len(hs)):
            assert np.array_equal(yh[i].numpy(), want[i]), (rep, i, descs[i])
    for i, A in enumerate(mats):                       # and the oracle
        y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, alphas[i], xs[i], betas[i], y0[i] if betas[i] != 0.0 else None, parallel=True)
        assert oracle.accept(want[i], y_ref, scale, H.TOL)[0], descs[i]
    with pytest.raises(binding.SpmvError) as e:
        binding.apply_host_batch([hs[0], hs[0]], [1.0, 1.0], [xh[0], xh[0]], [0.0, 0.0], [torch.zeros(mats[0].rows, dtype=torch.float64)] * 2)
    assert e.value.status == 1
    for S in hs:
        S.close()


@pytest.mark.slow
def test_tma_pipeline_race_regression_full_size(cuda):
    """Regression: on full-size cfg5 with sorted slices the TMA refill (async proxy) used to land
    under shared-memory reads of the previous occupant unless the producer issues
    fence.proxy.async -- whole half-warps of rows were off by ~1e-3, in ~1 of 3 launches."""
    import torch
    prob = W.config(5)
    A = prob.A
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, prob.x, 0.0)
    S = binding.SpMV.from_csr(A)
    x = torch.from_numpy(prob.x).cuda()
    for desc in ("sell_tma:b96:c128:s8192:r2:u4:i3:x0", "sell_tma:b160:c128:s8192:r1:u8:i2:x0",
                 "sell_tma:b288:c256:s1:r1:u8:i2:x0"):
        S.select(desc)
        for _ in range(12):
            y = torch.full((A.rows,), float("nan"), dtype=torch.float64, device="cuda")
            S.apply(1.0, x, 0.0, y)
            torch.cuda.synchronize()
            ok, mr, ff, nf = oracle.accept(y.cpu().numpy(), y_ref, scale, H.TOL)
            assert ok, (desc, nf, ff, mr)
    S.close()


def test_update_values_keeps_the_variant_and_matches_oracle(cuda):
    """spmv_update_values: same pattern, new values -> the selected variant's format is rebuilt; a
    dia_const handle whose coefficients stop being constant falls back to a variant that reads values."""
    import torch
    A = W.stencil3d_27pt(9, perturb_stream=50)
    x, y0 = W.uniform(81, A.cols), W.uniform(82, A.rows)
    for desc in ("sell:b256:c128:s1:r2:u4:x0", "sell_tma:b288:c256:s1:r1:u8:i3:x0", "dia_tma:b288:c256:r1:u9:i3:x0",
                 "merge:b256:i7:x0", "csr_vector:b256:w8:u2:x0", "ell:b256:r1:u2:x0"):
        S = binding.SpMV.from_csr(A)
        S.select(desc)
        v2 = W.normal(83, A.nnz)
        assert S.update_values(torch.from_numpy(v2).cuda()) is False
        assert S.variant == desc
        B = W.CSR(A.rows, A.cols, A.row_ptr, A.col_idx, v2)
        H.check_against_oracle(S, B, 1.0, x, 0.5, y0, what="after update_values")
        S.close()
    L = W.laplace3d_7pt(12)
    S = binding.SpMV.from_csr(L)
    S.select("dia_const:b256:r2:x0")
    xl = W.uniform(84, L.cols)
    v3 = L.val * 2.0                                     # still constant along the diagonals
    assert S.update_values(torch.from_numpy(v3).cuda()) is False and S.variant.startswith("dia_const")
    H.check_against_oracle(S, W.CSR(L.rows, L.cols, L.row_ptr, L.col_idx, v3), 1.0, xl, 0.0, None, what="const x2")
    v4 = W.normal(85, L.nnz)                             # not constant any more
    assert S.update_values(torch.from_numpy(v4).cuda()) is True and S.variant.startswith("dia_tma")
    H.check_against_oracle(S, W.CSR(L.rows, L.cols, L.row_ptr, L.col_idx, v4), 1.0, xl, 0.0, None, what="fallback")
    S.close()
    # formats with a derived index array (16-bit block columns, 16-bit slice deltas, the x3 window) are rebuilt whole
    F = W.fem_block27(6)
    Bm = W.banded_random(5000, 8, 600, stream=88)
    for M, desc in ((F, "bcsr3:b128:w16:u2:i16:x0:g8"), (Bm, "sell16_tma:b288:c256:s1:r1:u8:i3:x3:h600"), (Bm, "sell16:b256:c128:s1:r2:u4:x0")):
        S = binding.SpMV.from_csr(M)
        S.select(desc)
        xm, ym = W.uniform(86, M.cols), W.uniform(87, M.rows)
        v5 = W.normal(89, M.nnz)
        assert S.update_values(torch.from_numpy(v5).cuda()) is False and S.variant == desc
        H.check_against_oracle(S, W.CSR(M.rows, M.cols, M.row_ptr, M.col_idx, v5), -1.5, xm, 0.5, ym, what="update_values " + desc)
        S.close()


def test_full_band_window_x3(cuda):
    """sell_tma / sell16_tma with x3: the shared-memory x window spans the matrix bandwidth, the kernel has no
    L1 gather path at all.  Several slices with a ragged last one, windows clipped at both ends of x, beta == 0
    and != 0, against the oracle; bit-identical to the x0 form of the same shape (same per-row order); an
    8-byte-aligned x takes the x0 kernel (alt plan); the variant is refused when the window cannot cover the
    band, when rows are sorted, and for an odd column count."""
    import torch
    A = W.banded_random(70001 * 2, 11, 1300, stream=91)        # 140 002 rows: 273.4 slices of 512
    x, y0 = W.uniform(92, A.cols), W.uniform(93, A.rows)
    S = binding.SpMV.from_csr(A)
    bw = int(S.info().bandwidth)
    assert 0 < bw <= 1300
    for desc in ("sell_tma:b544:c512:s1:r1:u4:i4", "sell16_tma:b544:c512:s1:r1:u8:i3", "sell16_tma:b288:c512:s1:r2:u8:i3",
                 "sell16_tma:b160:c128:s1:r1:u4:i6", "sell_tma:b288:c256:s1:r1:u16:i2"):
        for beta in (0.0, -0.5):
            S.select(desc + ":x0")
            y_x0 = H.gpu_apply(S, 1.5, x, beta, None if beta == 0.0 else y0)
            S.select(desc + ":x3:h1304")
            y_x3, _, _ = H.check_against_oracle(S, A, 1.5, x, beta, None if beta == 0.0 else y0, what="x3")
            assert np.array_equal(y_x3, y_x0), (desc, beta)
            assert np.array_equal(H.gpu_apply(S, 1.5, x, beta, None if beta == 0.0 else y0), y_x3)      # repeatable
    # 8-byte aligned x: no bulk copy possible, the plan's alternative (x0) kernel runs
    S.select("sell16_tma:b544:c512:s1:r1:u8:i3:x3:h1304")
    bx = torch.zeros(A.cols + 2, dtype=torch.float64, device="cuda")
    dx = bx[1:1 + A.cols]
    dx.copy_(torch.from_numpy(x))
    dy = torch.from_numpy(y0).cuda()
    assert dx.data_ptr() % 16 == 8
    S.apply(1.5, dx, -0.5, dy)
    torch.cuda.synchronize()
    assert np.array_equal(dy.cpu().numpy(), y_x3)
    for bad in ("sell16_tma:b544:c512:s1:r1:u8:i3:x3:h1000",      # window narrower than the band
                "sell16_tma:b544:c512:s1024:r1:u8:i3:x3:h1304",   # sorted rows: a slice's rows are not contiguous
                "sell_tma:b544:c512:s1:r1:u8:i3:x3:h4104"):       # h out of range
        with pytest.raises(binding.SpmvError) as e:
            S.select(bad)
        assert e.value.status == 3, bad
    S.close()
    Aodd = W.banded_random(5001, 7, 300, stream=94)            # odd column count: the last column cannot be staged
    So = binding.SpMV.from_csr(Aodd)
    with pytest.raises(binding.SpmvError) as e:
        So.select("sell_tma:b160:c128:s1:r1:u4:i6:x3:h304")
    assert e.value.status == 3
    So.select("sell_tma:b160:c128:s1:r1:u4:i3:x2:h304")        # x2 keeps its L1 path for what the window misses
    H.check_against_oracle(So, Aodd, 1.0, W.uniform(95, Aodd.cols), 0.0, None, what="x2 odd")
    So.close()


def test_unaligned_vectors_take_the_fallback_paths(cuda):
    """x / y that are only 8-byte aligned: the bulk-copy (TMA) paths that need 16-byte aligned global
    addresses (dia_tma old-y stage, sell_tma x2 window) must fall back to plain loads, not fault."""
    import torch
    A = W.stencil3d_27pt(9, perturb_stream=51)
    x, y0 = W.uniform(111, A.cols), W.uniform(112, A.rows)
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x, 0.5, y0)
    S = binding.SpMV.from_csr(A)
    for desc in ("dia_tma:b288:c256:r1:u9:i3:x0", "dia_tma:b96:c128:r2:u4:i2:x0", "sell_tma:b288:c256:s1:r1:u8:i3:x2:h136",
                 "sell_tma:b160:c256:s1:r2:u4:i3:x0", "dia:b256:c128:r2:u4:x0", "sell:b256:c128:s1:r4:u2:x0",
                 "dia_win:b288:c256:r1:i2:x0", "dia_win:b96:c128:r2:i3:x0", "bcsr3:b256:w8:u1:x0"):
        if not _select_or_skip(S, desc):
            continue
        for xo, yo in ((1, 0), (0, 1), (1, 1)):
            bx = torch.zeros(A.cols + 2, dtype=torch.float64, device="cuda")
            by = torch.zeros(A.rows + 2, dtype=torch.float64, device="cuda")
            dx, dy = bx[xo:xo + A.cols], by[yo:yo + A.rows]
            assert dx.data_ptr() % 16 == 8 * xo and dy.data_ptr() % 16 == 8 * yo
            dx.copy_(torch.from_numpy(x)); dy.copy_(torch.from_numpy(y0))
            S.apply(1.0, dx, 0.5, dy)
            torch.cuda.synchronize()
            ok, mr, ff, nf = oracle.accept(dy.cpu().numpy(), y_ref, scale, H.TOL)
            assert ok, (desc, xo, yo, nf, ff, mr)
            assert float(by[0]) == 0.0 or yo == 0                 # nothing written before the view
            assert float(by[yo + A.rows:].abs().sum()) == 0.0     # nor after it
    S.close()


def test_fuzz_random_matrices_random_variants(cuda):
    """Seeded fuzz: random shapes / row-length laws / orderings x random candidates of the tuner's own
    enumeration (plus the representative list) x random scalars, each against the oracle."""
    rng = np.random.default_rng(2024)
    n_checked = 0
    for trial in range(24):
        rows = int(rng.integers(1, 2500))
        cols = int(rng.integers(1, 2500))
        law = trial % 4
        if law == 0:
            lengths = rng.integers(0, min(cols, 12) + 1, rows)
        elif law == 1:                                               # skewed: a few heavy rows
            lengths = np.minimum((rng.pareto(1.2, rows) * 2).astype(np.int64), cols)
        elif law == 2:                                               # many empty rows
            lengths = np.where(rng.random(rows) < 0.7, 0, rng.integers(1, min(cols, 40) + 1, rows))
        else:                                                        # constant length
            lengths = np.full(rows, int(rng.integers(1, min(cols, 9) + 1)))
        A = W.csr_from_lengths(lengths, cols, 200 + trial, sort=bool(trial % 3))
        x = W.uniform(300 + trial, cols)
        y0 = W.uniform(400 + trial, rows)
        alpha, beta = float(rng.normal()), float(rng.choice([0.0, 1.0, -0.75]))
        y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, alpha, x, beta, y0 if beta != 0.0 else None)
        S = binding.SpMV.from_csr(A)
        cands = S.variants()
        pick = list(rng.choice(cands, size=min(10, len(cands)), replace=False)) + \
            list(rng.choice(H.REPRESENTATIVE_VARIANTS, size=6, replace=False))
        for desc in pick:
            if not _select_or_skip(S, str(desc)):
                continue
            y = H.gpu_apply(S, alpha, x, beta, y0 if beta != 0.0 else None)
            ok, mr, ff, nf = oracle.accept(y, y_ref, scale, H.TOL)
            assert ok, (trial, rows, cols, law, str(desc), nf, ff, mr)
            n_checked += 1
        S.close()
    assert n_checked > 200


def test_fuzz_banded_and_block_matrices(cuda):
    """Seeded fuzz over the structured classes: banded matrices with random width (the tuner then enumerates the
    16-bit index formats and the full-band x window, x3) and 3x3-block FEM matrices (bcsr3 with 32- and 16-bit
    block columns): random candidates of the tuner's own enumeration, preferring those new forms, random scalars,
    non-finite x entries in every other trial, each against the oracle."""
    rng = np.random.default_rng(4242)
    n_checked, n_new = 0, 0
    for trial in range(14):
        if trial % 7 == 6:
            A = W.fem_block27(int(rng.integers(3, 8)), val_stream=500 + trial)
        else:
            rows = int(rng.integers(300, 9000))
            per_row = int(rng.integers(1, 14))
            half = int(rng.integers(per_row + 1, 3000))
            A = W.banded_random(rows, per_row, half, stream=500 + trial)
        x = W.uniform(600 + trial, A.cols)
        if trial % 2:
            x[int(rng.integers(0, A.cols))] = np.nan
            x[int(rng.integers(0, A.cols))] = -np.inf
        y0 = W.uniform(700 + trial, A.rows)
        alpha, beta = float(rng.normal()), float(rng.choice([0.0, 1.0, -0.75]))
        y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, alpha, x, beta, y0 if beta != 0.0 else None)
        S = binding.SpMV.from_csr(A)
        cands = S.variants()
        new = [c for c in cands if ":x3:h" in c or ":i16" in c or c.startswith("sell16")]
        pick = list(rng.choice(new, size=min(12, len(new)), replace=False)) if new else []
        pick += list(rng.choice(cands, size=min(6, len(cands)), replace=False))
        for desc in pick:
            if not _select_or_skip(S, str(desc)):
                continue
            y = H.gpu_apply(S, alpha, x, beta, y0 if beta != 0.0 else None)
            ok, mr, ff, nf = oracle.accept(y, y_ref, scale, H.TOL)
            assert ok, (trial, A.rows, str(desc), nf, ff, mr)
            n_checked += 1
            n_new += str(desc) in new
        S.close()
    assert n_checked > 150 and n_new > 80

"""Full BASELINE.json sizes, in the launch configuration bench.py times: each config is tuned with
the bench's own tuning options and the WINNER's output is compared with the oracle on every row
(the plain-C oracle finishes a full config in under a second, so nothing is sampled), then checked
for bit-identical repeats (north_star).  The fixed default variant is checked on the same inputs."""
import numpy as np
import pytest

import oracle
from paper_1309_1894_b200 import binding
from paper_1309_1894_b200 import workloads as W
from tests import helpers as H

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


def _run(S, prob, dx, dy0):
    import torch
    y = dy0.clone() if dy0 is not None else torch.full((prob.A.rows,), float("nan"), dtype=torch.float64, device=dx.device)
    S.apply(prob.alpha, dx, prob.beta, y)
    torch.cuda.synchronize()
    return y


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_full_size_winner_matches_oracle(cuda, cfg):
    import torch
    prob = W.config(cfg)
    A = prob.A
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, prob.alpha, prob.x, prob.beta, prob.y0)
    S = binding.SpMV.from_csr(A)
    dx = H.to_dev(prob.x)
    dy0 = H.to_dev(prob.y0) if prob.y0 is not None else None
    # the default variant (denominator of the reported speedup)
    ok, mr, ff, nf = oracle.accept(_run(S, prob, dx, dy0).cpu().numpy(), y_ref, scale, H.TOL)
    assert ok, ("default", nf, ff, mr)
    # bench.py's tuning call
    nbytes = W.algorithmic_bytes(A.rows, A.cols, A.nnz, prob.beta)
    warm = nbytes >= 4 * S.info().l2_bytes
    rep = S.tune(alpha=prob.alpha, beta=prob.beta, use_cache=2, flush_l2=not warm, seed=cfg)
    assert rep["n_rejected"] == 0 and rep["winner"] == S.variant
    y1 = _run(S, prob, dx, dy0)
    ok, mr, ff, nf = oracle.accept(y1.cpu().numpy(), y_ref, scale, H.TOL)
    assert ok, (S.variant, nf, ff, mr)
    for _ in range(3):
        assert torch.equal(_run(S, prob, dx, dy0), y1), f"{S.variant} not bit-identical across runs"
    print(f"cfg{cfg}: winner {S.variant} {rep['winner_us']:.1f} us (default {rep['default_us']:.1f} us), "
          f"max err/scale {mr:.2e}")
    S.close()


def test_full_size_cfg5_batch_over_streams(cuda):
    import torch
    probs = [W.config(5, member=m) for m in range(4)]
    hs = [binding.SpMV.from_csr(p.A) for p in probs]
    reps = [h.tune(alpha=1.0, beta=1.0, use_cache=(0 if i else 2), seed=5) for i, h in enumerate(hs)]
    assert all(r["cache_hit"] for r in reps[1:])              # same pattern -> same signature
    xs = [H.to_dev(p.x) for p in probs]
    y0s = [H.to_dev(p.y0) for p in probs]
    ys = [y.clone() for y in y0s]
    streams = [torch.cuda.current_stream()] + [torch.cuda.Stream() for _ in range(3)]
    best, times = binding.tune_batch(hs, [1.0] * 4, xs, [1.0] * 4, ys, streams)
    for y, y0 in zip(ys, y0s):
        y.copy_(y0)
    torch.cuda.synchronize()
    ev = torch.cuda.Event()
    ev.record()
    for s in streams[1:best]:
        s.wait_event(ev)
    binding.apply_batch(hs, [1.0] * 4, xs, [1.0] * 4, ys, streams[:best])
    torch.cuda.synchronize()
    for p, y in zip(probs, ys):
        y_ref, scale = oracle.spmv(p.A.row_ptr, p.A.col_idx, p.A.val, 1.0, p.x, 1.0, p.y0)
        ok, mr, ff, nf = oracle.accept(y.cpu().numpy(), y_ref, scale, H.TOL)
        assert ok, (hs[0].variant, nf, ff, mr)
    print(f"cfg5: winner {hs[0].variant}, streams {best}, batch times {times}")
    for h in hs:
        h.close()


def test_full_size_banded_matrix_16bit_indices(cuda):
    """The bench's banded matrix (2^21 rows, 24 per row within +-2000 of the diagonal): the tuner's winner and the
    best 16-bit-index variant both match the oracle on every row; the 16-bit format streams 10 B per entry."""
    import torch
    A = W.banded_random(1 << 21, 24, 2000)
    x = W.uniform(90, A.cols)
    prob = W.Problem("banded", A, x, None, 1.0, 0.0)
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x, 0.0, parallel=True)
    S = binding.SpMV.from_csr(A)
    dx = H.to_dev(x)
    with pytest.raises(binding.SpmvError):                      # thousands of diagonals: not a DIA matrix
        S.select("dia_tma:b288:c256:r1:u8:i3:x0")
    for flt in (None, "sell16"):
        rep = S.tune(alpha=1.0, beta=0.0, use_cache=2, variant_filter=flt, seed=7)
        assert rep["n_rejected"] == 0
        ok, mr, ff, nf = oracle.accept(_run(S, prob, dx, None).cpu().numpy(), y_ref, scale, H.TOL)
        assert ok, (S.variant, nf, ff, mr)
        print(f"banded: {flt or 'all'} -> {S.variant} {rep['winner_us']:.1f} us, format {S.info().format_bytes / 1e6:.0f} MB")
    assert S.variant.startswith("sell16") and S.info().format_bytes < 10.1 * A.nnz + 16 * A.rows
    # the shared-memory x window (x3: window = the band, double-buffered per slice, no L1 path): every row against
    # the oracle and 25 back-to-back repeats bit for bit (a refill landing under a reader would show up here)
    S.select("sell16_tma:b544:c512:s1:r1:u8:i3:x3:h2000")
    first = _run(S, prob, dx, None).clone()
    ok, mr, ff, nf = oracle.accept(first.cpu().numpy(), y_ref, scale, H.TOL)
    assert ok, (S.variant, nf, ff, mr)
    for _ in range(25):
        assert torch.equal(_run(S, prob, dx, None), first)
    S.close()


@pytest.mark.parametrize("cfg,world", [(4, 2), (3, 3), (5, 2)])
def test_full_size_host_pipeline_and_row_shards(cuda, cfg, world):
    """At BASELINE.json sizes: (i) spmv_apply_host's chunk pipeline equals the device apply bit for bit with the
    tuned variant; (ii) the matrix split into `world` nnz-balanced row shards (loopback transport, one GPU) gives
    the oracle's result on every row, with the halo exchanged through the library's pack / unpack kernels."""
    import torch
    from paper_1309_1894_b200 import sharded
    prob = W.config(cfg)
    A = prob.A
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, prob.alpha, prob.x, prob.beta, prob.y0, parallel=True)
    S = binding.SpMV.from_csr(A)
    S.tune(alpha=prob.alpha, beta=prob.beta, use_cache=0, seed=cfg)
    dx = H.to_dev(prob.x)
    dy0 = H.to_dev(prob.y0) if prob.y0 is not None else None
    y_dev = _run(S, prob, dx, dy0).cpu().numpy()
    xh = torch.from_numpy(prob.x).pin_memory()
    yh = torch.from_numpy((prob.y0 if prob.y0 is not None else np.full(A.rows, np.nan)).copy()).pin_memory()
    S.apply_host(prob.alpha, xh, prob.beta, yh)
    assert np.array_equal(yh.numpy(), y_dev), S.variant
    assert oracle.accept(y_dev, y_ref, scale, H.TOL)[0]
    variant = S.variant
    S.close()
    del dx, dy0
    torch.cuda.empty_cache()
    hub = sharded.LoopbackTransport(world)
    shards = [sharded.ShardedSpMV(A, hub.view(r), align=768) for r in range(world)]
    for sh in shards:
        sh.finish_setup()
        sh.tune(alpha=prob.alpha, beta=prob.beta, use_cache=2, search=1, seed=cfg)
        sh.x_owned.copy_(torch.from_numpy(prob.x[sh.lo:sh.hi]))
    nnz = [sh.nnz_local for sh in shards]
    assert max(nnz) <= 1.05 * A.nnz / world + 20000 * 768       # nnz-balanced up to the alignment
    ys = [(H.to_dev(prob.y0[sh.lo:sh.hi]).clone() if prob.y0 is not None else
           torch.full((sh.rows_local,), float("nan"), dtype=torch.float64, device="cuda")) for sh in shards]
    sharded.run_lockstep(shards, prob.alpha, prob.beta, ys)
    torch.cuda.synchronize()
    y = np.concatenate([t.cpu().numpy() for t in ys])
    ok, mr, ff, nf = oracle.accept(y, y_ref, scale, H.TOL)
    assert ok, (cfg, world, [sh.S.variant for sh in shards], nf, ff, mr)
    print(f"cfg{cfg}: whole {variant}; {world} shards {[sh.S.variant for sh in shards]}, halo {[sh.halo.bytes_received() for sh in shards]} B, "
          f"split {[sh.split for sh in shards]}")
    for sh in shards:
        sh.close()


def test_nnz_near_the_int32_limit(cuda):
    """Maximum sizes: 16 777 216 rows x 127 entries = 2 130 706 432 non-zeros (99.2 % of 2^31-1), built on
    the device from a closed-form pattern.  Values and x are small integers, so every variant must agree
    BITWISE with the oracle, which is evaluated on sampled rows (the same pattern, rebuilt on the host).
    Exercises 64-bit offsets in the kernels and converters; merge-path (rows + nnz over int32) must be refused."""
    import torch
    free, _ = torch.cuda.mem_get_info()
    if free < 90 * 2**30:
        pytest.skip("needs ~80 GB of free device memory")
    rows = cols = 1 << 24
    L = 127
    stride = cols // L
    dev = "cuda:0"
    rp = (torch.arange(rows + 1, dtype=torch.int64, device=dev) * L).to(torch.int32)
    i32 = torch.arange(rows, dtype=torch.int32, device=dev)
    j32 = torch.arange(L, dtype=torch.int32, device=dev)
    ci = (j32[None, :] * stride + (i32 % stride)[:, None]).reshape(-1).contiguous()
    val = (((i32[:, None] + j32[None, :]) % 7) - 3).to(torch.float64).reshape(-1).contiguous()
    assert ci.numel() == rows * L == 2130706432 and int(rp[-1]) == rows * L
    x = ((torch.arange(cols, dtype=torch.int32, device=dev) % 5) - 2).to(torch.float64)
    # oracle on sampled rows: the same closed form on the host, as a small CSR of its own
    rng = np.random.default_rng(7)
    sample = np.unique(np.r_[np.arange(5), rows - 1 - np.arange(5), rng.integers(0, rows, 2000),
                             (np.arange(1, 128) * (1 << 17)) - 1])          # incl. rows around 2^31-byte boundaries
    j = np.arange(L, dtype=np.int64)
    s_ci = (j[None, :] * stride + (sample % stride)[:, None]).astype(np.int32).reshape(-1)
    s_val = (((sample[:, None] + j[None, :]) % 7) - 3).astype(np.float64).reshape(-1)
    s_rp = (np.arange(sample.size + 1) * L).astype(np.int32)
    xh = ((np.arange(cols) % 5) - 2).astype(np.float64)
    y0_s = (sample % 3).astype(np.float64)
    y_ref, _ = oracle.spmv(s_rp, s_ci, s_val, 2.0, xh, -1.0, y0_s)
    assert np.array_equal(ci[torch.from_numpy(sample[:3] * L).to(dev)].cpu().numpy(), s_ci[::L][:3])
    S = binding.SpMV(rows, cols, rp, ci, val)
    info = S.info()
    assert info.nnz == rows * L and info.min_row_len == info.max_row_len == L and info.cols_sorted == 1
    with pytest.raises(binding.SpmvError) as e:
        S.select("merge:b256:i7:x0")
    assert e.value.status == 3
    y0 = (torch.arange(rows, dtype=torch.int32, device=dev) % 3).to(torch.float64)
    idx = torch.from_numpy(sample).to(dev)
    for desc in ("default", "csr_vector:b256:w32:u4:x0", "sell:b256:c128:s1:r2:u4:x0", "sell_tma:b288:c256:s1:r1:u16:i2:x0"):
        S.select(desc)
        y = y0.clone()
        S.apply(2.0, x, -1.0, y)
        torch.cuda.synchronize()
        got = y[idx].cpu().numpy()
        assert np.array_equal(got, y_ref), (desc, np.flatnonzero(got != y_ref)[:5])
        assert bool(torch.isfinite(y).all()) and float(y.abs().max()) <= 2.0 * 6 * L + 2
    S.close()

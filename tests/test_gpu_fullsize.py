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

"""Small driver for ncu / compute-sanitizer: a few applies of one variant on one config.

    python -m paper_1309_1894_b200.prof --cfg 2 [--scale 1.0] [--variant DESC | --tune] [--iters 5]

Prints the time per apply (CUDA events, L2 flushed before each) so the same command can be
run plain first and under ncu afterwards (numbers printed under ncu are not bench values).
"""
import argparse

import numpy as np
import torch

from . import binding, workloads as W


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cfg", type=int, default=2)
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--variant", default="default")
    ap.add_argument("--tune", action="store_true")
    ap.add_argument("--iters", type=int, default=5)
    ap.add_argument("--no-flush", action="store_true")
    a = ap.parse_args()
    prob = W.config(a.cfg, a.scale)
    A = prob.A
    S = binding.SpMV.from_csr(A)
    x = torch.from_numpy(prob.x).cuda()
    y0 = torch.from_numpy(prob.y0 if prob.y0 is not None else np.zeros(A.rows)).cuda()
    y = y0.clone()
    if a.tune:
        rep = S.tune(alpha=prob.alpha, beta=prob.beta, use_cache=2, flush_l2=not a.no_flush)
        print("tuned:", rep["winner"], rep["winner_us"], "us; default", rep["default_us"], "us")
    else:
        S.select(a.variant)
    flush = torch.empty(int(2 * S.info().l2_bytes // 8), dtype=torch.float64, device="cuda")
    ts = []
    for _ in range(a.iters):
        if not a.no_flush:
            flush.fill_(1.0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        S.apply(prob.alpha, x, prob.beta, y)
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1) * 1e3)
    nb = W.algorithmic_bytes(A.rows, A.cols, A.nnz, prob.beta)
    t = float(np.median(ts))
    print(f"{prob.name} | {S.variant} | {t:.2f} us/apply | {nb / t / 1e3:.1f} GB/s effective | "
          f"format bytes {S.info().format_bytes}")
    S.close()


if __name__ == "__main__":
    main()

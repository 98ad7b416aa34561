"""Driver for the compute-sanitizer passes (SURVEY.md sec. 4 T7, sec. 5 "Race detection / sanitizers"); not a test.

    compute-sanitizer --tool memcheck   python -m tests.sanitizer_zoo
    compute-sanitizer --tool initcheck  python -m tests.sanitizer_zoo
    compute-sanitizer --tool synccheck  python -m tests.sanitizer_zoo --subset smem
    compute-sanitizer --tool racecheck  python -m tests.sanitizer_zoo --subset smem

Runs the small test zoo (tests/helpers.py) through every representative variant that is eligible for each matrix --
conversion kernels, one apply with beta != 0 and one with beta == 0, checked against oracle/ -- then the row-range
apply, the host-vector pipeline, the CG loops (fused single kernel and graph form), the Jacobi loop, one short tune and
the no-allocation entry point.  `--subset smem` keeps the kernels that stage data in shared memory or synchronise
through mbarriers (sell_tma x0/x2/x3, sell16_tma, dia_tma, dia_win, dia_cwin, merge, row-split fix-ups, bcsr3) on a
few matrices: racecheck and synccheck are an order of magnitude slower.  Prints one summary line; the sanitizer's own
report goes where --log-file says.

Round 3: the GPU pool this repository is built on refuses compute-sanitizer ("closed on this pool": runs under it left
GPUs needing a reset), so no sanitizer report is committed; DESIGN.md sec. 8 records that.  Run plainly
(`python -m tests.sanitizer_zoo`) the driver is still a sweep of every kernel family against the oracle."""
import argparse
import sys

import numpy as np
import torch

import oracle
from paper_1309_1894_b200 import binding, workloads as W
from tests import helpers as H

SMEM_FAMILIES = ("sell_tma", "sell16_tma", "dia_tma", "dia_win", "dia_cwin", "merge", "bcsr3", "dia_const")
SMEM_MATRICES = ("lap3d_11", "st27_9", "fem_5", "powerlaw_3k", "banded_4k", "lengths_ladder", "empty_rows_runs")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--subset", default="all", choices=["all", "smem"])
    args = ap.parse_args()
    smem = args.subset == "smem"
    n_apply = n_var = 0
    kernels = set()
    for name, A in H.zoo():
        if smem and name not in SMEM_MATRICES:
            continue
        rng = np.random.default_rng(abs(hash(name)) % 1000)
        x = rng.uniform(-1, 1, A.cols)
        y0 = rng.uniform(-1, 1, A.rows)
        S = binding.SpMV.from_csr(A)
        eligible = set(S.variants())
        eligible_fams = {v.split(":")[0] for v in eligible}
        for desc in H.REPRESENTATIVE_VARIANTS:
            fam = desc.split(":")[0]
            if smem and not (fam in SMEM_FAMILIES or ":l" in desc):
                continue
            try:
                S.select(desc)
            except binding.SpmvError as e:
                if e.status in (1, 3):          # not eligible for this matrix
                    continue
                raise
            n_var += 1
            kernels.add(fam + (":split" if ":l" in desc else "") + (":x%s" % desc.split(":x")[1][0] if ":x" in desc else ""))
            for alpha, beta, yy in ((1.25, -0.5, y0), (1.0, 0.0, None)):
                H.check_against_oracle(S, A, alpha, x, beta, yy, what=f"{name}")
                n_apply += 1
        # row-range form and the host-vector pipeline of one range-capable variant
        range_ok = A.rows >= 256 and "sell" in eligible_fams
        if range_ok:
            try:
                S.select("sell:b256:c128:s1:r1:u1:x0")
            except binding.SpmvError as e:      # e.g. the built format is too padded to keep
                if e.status != 3:
                    raise
                range_ok = False
        if range_ok:
            al = S.range_align()
            mid = (A.rows // 2) // al * al
            dx, dy = H.to_dev(x), H.to_dev(y0).clone()
            S.apply_rows(1.0, dx, 0.5, dy, 0, mid)
            S.apply_rows(1.0, dx, 0.5, dy, mid, A.rows)
            torch.cuda.synchronize()
            y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x, 0.5, y0)
            assert oracle.accept(dy.cpu().numpy(), y_ref, scale, H.TOL)[0]
            xh, yh = torch.from_numpy(x).pin_memory(), torch.from_numpy(y0.copy()).pin_memory()
            S.apply_host(1.0, xh, 0.5, yh)
            assert oracle.accept(yh.numpy(), y_ref, scale, H.TOL)[0]
            kernels.update(("apply_rows", "apply_host"))
        S.close()
    # solver loops, tuner and the no-allocation entry point on small SPD systems
    for A, tag in ((W.laplace2d_5pt(24), "lap2d"), (W.laplace3d_7pt(12), "lap3d")):
        S = binding.SpMV.from_csr(A)
        b = H.to_dev(W.uniform(5, A.rows))
        for sel, kw in (("dia_const:b256:r1:x0", {}), ("dia_const:b256:r1:x0", {"no_fused": True}),
                        ("sell:b256:c128:s1:r1:u1:x0", {"no_fused": True, "no_graph": True})):
            S.select(sel)
            xs = torch.zeros(A.rows, dtype=torch.float64, device="cuda:0")
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                r = S.cg(b, xs, tol=1e-8, max_iters=200, **kw)
                st.synchronize()
            assert r["converged"], (tag, sel, kw, r)
            xs.zero_()
            with torch.cuda.stream(st):
                r = S.jacobi(b, xs, omega=0.8, tol=1e-3, max_iters=400, no_fused=bool(kw.get("no_fused")))
                st.synchronize()
        kernels.update(("cg_fused", "cg_graph", "cg_plain", "jacobi_fused", "jacobi"))
        if not smem:
            S.tune(alpha=1.0, beta=0.5, use_cache=2, reps=1, min_batch_ms=0.01, search=1)
            kernels.add("tuner(search=1)")
        S.close()
    A = W.powerlaw(3000, lmax=2500)
    d = [H.to_dev(a) for a in (A.row_ptr, A.col_idx, A.val)]
    x = W.uniform(8, A.cols)
    dy = torch.zeros(A.rows, dtype=torch.float64, device="cuda:0")
    for _ in range(2):
        binding.merge_apply_noalloc(A.rows, A.cols, *d, 1.0, H.to_dev(x), 0.0, dy)
    torch.cuda.synchronize()
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x, 0.0, None)
    assert oracle.accept(dy.cpu().numpy(), y_ref, scale, H.TOL)[0]
    kernels.add("merge_apply_noalloc")
    print(f"sanitizer_zoo[{args.subset}]: {n_var} (matrix, variant) selections, {n_apply} applies checked against the oracle; "
          f"covered: {', '.join(sorted(kernels))}")
    return 0


if __name__ == "__main__":
    sys.exit(main())

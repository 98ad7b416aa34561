"""Failure paths of the handle: after an allocation failure in the middle of
spmv_tune / spmv_select / spmv_update_values the next spmv_apply must still be correct (never a launch plan that points
into released formats); a cached tuning winner is verified before it is adopted; x and y may not alias."""
import ctypes
import json
import os
import subprocess
import sys

import numpy as np
import pytest

import oracle
from paper_1309_1894_b200 import binding, workloads as W
from tests import helpers as H

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ---------------------------------------------------------------------------------------------------------------
# scenario runner (own process: a use-after-free on the device would leave a sticky CUDA error behind)
# ---------------------------------------------------------------------------------------------------------------
def _cudart():
    import torch  # noqa: F401  (loads libcudart into the process)
    for name in ("libcudart.so.12", "libcudart.so"):
        try:
            return ctypes.CDLL(name)
        except OSError:
            continue
    libdir = os.path.join(os.path.dirname(__import__("torch").__file__), "lib")
    for f in sorted(os.listdir(libdir)):
        if f.startswith("libcudart"):
            return ctypes.CDLL(os.path.join(libdir, f))
    raise RuntimeError("libcudart not found")


class FailingAllocator:
    """spmv_allocator_t over torch's caching allocator that (a) refuses every request once `fail_after` further
    requests have been served and (b) overwrites a block with 0xFF bytes before giving it back, so that a kernel
    still reading a released format computes garbage (NaN values, -1 indices) instead of the old, still intact data."""

    def __init__(self):
        import torch
        self.torch = torch
        self.rt = _cudart()
        self.rt.cudaMemset.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t]
        self.live = {}
        self.budget = None            # None: unlimited
        self.refused = 0
        self.struct = binding.Allocator(binding.ALLOC_FN(self._alloc), binding.FREE_FN(self._free), None)

    def _alloc(self, nbytes, stream, ctx):
        if self.budget is not None:
            if self.budget <= 0:
                self.refused += 1
                return 0
            self.budget -= 1
        try:
            p = self.torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream or 0))
        except Exception:
            return 0
        self.live[p] = int(nbytes)
        return p

    def _free(self, ptr, ctx):
        n = self.live.pop(int(ptr), 0)
        if n:
            self.torch.cuda.synchronize()
            self.rt.cudaMemset(ctypes.c_void_p(int(ptr)), 0xFF, n)
            self.torch.cuda.synchronize()
        self.torch.cuda.caching_allocator_delete(int(ptr))


def _scenarios():
    import torch
    out = []
    A = W.fem_block27(6)                      # 3x3 blocks: bcsr3 (both index widths), sell, merge, csr all eligible
    rng = np.random.default_rng(11)
    x = rng.uniform(-1, 1, A.cols)
    y0 = rng.uniform(-1, 1, A.rows)
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x, 0.5, y0)
    dx = H.to_dev(x)

    def apply_ok(S):
        dy = H.to_dev(y0).clone()
        S.apply(1.0, dx, 0.5, dy)
        torch.cuda.synchronize()
        ok, mr, ff, nf = oracle.accept(dy.cpu().numpy(), y_ref, scale, H.TOL)
        return bool(ok), float(mr) if np.isfinite(mr) else -1.0, int(nf)

    starts = ["sell:b256:c128:s1:r1:u1:x0", "bcsr3:b128:w8:u2:i16:x0", "merge:b256:i7:x0", "sell_tma:b288:c256:s1:r1:u8:i3:x0"]
    for start in starts:
        for budget in (0, 1, 2, 4, 7, 12, 25, 60):
            al = FailingAllocator()
            S = binding.SpMV.from_csr(A, allocator=al.struct)
            S.select(start)
            rec = {"op": "tune", "start": start, "budget": budget, "before": apply_ok(S)}
            al.budget = budget
            try:
                S.tune(alpha=1.0, beta=0.5, use_cache=2, reps=1, min_batch_ms=0.02)
                rec["status"] = "ok"
            except binding.SpmvError as e:
                rec["status"] = binding.STATUS_NAMES[e.status]
            al.budget = None
            rec["refused"] = al.refused
            rec["variant_after"] = S.variant
            rec["after"] = apply_ok(S)
            S.close()
            out.append(rec)
    # select of another family fails half-way: the previous selection stays usable
    for start, target in (("bcsr3:b128:w8:u2:i16:x0", "bcsr3:b256:w4:u1:x0"), ("sell:b256:c128:s1:r1:u1:x0", "bcsr3:b128:w8:u2:i16:x0"),
                          ("bcsr3:b256:w4:u1:x0", "sell16:b256:c128:s1:r1:u2:x0")):
        for budget in (0, 1, 2, 3, 5):
            al = FailingAllocator()
            S = binding.SpMV.from_csr(A, allocator=al.struct)
            S.select(start)
            al.budget = budget
            rec = {"op": "select", "start": start, "target": target, "budget": budget}
            try:
                S.select(target)
                rec["status"] = "ok"
            except binding.SpmvError as e:
                rec["status"] = binding.STATUS_NAMES[e.status]
            al.budget = None
            rec["refused"] = al.refused
            rec["variant_after"] = S.variant
            rec["after"] = apply_ok(S)
            S.close()
            out.append(rec)
    # update_values with a failing allocator: every format is rebuilt from the new values
    val2 = torch.from_numpy(A.val * 1.0).cuda()
    for start in ("bcsr3:b128:w8:u2:i16:x0", "sell:b256:c128:s1:r1:u1:x0", "merge:b256:i7:x0"):
        for budget in (0, 1, 2, 4):
            al = FailingAllocator()
            S = binding.SpMV.from_csr(A, allocator=al.struct)
            S.select(start)
            al.budget = budget
            rec = {"op": "update_values", "start": start, "budget": budget}
            try:
                S.update_values(val2)
                rec["status"] = "ok"
            except binding.SpmvError as e:
                rec["status"] = binding.STATUS_NAMES[e.status]
            al.budget = None
            rec["refused"] = al.refused
            rec["variant_after"] = S.variant
            rec["after"] = apply_ok(S)
            S.close()
            out.append(rec)
    return out


if __name__ == "__main__":
    print("SCENARIOS " + json.dumps(_scenarios()))
    sys.exit(0)


def test_apply_is_correct_after_an_allocation_failure_anywhere(cuda):
    r = subprocess.run([sys.executable, "-m", "tests.test_gpu_robustness"], cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, (r.stdout[-1500:], r.stderr[-3000:])
    recs = json.loads([l for l in r.stdout.splitlines() if l.startswith("SCENARIOS ")][-1][len("SCENARIOS "):])
    assert len(recs) >= 50
    failed = [x for x in recs if x["status"] != "ok"]
    assert len(failed) >= 10, "the failing allocator never made an operation fail: the scenarios test nothing"
    assert any(x["op"] == "tune" for x in failed) and any(x["op"] == "select" for x in failed) and any(x["op"] == "update_values" for x in failed)
    for x in recs:
        assert x["after"][0], f"apply after {x['op']} ({x['status']}, {x['refused']} refusals) is wrong: {x}"
        if x["status"] == "SPMV_ERR_ALLOC":
            assert x["refused"] > 0


def test_cached_winner_is_verified_before_it_is_adopted(cuda, tmp_path):
    """A cache file that names an eligible variant which computes wrong results (fault injection stands in for a stale
    or hand-edited entry): the hit is verified, rejected, and the full search picks something else."""
    A = W.laplace3d_7pt(24)
    S = binding.SpMV.from_csr(A)
    path = str(tmp_path / "tune.cache")
    binding.clear_cache()
    r1 = S.tune(use_cache=0, cache_path=path, reps=1, min_batch_ms=0.02, variant_filter="csr_vector,sell:")
    assert not r1["cache_hit"]
    key = open(path).read().split()[0]
    fam = r1["winner"].split(":")[0]
    # a clean second handle: the entry is verified and adopted
    binding.clear_cache()
    S2 = binding.SpMV.from_csr(A)
    r2 = S2.tune(use_cache=0, cache_path=path, reps=1, min_batch_ms=0.02, variant_filter="csr_vector,sell:")
    assert r2["cache_hit"] and r2["winner"] == r1["winner"]
    assert any(l[1] == "cache_hit_verified" for l in r2["log"])
    # the same entry, but that family now computes garbage: rejected, searched again, another family wins
    binding.clear_cache()
    S3 = binding.SpMV.from_csr(A)
    r3 = S3.tune(use_cache=0, cache_path=path, reps=1, min_batch_ms=0.02, variant_filter="csr_vector,sell:", fault_inject=fam)
    assert not r3["cache_hit"]
    assert any(l[1] == "cache_entry_rejected" and l[0] == r1["winner"] for l in r3["log"])
    assert r3["winner"].split(":")[0] != fam and r3["n_rejected"] > 0
    x = W.uniform(3, A.cols)
    H.check_against_oracle(S3, A, 1.0, x, 0.0, None, what="after a rejected cache entry")
    # a hand-written line naming an ineligible / unparsable variant is ignored
    with open(path, "a") as f:
        f.write(f"{key} bcsr3:b128:w8:u2:x0 1.0\n{key} nonsense:b1 1.0\n")
    binding.clear_cache()
    S4 = binding.SpMV.from_csr(A)
    r4 = S4.tune(use_cache=0, cache_path=path, reps=1, min_batch_ms=0.02, variant_filter="csr_vector,sell:")
    assert r4["winner"].split(":")[0] in ("csr_vector", "sell")
    for s in (S, S2, S3, S4):
        s.close()


def test_apply_rejects_aliased_vectors(cuda):
    import torch
    A = W.laplace2d_5pt(16)
    S = binding.SpMV.from_csr(A)
    v = torch.ones(A.rows, dtype=torch.float64, device="cuda:0")
    with pytest.raises(binding.SpmvError) as e:
        S.apply(1.0, v, 0.0, v)
    assert e.value.status == 1 and "alias" in str(e.value)
    S.apply(0.0, v, 2.0, v)            # alpha == 0: x is not referenced, y = beta*y
    torch.cuda.synchronize()
    assert torch.equal(v, torch.full_like(v, 2.0))
    S.close()


@pytest.mark.parametrize("variant", ["merge:b256:i7:x0", "sell:b256:c128:s8192:l16:r2:u2:x0"])
def test_workspace_variants_are_ordered_across_streams(cuda, variant):
    """merge-path and row-split SELL own ONE workspace per handle.  Applies of one handle enqueued on two streams with
    nothing between them used to be the caller's problem (their kernels overlap and mix their carries); the library
    now chains them through an event.  Different x per stream, many rounds, every result against the oracle."""
    import torch
    A = W.powerlaw(400000, lmax=20000)
    S = binding.SpMV.from_csr(A)
    S.select(variant)
    xs = [W.uniform(70 + i, A.cols) for i in range(2)]
    dxs = [H.to_dev(x) for x in xs]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    dys = [torch.full((A.rows,), float("nan"), dtype=torch.float64, device="cuda:0") for _ in range(2)]
    torch.cuda.synchronize()
    for _ in range(25):
        for i in (0, 1):
            S.apply(1.0, dxs[i], 0.0, dys[i], stream=streams[i])
    torch.cuda.synchronize()
    for i in (0, 1):
        y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, xs[i], 0.0, None, parallel=True)
        ok, mr, ff, nf = oracle.accept(dys[i].cpu().numpy(), y_ref, scale, H.TOL)
        assert ok, f"{variant} stream {i}: {nf} rows wrong, first {ff}, max err/scale {mr:.3e}"
    # a graph captured from such a variant still works (no event is touched inside the capture)
    g = S.graph(1.0, dxs[0], 0.0, dys[0], 3)
    g.launch()
    torch.cuda.synchronize()
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, xs[0], 0.0, None, parallel=True)
    assert oracle.accept(dys[0].cpu().numpy(), y_ref, scale, H.TOL)[0]
    g.close()
    S.close()

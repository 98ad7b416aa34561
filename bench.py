#!/usr/bin/env python
"""bench.py -- fp64 SpMV effective GB/s & fraction of B200 HBM peak (autotuned vs default).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--configs 2[,1,3,4,5]] [--impl reference]

One "step" is one pass of the hot path, y = alpha*A*x + beta*y through spmv_apply with the
autotuned variant, on BASELINE.json:configs[1] (cfg2: 3D 7-point Laplacian 128^3, alpha=1,
beta=0.5), inputs resident in HBM.  Cold-cache protocol: the steps rotate over several device
copies of the inputs (combined footprint > 3x the 126 MB L2), run back to back and are bracketed
by one CUDA event pair on the launching stream (cfg1 is too small for that: L2 flush per step).  `value` = algorithmic bytes (nnz*12 + (rows+1)*4 + 8*cols + 8*rows
[+ 8*rows if beta != 0]) / time, whole job.  `e2e` is the same metric through spmv_apply_host
with pinned HOST vectors (H2D of x and y, apply, D2H of y inside the timed region).
N > 1: N independent replicas (the path is single-GPU; "replicas only"),
barrier + max over ranks, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "fp64 SpMV effective GB/s & fraction of B200 HBM peak (autotuned vs default)"
NOMINAL_HBM_GBS = 8000.0      # BASELINE.json:north_star "~8 TB/s"
FALLBACK_HBM_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md fallback


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(variant: str, cfg: int):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture, or None."""
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
        e = t.get(f"cfg{cfg}", {})
        # the capture is of one instantiation of the family; DRAM traffic is a property of the format
        return e.get("dram_bytes_per_launch") if e.get("variant", "").split(":")[0] == variant.split(":")[0] else None
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [q.strip() for q in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def cpu_oracle_times(prob, reps=5):
    """The oracle as it stands on the host cores: serial and row-parallel (bit-identical)."""
    import oracle
    A = prob.A
    rp = np.ascontiguousarray(A.row_ptr, dtype=np.int32)
    ci = np.ascontiguousarray(A.col_idx, dtype=np.int32)
    va = np.ascontiguousarray(A.val, dtype=np.float64)
    x = np.ascontiguousarray(prob.x)
    y0 = prob.y0 if prob.y0 is not None else np.zeros(A.rows)
    scale = np.empty(A.rows)
    out = {}
    for par in (False, True):
        ts, threads = [], 1
        for i in range(reps + 1):
            y = y0.copy()
            t0 = time.perf_counter()
            threads = oracle.spmv_inplace(rp, ci, va, prob.alpha, x, prob.beta, y, scale, parallel=par)
            ts.append(time.perf_counter() - t0)
        out["parallel" if par else "serial"] = (float(np.median(ts[1:])), int(threads))
    return out


def run_reference(args, W):
    """--impl reference: the oracle (row-parallel form of the same loop) on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cfg = int(args.configs.split(",")[0])
    prob = W.config(cfg)
    A = prob.A
    nbytes = W.algorithmic_bytes(A.rows, A.cols, A.nnz, prob.beta)
    rp, ci, va = (np.ascontiguousarray(A.row_ptr), np.ascontiguousarray(A.col_idx), np.ascontiguousarray(A.val))
    y0 = prob.y0 if prob.y0 is not None else np.zeros(A.rows)
    scale = np.empty(A.rows)
    y = y0.copy()
    threads = 1
    steps = min(args.steps, 50)          # bounded sample: at most 50 full applies
    for _ in range(min(args.warmup, 3)):
        threads = oracle.spmv_inplace(rp, ci, va, prob.alpha, prob.x, prob.beta, y, scale, parallel=True)
    t0 = time.perf_counter()
    for _ in range(steps):
        threads = oracle.spmv_inplace(rp, ci, va, prob.alpha, prob.x, prob.beta, y, scale, parallel=True)
    dt = (time.perf_counter() - t0) / steps
    gbs = nbytes / dt / 1e9
    sample = f"{steps} full applies of {prob.name} (whole matrix, {A.nnz} nnz)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": gbs, "unit": "GB/s", "n_gpus": args.gpus,
        "steps": steps, "warmup": min(args.warmup, 3), "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": prob.name, "rows": A.rows, "nnz": A.nnz},
        "cpu_baseline": {"value": gbs, "unit": "GB/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": gbs, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gflops": 2.0 * A.nnz / dt / 1e9,
    }))


def bench_config(cfg, args, torch, binding, W, dist_max, device, primary):
    """Tune + time one config on this rank; returns a result dict."""
    members = 4 if cfg == 5 else 1
    probs = [W.config(cfg, member=m) for m in range(members)]
    A0 = probs[0].A
    alpha, beta = probs[0].alpha, probs[0].beta
    nbytes = sum(W.algorithmic_bytes(p.A.rows, p.A.cols, p.A.nnz, p.beta) for p in probs)
    nnz = sum(p.A.nnz for p in probs)
    l2 = torch.cuda.get_device_properties(device).L2_cache_size
    # Cold-cache protocol (timing rules: "flush L2 or use inputs larger than L2"):
    #  rotate: the step cycles through `copies` independent device copies of the inputs whose
    #          combined footprint exceeds 3x L2, so every apply streams its matrix from HBM and
    #          the K steps run back to back inside ONE event pair;
    #  flush : (cfg1, 0.3 MB) a 2xL2 buffer is overwritten before every step, per-step events.
    #  warm  : working set >> L2 already (cfg3-5), K steps back to back.
    if nbytes >= 4 * l2:
        mode, copies = "warm", 1
    elif nbytes * 16 >= 3 * l2:
        mode, copies = "rotate", int(np.ceil(3 * l2 / nbytes)) + 1
    else:
        mode, copies = "flush", 1
    handles, xs, ys, y0s = [], [], [], []
    for c in range(copies):
        for p in probs:
            handles.append(binding.SpMV.from_csr(p.A, device=device))
            xs.append(torch.from_numpy(p.x).to(device))
            y0 = p.y0 if p.y0 is not None else np.zeros(p.A.rows)
            y0s.append(torch.from_numpy(y0).to(device))
            ys.append(y0s[-1].clone())
    flush = torch.empty(int(2 * l2 // 8), dtype=torch.float64, device=device) if mode == "flush" else None
    step_no = [0]

    def one_step():
        if members == 1:
            i = step_no[0] % copies
            step_no[0] += 1
            handles[i].apply(alpha, xs[i], beta, ys[i])
        else:
            binding.apply_batch(handles, [alpha] * members, xs, [beta] * members, ys, streams[:nstreams])

    def fork_join_step(ev):
        for s in streams[1:nstreams]:
            s.wait_event(ev)
        one_step()
        for s in streams[1:nstreams]:
            j = torch.cuda.Event()
            j.record(s)
            torch.cuda.current_stream().wait_event(j)

    def timed(steps, warmup):
        """returns (total seconds, median seconds per step, min seconds per step)"""
        for _ in range(warmup):
            one_step()
        torch.cuda.synchronize()
        if mode == "flush":
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
            for a, b in evs:
                flush.fill_(1.0)
                a.record()
                one_step()
                b.record()
            torch.cuda.synchronize()
            ts = np.array([a.elapsed_time(b) for a, b in evs]) * 1e-3
            return float(ts.sum()), float(np.median(ts)), float(ts.min())
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(steps):
            if members > 1:
                fork_join_step(a)
            else:
                one_step()
        b.record()
        torch.cuda.synchronize()
        t = a.elapsed_time(b) * 1e-3
        return t, t / steps, t / steps

    # ---- default variant, then tune (tuning is setup, outside the timed region)
    streams, nstreams = [torch.cuda.current_stream()], 1
    tsum_d, tmed_d, _ = timed(max(10, args.steps // 10), 3)
    # second fixed baseline (SURVEY A17 "heuristic default"): sub-warp width = smallest power of two >= mean row length
    mean_len = handles[0].info().mean_row_len
    w_h = int(min(32, max(2, 2 ** int(np.ceil(np.log2(max(mean_len, 1.0)))))))
    heuristic = f"csr_vector:b256:w{w_h}:u1:x0"
    for h in handles:
        h.select(heuristic)
    _, tmed_h, _ = timed(max(10, args.steps // 10), 3)
    t0 = time.perf_counter()
    reports = [h.tune(alpha=alpha, beta=beta, use_cache=(0 if (i or args.tune_cache) else 2),
                      cache_path=args.tune_cache, flush_l2=(mode != "warm"), seed=cfg,
                      variant_filter=args.variant_filter)
               for i, h in enumerate(handles)]
    stream_times = {}
    if members > 1:
        streams = [torch.cuda.current_stream()] + [torch.cuda.Stream(device=device) for _ in range(3)]
        nstreams, stream_times = binding.tune_batch(handles, [alpha] * members, xs, [beta] * members, ys, streams)
    tune_s = time.perf_counter() - t0
    variant = handles[0].variant
    # merge-path and row-split SELL add one small ordered fix-up kernel per apply
    launches_per_step = members * (2 if (variant.startswith("merge") or ":l" in variant) else 1)
    for y, y0 in zip(ys, y0s):
        y.copy_(y0)

    # ---- the timed region: barrier + sync on both sides, max over ranks
    sampler = ClockSampler(torch.cuda.current_device()) if primary else None
    for _ in range(args.warmup):
        one_step()
    torch.cuda.synchronize()
    dist_max(0.0)                               # barrier
    tsum, tmed, tmin = timed(args.steps, 0)
    tsum = dist_max(tsum)
    # keep the GPU under the same load a little longer so the clock sampler sees it
    if sampler is not None:
        t_end = time.time() + 0.6
        while time.time() < t_end:
            for _ in range(50):
                one_step()
            torch.cuda.synchronize()
    clocks = sampler.stop() if sampler is not None else None

    # ---- the other cache state: warm (same buffers back to back) for the configs whose headline is cold
    t_warm_us = None
    if mode != "warm" and members == 1:
        for _ in range(5):
            handles[0].apply(alpha, xs[0], beta, ys[0])
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(args.steps):
            handles[0].apply(alpha, xs[0], beta, ys[0])
        b.record()
        torch.cuda.synchronize()
        t_warm_us = a.elapsed_time(b) * 1e3 / args.steps

    # ---- parity of what was just timed (sampled rows through the oracle would need the CPU
    # oracle; the full check lives in tests/ -- here: determinism + finite output)
    def first_members():
        for y, y0 in zip(ys[:members], y0s[:members]):
            y.copy_(y0)
        if members == 1:
            handles[0].apply(alpha, xs[0], beta, ys[0])
        else:
            binding.apply_batch(handles, [alpha] * members, xs, [beta] * members, ys, streams[:1])
        torch.cuda.synchronize()
        return [y.clone() for y in ys[:members]]
    first = first_members()
    deterministic = all(torch.equal(a, b) for a, b in zip(first, first_members()))
    finite = all(bool(torch.isfinite(y).all()) for y in ys)

    # ---- e2e through spmv_apply_host with pinned host vectors
    e2e = None
    if members == 1:
        xh = torch.from_numpy(probs[0].x).pin_memory()
        yh = torch.from_numpy((probs[0].y0 if probs[0].y0 is not None else np.zeros(A0.rows)).copy()).pin_memory()
        for _ in range(3):
            handles[0].apply_host(alpha, xh, beta, yh)
        n_e2e = max(5, min(args.steps, 50))
        torch.cuda.synchronize(); dist_max(0.0)
        t1 = time.perf_counter()
        for _ in range(n_e2e):
            handles[0].apply_host(alpha, xh, beta, yh)      # synchronises the stream itself
        te = dist_max((time.perf_counter() - t1) / n_e2e)
        e2e = {"value": nbytes / te / 1e9, "unit": "GB/s", "ms_per_step": te * 1e3, "steps": n_e2e,
               "h2d_bytes_per_step": 8 * A0.cols + (8 * A0.rows if beta != 0 else 0),
               "d2h_bytes_per_step": 8 * A0.rows}
    # ---- solver loop around apply: fixed-count CG on the SPD configs
    cg = None
    if cfg in (1, 2) and members == 1:
        st = torch.cuda.Stream(device=device)
        with torch.cuda.stream(st):
            bvec = torch.zeros(A0.rows, dtype=torch.float64, device=device)
            handles[0].apply(1.0, xs[0], 0.0, bvec)                  # b = A x_true
            n_it = 200
            best = None
            for _ in range(3):
                xg = torch.zeros(A0.rows, dtype=torch.float64, device=device)
                r = handles[0].cg(bvec, xg, tol=1e-300, max_iters=n_it, check_every=25)
                if best is None or r["device_seconds"] < best["device_seconds"]:
                    best = r
            st.synchronize()
        # per iteration: one SpMV (algorithmic bytes with beta = 0) + dot (16 B/row) + x/r update (48) + p update (24)
        it_bytes = W.algorithmic_bytes(A0.rows, A0.cols, A0.nnz, 0.0) + 88 * A0.rows
        cg = {"iters": best["iters"], "us_per_iteration": best["device_seconds"] / max(best["iters"], 1) * 1e6,
              "eff_gbs": it_bytes * best["iters"] / best["device_seconds"] / 1e9,
              "rel_residual": best["rel_residual"], "graph_replays": best["graph_replays"],
              "fused_single_kernel": bool(best["fused"]),
              "launches_per_iteration": 0 if best["fused"] else 4 + launches_per_step,
              "bytes_per_iteration_algorithmic": it_bytes}
    info = handles[0].info()
    peak_meas, _ = measured_peak()
    eff = nbytes * args.steps / tsum / 1e9
    res = {"cfg": cfg, "workload": probs[0].name if members == 1 else W.CONFIG_NAMES[5],
           "rows": A0.rows, "cols": A0.cols, "nnz": nnz, "members": members,
           "bytes_algorithmic": nbytes, "bytes_format_actual": int(sum(h.info().format_bytes for h in handles[:members])),
           "variant": variant, "nstreams": nstreams, "stream_times_us": stream_times,
           "t_sum_s": tsum, "t_median_us": tmed * 1e6, "t_min_us": tmin * 1e6,
           "eff_gbs": eff, "frac_hbm_nominal_8TBs": eff / NOMINAL_HBM_GBS, "frac_hbm_measured": eff / peak_meas,
           "bytes_actual": int(sum(h.info().format_bytes for h in handles[:members]) +
                               sum(8 * p.A.cols + 8 * p.A.rows * (2 if p.beta != 0 else 1) for p in probs)),
           "format_gbs": float(sum(h.info().format_bytes for h in handles[:members]) +
                               sum(8 * p.A.cols + 8 * p.A.rows * (2 if p.beta != 0 else 1) for p in probs))
                         * args.steps / tsum / 1e9,
           "gathers_per_s": nnz * args.steps / tsum, "gflops": 2.0 * nnz * args.steps / tsum / 1e9,
           "t_default_us": tmed_d * 1e6, "speedup_vs_default": tmed_d / tmed,
           "heuristic_variant": heuristic, "t_heuristic_us": tmed_h * 1e6, "speedup_vs_heuristic": tmed_h / tmed,
           "t_warm_us": t_warm_us if t_warm_us is not None else tmed * 1e6,
           "t_cold_us": tmed * 1e6 if mode != "warm" else None,
           "tune_seconds": tune_s, "tune_reports": [{k: v for k, v in r.items() if k != "log"} for r in reports],
           "launches_per_step": launches_per_step, "timing": {"rotate": f"cold: steps rotate over {copies} device copies of the inputs (footprint > 3x L2), back to back in one event pair",
                      "flush": "cold: 2xL2 buffer overwritten before every step, per-step events",
                      "warm": "working set >= 4x L2, steps back to back in one event pair"}[mode],
           "deterministic": deterministic, "finite": finite, "e2e": e2e, "clocks": clocks, "cg": cg,
           "sm_count": info.sm_count, "l2_bytes": info.l2_bytes, "device": info.device_name.decode()}
    for h in handles:
        h.close()
    return res, probs[0]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--configs", default="2", help="comma list; the first is the headline (default cfg2)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--variant-filter", default=None,
                    help="comma list of descriptor prefixes the tuner may use (spmv_tune variant_filter), e.g. "
                         "'csr_scalar,csr_vector,sell:,sell_tma,ell,merge,bcsr3,dia:,dia_tma' = everything that still "
                         "reads the matrix values (no constant-coefficient elision)")
    ap.add_argument("--cpu-all", action="store_true", help="time the CPU oracle on every config of --configs, not only the headline")
    ap.add_argument("--tune-cache", default=None,
                    help="file persisting tuning winners (spmv_tune cache_path); a second run then skips the search")
    args = ap.parse_args()
    args.warmup = max(3, args.warmup)

    from paper_1309_1894_b200 import workloads as W
    if args.impl == "reference":
        run_reference(args, W)
        return

    import torch
    from paper_1309_1894_b200 import binding
    binding.lib()                               # fail loudly if the CUDA library is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    device = f"cuda:{local}"
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(device))
    from paper_1309_1894_b200.dist import make_dist_max
    dist_max = make_dist_max(torch, world, device)

    cfgs = [int(c) for c in args.configs.split(",")]
    results = []
    head_prob = None
    for i, cfg in enumerate(cfgs):
        res, prob = bench_config(cfg, args, torch, binding, W, dist_max, device, primary=(rank == 0))
        if args.cpu_all and rank == 0 and i > 0:
            t = cpu_oracle_times(prob, reps=3)
            res["cpu_oracle"] = {"serial_seconds": t["serial"][0], "parallel_seconds": t["parallel"][0],
                                 "cores": t["parallel"][1], "sample": "first matrix of the config, median of 3 applies"}
        results.append(res)
        if i == 0:
            head_prob = prob
    head = results[0]
    peak, peak_src = measured_peak()
    # whole job: every rank ran the same work; time is the max over ranks
    value = head["eff_gbs"] * world
    line = {
        "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": head["t_sum_s"] / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": head["workload"], "rows": head["rows"], "nnz": head["nnz"],
                   "variant": head["variant"], "variant_filter": args.variant_filter, "l2": head["timing"],
                   "parallelism": "replicas only (no data-path collective)" if world > 1 else "1 GPU"},
        "gpu_launches": head["launches_per_step"] * args.steps,
        "clocks": head["clocks"],
        "e2e": ({"value": head["e2e"]["value"] * world, "unit": "GB/s",
                 "h2d_bytes_per_step": head["e2e"]["h2d_bytes_per_step"],
                 "d2h_bytes_per_step": head["e2e"]["d2h_bytes_per_step"],
                 "ms_per_step": head["e2e"]["ms_per_step"]} if head["e2e"] else None),
        "roofline": {"bound": "hbm", "achieved": head["eff_gbs"], "peak": peak, "unit": "GB/s",
                     "frac": head["eff_gbs"] / peak, "peak_source": peak_src,
                     "frac_of_nominal_8TBs": head["eff_gbs"] / NOMINAL_HBM_GBS,
                     "traffic": ncu_traffic(head["variant"], head["cfg"]),
                     "actual_gbs": head["format_gbs"], "frac_actual": head["format_gbs"] / peak,
                     "actual_bytes_per_launch": head["bytes_actual"],
                     "note": "achieved = algorithmic (CSR byte model) bytes / time, as the metric defines it; the winning "
                             "format streams fewer bytes (actual_*), so frac can exceed 1",
                     "kernel": head["variant"], "algorithmic_bytes_per_launch": head["bytes_algorithmic"],
                     "format_bytes_per_launch": head["bytes_format_actual"]},
        "gflops": head["gflops"] * world, "speedup_vs_default": head["speedup_vs_default"],
        "tune_seconds": head["tune_seconds"], "deterministic": head["deterministic"], "cg": head["cg"],
        "per_config": [{k: v for k, v in r.items() if k not in ("clocks",)} for r in results],
    }
    if rank == 0:
        # ceilings measured in the same run with the library's own kernels
        torch.cuda.synchronize()
        ceil = {"copy_gbs_1GiB": binding.measure_ceiling(0, 1 << 30, 5),
                "read_gbs_1GiB": binding.measure_ceiling(1, 1 << 30, 5),
                "read_gbs_at_headline_size": binding.measure_ceiling(1, max(1 << 20, int(head["bytes_actual"])), 5),
                "empty_launch_us": binding.measure_ceiling(2, 0, 200),
                "random_gather_G_per_s_32MiB_table": binding.measure_ceiling(3, 1 << 25, 3)}
        line["ceilings"] = ceil
        try:
            cpu_model = [l.split(":", 1)[1].strip() for l in open("/proc/cpuinfo") if l.startswith("model name")][0]
        except Exception:
            cpu_model = "unknown"
        line["host"] = {"cpu_model": cpu_model, "cores": os.cpu_count(), "cuda": torch.version.cuda,
                        "driver": torch.cuda.get_device_properties(device).name, "torch": torch.__version__}
        for r in line["per_config"]:
            # unstructured columns: every x gather is its own L1->XBAR request (profiles/r01_cfg3_*.md)
            r["frac_of_gather_ceiling"] = r["gathers_per_s"] / 1e9 / ceil["random_gather_G_per_s_32MiB_table"]
            # what bounds this config's winner and the fraction of that bound
            if r["cfg"] == 1:
                r["roofline"] = {"bound": "launch", "achieved": r["t_median_us"], "peak": ceil["empty_launch_us"],
                                 "unit": "us (lower is better; cold apply vs empty-kernel launch)",
                                 "frac": ceil["empty_launch_us"] / r["t_median_us"]}
            elif r["cfg"] == 3:
                r["roofline"] = {"bound": "l1-xbar gather requests", "achieved": r["gathers_per_s"] / 1e9,
                                 "peak": ceil["random_gather_G_per_s_32MiB_table"], "unit": "G gathers/s",
                                 "frac": r["frac_of_gather_ceiling"]}
            else:
                r["roofline"] = {"bound": "hbm", "achieved": r["eff_gbs"], "peak": peak, "unit": "GB/s",
                                 "frac": r["eff_gbs"] / peak, "actual_gbs": r["format_gbs"],
                                 "frac_actual": r["format_gbs"] / peak,
                                 "traffic": ncu_traffic(r["variant"], r["cfg"])}
    if rank == 0 and not args.no_cpu_baseline:
        t = cpu_oracle_times(head_prob)
        nb = W.algorithmic_bytes(head_prob.A.rows, head_prob.A.cols, head_prob.A.nnz, head_prob.beta)
        line["cpu_baseline"] = {"value": nb / t["parallel"][0] / 1e9, "unit": "GB/s", "cores": t["parallel"][1],
                                "kind": "oracle", "sample": f"whole {head_prob.name} matrix, median of 5 applies",
                                "serial_value": nb / t["serial"][0] / 1e9, "serial_seconds": t["serial"][0],
                                "parallel_seconds": t["parallel"][0]}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- fp64 SpMV effective GB/s & fraction of B200 HBM peak (autotuned vs default).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--configs 4,1,2,3,5] [--impl reference]
    python bench.py --profile-one CFG [--variant DESC|tuned] [--iters 5]      (ncu / sanitizer driver)

One "step" is one pass of the hot path, y = alpha*A*x + beta*y through spmv_apply with the autotuned
variant (cfg5: the batch of four applies through spmv_apply_batch), inputs resident in HBM.  Every
config of --configs is tuned (every candidate verified against oracle/'s result for the config's inputs),
checked against the oracle on every row and timed; the FIRST one is the headline (default cfg4, the largest
single matrix: 2.58 GB as CSR).  stdout carries ONE compact JSON line (< 2 KB: contract fields, roofline,
cpu_baseline, e2e, clocks, one summary entry per config); the full record goes to gpurun_out/bench_detail.json.

Three numbers per config, never conflated:
  eff_gbs       algorithmic bytes of the CSR byte model (nnz*12 + (rows+1)*4 + 8*cols + 8*rows
                [+ 8*rows if beta != 0]) / time -- the metric's own definition, `value`;
  roofline      bytes the WINNING format must move (its matrix arrays + x + y, `bytes_actual`) / time
                against MEASURED_PEAKS.json:hbm_gbs -- a real roofline fraction (<= ~1.1);
  traffic       DRAM bytes per launch measured by ncu (profiles/traffic.json), when captured.

Timing: W warm-up steps, then batches of K steps; a batch is bracketed by one CUDA event pair on the
launching stream (per-step pairs in `flush` mode) and batches repeat until the timed region lasts
>= --min-ms (50 ms), the reported time per step is the MEDIAN batch / K, max over ranks.  Cache
state: `warm` when the winner's bytes are >= 4x L2 (cfg3-5: every apply streams from HBM anyway),
`rotate` over enough device copies that the rotated footprint exceeds 3x L2 (cfg2), `flush` (a 2x L2
buffer overwritten before every step) when even that would need too many copies (cfg1).
`e2e` is the same metric through spmv_apply_host with pinned HOST vectors (H2D of x and y, apply,
D2H of y inside the timed region).  N > 1: N independent replicas (the path is
single-GPU; "replicas only"), barrier + max over ranks, no data-path collective.
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
DEFAULT_CONFIGS = "4,1,2,3,5"
VALUE_STREAMING_FILTER = "csr_scalar,csr_vector,sell:,sell_tma,sell16,ell,merge,bcsr3,dia:,dia_tma,dia_win"


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
        # (the index width is part of the format: bcsr3 with and without i16 stream different bytes)
        key = lambda v: (v.split(":")[0], ":i16" in v)
        return e.get("dram_bytes_per_launch") if key(e.get("variant", "")) == key(variant) else None
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


# ------------------------------------------------------------------------------------------------
# the oracle on the host cores: ONE protocol for the cpu_baseline leg and for --impl reference
# ------------------------------------------------------------------------------------------------
def oracle_time(prob, warmup: int, steps: int, parallel: bool = True):
    """`warmup` untimed then `steps` timed applies of the oracle as it stands, back to back and in
    place on one y vector (no allocation inside the timed region).  Returns (mean seconds per
    apply, threads used)."""
    import oracle
    A = prob.A
    rp = np.ascontiguousarray(A.row_ptr, dtype=np.int32)
    ci = np.ascontiguousarray(A.col_idx, dtype=np.int32)
    va = np.ascontiguousarray(A.val, dtype=np.float64)
    x = np.ascontiguousarray(prob.x)
    y = (prob.y0 if prob.y0 is not None else np.zeros(A.rows)).copy()
    scale = np.empty(A.rows)
    threads = 1
    for _ in range(warmup):
        threads = oracle.spmv_inplace(rp, ci, va, prob.alpha, x, prob.beta, y, scale, parallel=parallel)
    t0 = time.perf_counter()
    for _ in range(steps):
        threads = oracle.spmv_inplace(rp, ci, va, prob.alpha, x, prob.beta, y, scale, parallel=parallel)
    return (time.perf_counter() - t0) / max(steps, 1), int(threads)


def cpu_baseline(prob, W, steps_parallel=5, steps_serial=2):
    """cpu_baseline object for one config: the oracle's row-parallel form (bit-identical to the
    serial loop) on every host core, plus the serial figure."""
    nb = W.algorithmic_bytes(prob.A.rows, prob.A.cols, prob.A.nnz, prob.beta)
    tp, threads = oracle_time(prob, 1, steps_parallel, parallel=True)
    ts, _ = oracle_time(prob, 1, steps_serial, parallel=False)
    return {"value": nb / tp / 1e9, "unit": "GB/s", "cores": threads, "kind": "oracle",
            "sample": f"whole matrix of {prob.name} ({prob.A.nnz} nnz): 1 warm-up + {steps_parallel} applies "
                      "back to back, in place, mean",
            "parallel_seconds": tp, "serial_seconds": ts, "serial_value": nb / ts / 1e9,
            "gflops": 2.0 * prob.A.nnz / tp / 1e9}


def oracle_reference(prob):
    """(y_ref, scale) of the whole config from oracle/ (its row-parallel form, bit-identical to the serial loop)."""
    import oracle
    A = prob.A
    return oracle.spmv(A.row_ptr, A.col_idx, A.val, prob.alpha, prob.x, prob.beta, prob.y0, parallel=True)


def oracle_check(prob, y_gpu: np.ndarray, ref=None, tol: float = 1e-12):
    """Parity of what was timed, on EVERY row: the oracle (oracle/, plain CPU row loop) recomputes the whole
    product from the same inputs (`ref`: its (y_ref, scale) when already computed for the tuner); acceptance rule
    and tolerance are north_star's (1e-12 relative to scale_i).  Returns a small report dict."""
    import oracle
    y_ref, scale = ref if ref is not None else oracle_reference(prob)
    ok, mr, ff, nf = oracle.accept(y_gpu, y_ref, scale, tol)
    return {"rows_checked": int(prob.A.rows), "ok": bool(ok), "max_err_over_scale": float(mr), "n_fail": int(nf),
            "first_fail_row": int(ff) if nf else -1, "tolerance": tol}


def run_reference(args, W):
    """--impl reference: the oracle (row-parallel form of the same loop) on the host cores, on the
    product arm's headline config, --warmup W and --steps K honoured as given."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = int(args.configs.split(",")[0])
    prob = W.config(cfg)
    A = prob.A
    nbytes = W.algorithmic_bytes(A.rows, A.cols, A.nnz, prob.beta) * (4 if cfg == 5 else 1)
    nnz = A.nnz * (4 if cfg == 5 else 1)
    dt, threads = oracle_time(prob, args.warmup, args.steps, parallel=True)
    if cfg == 5:
        dt *= 4           # a step of cfg5 is four applies; the four matrices share one pattern
    gbs = nbytes / dt / 1e9
    sample = (f"{args.steps} applies of the whole matrix of {prob.name} ({A.nnz} nnz), in place, back to back"
              + ("; a step = 4 x that time" if cfg == 5 else ""))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": gbs, "unit": "GB/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": headline_config(W, cfg, A.rows, nnz),
        "cpu_baseline": {"value": gbs, "unit": "GB/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": gbs, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gflops": 2.0 * nnz / dt / 1e9,
    }))


def headline_config(W, cfg, rows, nnz):
    """The `config` object: identical in both arms (workload only; what was selected is `selection`)."""
    big = 12 * int(nnz) + 20 * int(rows) >= 4 * 126 * (1 << 20)
    return {"workload": W.CONFIG_NAMES[cfg], "rows": int(rows), "nnz": int(nnz),
            "l2": "inputs >= 4x L2: no flush" if big else "cold: rotated copies > 3x L2, or 2x L2 flush per step"}


# ------------------------------------------------------------------------------------------------
# one config on this rank
# ------------------------------------------------------------------------------------------------
def bench_config(cfg, args, torch, binding, W, dist_max, device, primary):
    members = 4 if cfg == 5 else 1
    probs = [W.config(cfg, member=m) for m in range(members)]
    A0 = probs[0].A
    alpha, beta = probs[0].alpha, probs[0].beta
    nbytes = sum(W.algorithmic_bytes(p.A.rows, p.A.cols, p.A.nnz, p.beta) for p in probs)
    nnz = sum(p.A.nnz for p in probs)
    vec_bytes = sum(8 * p.A.cols + 8 * p.A.rows * (2 if p.beta != 0 else 1) for p in probs)
    l2 = torch.cuda.get_device_properties(device).L2_cache_size

    handles, xs, ys, y0s = [], [], [], []

    def add_copy():
        for p in probs:
            handles.append(binding.SpMV.from_csr(p.A, device=device))
            xs.append(torch.from_numpy(p.x).to(device))
            y0 = p.y0 if p.y0 is not None else np.zeros(p.A.rows)
            y0s.append(torch.from_numpy(y0).to(device))
            ys.append(y0s[-1].clone())

    add_copy()
    # the oracle's result for the config's own inputs: the reference EVERY tuner candidate is verified against
    # (north_star (d)) and, after the timed region, the every-row parity check of the timed variant
    refs, drefs = [], []
    if not args.no_oracle_check:
        refs = [oracle_reference(p) for p in probs]
        drefs = [(torch.from_numpy(yr).to(device), torch.from_numpy(sc).to(device)) for yr, sc in refs]
    state = {"copies": 1, "mode": "warm", "step": 0, "nstreams": 1}
    streams = [torch.cuda.current_stream()]
    flush = None

    def one_step():
        if members == 1:
            i = state["step"] % state["copies"]
            state["step"] += 1
            handles[i].apply(alpha, xs[i], beta, ys[i])
        else:
            binding.apply_batch(handles[:members], [alpha] * members, xs[:members], [beta] * members, ys[:members],
                                streams[:state["nstreams"]])

    def fork_join_step(ev):
        for s in streams[1:state["nstreams"]]:
            s.wait_event(ev)
        one_step()
        for s in streams[1:state["nstreams"]]:
            j = torch.cuda.Event()
            j.record(s)
            torch.cuda.current_stream().wait_event(j)

    def batch(steps):
        """K steps; returns seconds per step of this batch (device time, CUDA events on the launching stream)."""
        if state["mode"] == "flush":
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
            for a, b in evs:
                flush.fill_(1.0)
                a.record()
                one_step()
                b.record()
            torch.cuda.synchronize()
            return float(np.sum([a.elapsed_time(b) for a, b in evs])) * 1e-3 / steps
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(steps):
            if members > 1:
                fork_join_step(a)
            else:
                one_step()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) * 1e-3 / steps

    def timed(steps, warmup, min_ms, max_batches=400):
        """returns (list of per-step seconds, one entry per batch)"""
        for _ in range(warmup):
            one_step()
        torch.cuda.synchronize()
        ts = [batch(steps)]
        while sum(ts) * steps * 1e3 < min_ms and len(ts) < max_batches:
            ts.append(batch(steps))
        return ts

    # ---- tune first (setup, outside the timed region); the two fixed baselines are timed below under the
    # same cache protocol as the winner
    def tune(i, first, **kw):
        # the cold protocol applies when the CSR-model footprint is below 4x L2 (decided before the winner is known)
        m = i % members
        ref = dict(x=xs[i], y0=y0s[i], y_ref=drefs[m][0], scale=drefs[m][1]) if drefs else {}
        opts = dict(alpha=alpha, beta=beta, use_cache=(0 if (not first or args.tune_cache) else 2),
                    cache_path=args.tune_cache, flush_l2=(nbytes < 4 * l2), seed=cfg,
                    variant_filter=args.variant_filter)
        opts.update(ref)
        opts.update(kw)
        return handles[i].tune(**opts)
    t0 = time.perf_counter()
    reports = [tune(i, i == 0) for i in range(len(handles))]
    stream_times = {}
    if members > 1:
        streams = [torch.cuda.current_stream()] + [torch.cuda.Stream(device=device) for _ in range(3)]
        state["nstreams"], stream_times = binding.tune_batch(handles, [alpha] * members, xs, [beta] * members, ys, streams)
    tune_s = time.perf_counter() - t0
    variant = handles[0].variant
    # the feature-guided search on the same matrix and reference: its cost and its winner
    guided = None
    if not args.no_extras:
        rg = tune(0, True, use_cache=2, cache_path=None, search=1)
        guided = {"tune_seconds": rg["tune_seconds"], "winner": rg["winner"], "winner_us": rg["winner_us"],
                  "n_timed": rg["n_timed"], "exhaustive_tune_seconds": reports[0]["tune_seconds"],
                  "exhaustive_winner_us": reports[0]["winner_us"], "exhaustive_n_timed": reports[0]["n_timed"]}
        handles[0].select(variant)
    fmt_bytes = int(sum(h.info().format_bytes for h in handles[:members]))
    bytes_actual = fmt_bytes + vec_bytes
    # merge-path and row-split SELL add one small ordered fix-up kernel per apply
    launches_per_step = members * (2 if (variant.startswith("merge") or ":l" in variant) else 1)

    # ---- cache protocol, sized from what the WINNER streams (not from the CSR byte model)
    if bytes_actual >= 4 * l2:
        state["mode"] = "warm"
    else:
        copies = int(np.ceil(3.0 * l2 / bytes_actual)) + 1
        if members == 1 and copies <= 16:
            state["mode"] = "rotate"
            for _ in range(copies - 1):
                add_copy()
                tune(len(handles) - 1, False)     # in-process cache hit: same variant
            state["copies"] = copies
        else:
            state["mode"] = "flush"
            flush = torch.empty(int(2 * l2 // 8), dtype=torch.float64, device=device)
    # ---- the two fixed baselines, same cache protocol (default: SURVEY A17; heuristic: sub-warp width = smallest
    # power of two >= the mean row length), then back to the tuned variant
    mean_len = handles[0].info().mean_row_len
    w_h = int(min(32, max(2, 2 ** int(np.ceil(np.log2(max(mean_len, 1.0)))))))
    heuristic = f"csr_vector:b256:w{w_h}:u1:x0"
    k_base = max(5, args.steps // 4)
    base_t = {}
    for name in ("default", heuristic):
        for h in handles:
            h.select(name)
        base_t[name] = float(np.median(timed(k_base, 3, 5.0, max_batches=20)))
    t_default, t_heur = base_t["default"], base_t[heuristic]
    for h in handles:
        h.select(variant)
    assert all(h.variant == variant for h in handles), "copies must run the tuned variant"
    for y, y0 in zip(ys, y0s):
        y.copy_(y0)
    timing_note = {
        "rotate": f"cold: steps rotate over {state['copies']} device copies of the inputs ({state['copies']} x "
                  f"{bytes_actual / 1e6:.1f} MB streamed by the winner > 3x L2), back to back in one event pair per batch",
        "flush": "cold: 2xL2 buffer overwritten before every step, per-step event pairs",
        "warm": f"winner streams {bytes_actual / 1e6:.0f} MB per step >= 4x L2: steps back to back in one event pair per batch",
    }[state["mode"]]

    # ---- the timed region: barrier + sync on both sides, median batch, max over ranks
    sampler = ClockSampler(torch.cuda.current_device()) if primary else None
    for _ in range(args.warmup):
        one_step()
    torch.cuda.synchronize()
    dist_max(0.0)                               # barrier
    ts = timed(args.steps, 0, args.min_ms)
    t_step = dist_max(float(np.median(ts)))
    n_batches = len(ts)
    if sampler is not None:                     # keep the same load a little longer so the sampler sees it
        t_end = time.time() + 0.5
        while time.time() < t_end:
            for _ in range(20):
                one_step()
            torch.cuda.synchronize()
    clocks = sampler.stop() if sampler is not None else None

    # ---- where the winner reads no matrix values (constant-coefficient stencil): the best variant that DOES stream
    # them, same cache protocol -- what the stencil kernels do on a variable-coefficient matrix of this shape
    with_values = None
    if members == 1 and variant.split(":")[0] in ("dia_const", "dia_cwin") and not args.no_extras:
        rv = tune(0, True, use_cache=2, cache_path=None, variant_filter=VALUE_STREAMING_FILTER)
        for h in handles:
            h.select(rv["winner"])
        tv = float(np.median(timed(k_base, 3, 5.0, max_batches=20)))
        fbv = int(handles[0].info().format_bytes) + vec_bytes
        with_values = {"variant": rv["winner"], "t_us": tv * 1e6, "eff_gbs": nbytes / tv / 1e9,
                       "bytes_actual": fbv, "actual_gbs": fbv / tv / 1e9, "frac_actual_of_measured": fbv / tv / 1e9 / measured_peak()[0],
                       "filter": VALUE_STREAMING_FILTER}
        for h in handles:
            h.select(variant)

    # ---- the other cache state: warm (same buffers back to back) where the headline is cold
    t_warm = t_step
    if state["mode"] != "warm" and members == 1:
        keep = (state["mode"], state["copies"])
        state["mode"], state["copies"] = "warm", 1
        t_warm = float(np.median(timed(args.steps, 5, 5.0)))
        state["mode"], state["copies"] = keep

    # ---- host cost of one spmv_apply call: wall clock of n enqueues on an idle stream / n
    torch.cuda.synchronize()
    n_host = 256                                 # below the launch-queue depth even for two-launch variants
    h0, x0d, y0d = handles[0], xs[0], ys[0]
    t1 = time.perf_counter()
    for _ in range(n_host):
        h0.apply(alpha, x0d, beta, y0d)
    host_us = (time.perf_counter() - t1) / n_host * 1e6
    torch.cuda.synchronize()

    # ---- parity of what was timed: determinism, and the oracle on sampled rows
    def first_members():
        for y, y0 in zip(ys[:members], y0s[:members]):
            y.copy_(y0)
        if members == 1:
            handles[0].apply(alpha, xs[0], beta, ys[0])
        else:
            binding.apply_batch(handles[:members], [alpha] * members, xs[:members], [beta] * members, ys[:members],
                                streams[:state["nstreams"]])
        torch.cuda.synchronize()
        return [y.clone() for y in ys[:members]]
    first = first_members()
    deterministic = all(torch.equal(a, b) for a, b in zip(first, first_members()))
    parity = None
    if primary and not args.no_oracle_check:
        checks = [oracle_check(p, y.cpu().numpy(), ref=r) for p, y, r in zip(probs, first, refs)]
        parity = {"ok": all(c["ok"] for c in checks), "rows_checked": sum(c["rows_checked"] for c in checks),
                  "max_err_over_scale": max(c["max_err_over_scale"] for c in checks),
                  "n_fail": sum(c["n_fail"] for c in checks), "tolerance": 1e-12,
                  "rows": int(sum(p.A.rows for p in probs)),
                  "what": "one apply of the timed variant from y0 vs oracle/ on every row"}
        if not parity["ok"]:
            raise SystemExit(f"bench: cfg{cfg} {variant} FAILED the oracle check: {checks}")

    # ---- e2e through spmv_apply_host (cfg5: spmv_apply_host_batch over the four members) with pinned host vectors
    xh = [torch.from_numpy(p.x).pin_memory() for p in probs]
    yh = [torch.from_numpy((p.y0 if p.y0 is not None else np.zeros(p.A.rows)).copy()).pin_memory() for p in probs]

    def e2e_step():
        if members == 1:
            handles[0].apply_host(alpha, xh[0], beta, yh[0])     # synchronises the stream itself
        else:                                                    # cfg5: the members' pipelines enqueued together, one synchronise
            binding.apply_host_batch(handles[:members], [alpha] * members, xh[:members], [beta] * members, yh[:members])
    for _ in range(3):
        e2e_step()
    n_e2e = max(5, min(args.steps, 50))
    torch.cuda.synchronize()
    dist_max(0.0)
    t1 = time.perf_counter()
    for _ in range(n_e2e):
        e2e_step()
    te = dist_max((time.perf_counter() - t1) / n_e2e)
    e2e = {"value": nbytes / te / 1e9, "unit": "GB/s", "ms_per_step": te * 1e3, "steps": n_e2e,
           "h2d_bytes_per_step": int(sum(8 * p.A.cols + (8 * p.A.rows if p.beta != 0 else 0) for p in probs)),
           "d2h_bytes_per_step": int(sum(8 * p.A.rows for p in probs))}

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
                r = handles[0].cg(bvec, xg, tol=1e-300, max_iters=n_it, check_every=25, tune_loop=True)
                if best is None or r["device_seconds"] < best["device_seconds"]:
                    best = r
            st.synchronize()
        # per iteration: one SpMV (algorithmic bytes with beta = 0) + dot (16 B/row) + x/r update (48) + p update (24)
        it_bytes = W.algorithmic_bytes(A0.rows, A0.cols, A0.nnz, 0.0) + 88 * A0.rows
        cg = {"iters": best["iters"], "us_per_iteration": best["device_seconds"] / max(best["iters"], 1) * 1e6,
              "eff_gbs": it_bytes * best["iters"] / best["device_seconds"] / 1e9,
              "rel_residual": best["rel_residual"], "graph_replays": best["graph_replays"],
              "fused_single_kernel": bool(best["fused"]), "fused_dot": bool(best["fused_dot"]),
              "kernels_per_iteration": best["kernels_per_iteration"], "loop_variant": best["loop_variant"],
              "bytes_per_iteration_algorithmic": it_bytes}
        for h in handles:                      # tune_loop may have adopted another leader: back to the apply winner
            h.select(variant)
        # the second solver loop (weighted Jacobi, omega = 0.8): SpMV + one fused pass (b, t, d, x read, x written: 40 B/row)
        with torch.cuda.stream(st):
            bestj = None
            for _ in range(3):
                xg = torch.zeros(A0.rows, dtype=torch.float64, device=device)
                r = handles[0].jacobi(bvec, xg, omega=0.8, tol=1e-300, max_iters=n_it, check_every=24)
                if bestj is None or r["device_seconds"] < bestj["device_seconds"]:
                    bestj = r
            st.synchronize()
        jb = W.algorithmic_bytes(A0.rows, A0.cols, A0.nnz, 0.0) + 40 * A0.rows
        cg["jacobi"] = {"iters": bestj["iters"], "us_per_iteration": bestj["device_seconds"] / max(bestj["iters"], 1) * 1e6,
                        "eff_gbs": jb * bestj["iters"] / bestj["device_seconds"] / 1e9, "rel_residual": bestj["rel_residual"],
                        "kernels_per_iteration": bestj["kernels_per_iteration"], "bytes_per_iteration_algorithmic": jb,
                        "note": "device_seconds includes the one-off diagonal extraction (one pass over the CSR arrays)"}

    # ---- K applies replayed as one CUDA graph (launch-bound configs; a clearly labelled extra line)
    graph = None
    if members == 1 and cfg in (1, 2):
        kg = 50
        g = handles[0].graph(alpha, xs[0], beta, ys[0], kg)
        for _ in range(3):
            g.launch()
        torch.cuda.synchronize()
        tg = []
        for _ in range(20):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            g.launch()
            b.record()
            torch.cuda.synchronize()
            tg.append(a.elapsed_time(b) * 1e3 / kg)
        g.close()
        graph = {"applies_per_graph": kg, "us_per_apply": float(np.median(tg)),
                 "eff_gbs": nbytes / float(np.median(tg)) / 1e3,
                 "note": "ADDITIONAL line, not the headline: spmv_graph_create captures 50 back-to-back applies on ONE "
                         "set of buffers (warm caches), one cudaGraphLaunch replays them; launch cost amortised"}

    info = handles[0].info()
    peak_meas, _ = measured_peak()
    res = {"cfg": cfg, "workload": W.CONFIG_NAMES[cfg], "rows": A0.rows, "cols": A0.cols, "nnz": nnz, "members": members,
           "variant": variant, "nstreams": state["nstreams"], "stream_times_us": stream_times,
           "bytes_algorithmic": nbytes, "bytes_format_actual": fmt_bytes, "bytes_actual": bytes_actual,
           "t_step_us": t_step * 1e6, "t_batches_us": {"n": n_batches, "min": float(np.min(ts)) * 1e6,
                                                      "median": float(np.median(ts)) * 1e6, "max": float(np.max(ts)) * 1e6},
           "timed_region_ms": float(np.sum(ts)) * args.steps * 1e3,
           "eff_gbs": nbytes / t_step / 1e9, "actual_gbs": bytes_actual / t_step / 1e9,
           "frac_effective_of_8TBs": nbytes / t_step / 1e9 / NOMINAL_HBM_GBS,
           "frac_effective_of_measured": nbytes / t_step / 1e9 / peak_meas,
           "frac_actual_of_measured": bytes_actual / t_step / 1e9 / peak_meas,
           "gathers_per_s": nnz / t_step, "gflops": 2.0 * nnz / t_step / 1e9,
           "t_default_us": t_default * 1e6, "speedup_vs_default": t_default / t_step,
           "heuristic_variant": heuristic, "t_heuristic_us": t_heur * 1e6, "speedup_vs_heuristic": t_heur / t_step,
           "t_warm_us": t_warm * 1e6, "t_cold_us": t_step * 1e6 if state["mode"] != "warm" else None,
           "host_us_per_apply": host_us, "gpu_launches": launches_per_step * args.steps * n_batches,
           "tune_seconds": tune_s, "tune_reports": [{k: v for k, v in r.items() if k != "log"} for r in reports[:members]],
           "launches_per_step": launches_per_step, "timing": timing_note, "cache_mode": state["mode"],
           "deterministic": deterministic, "parity": parity, "e2e": e2e, "clocks": clocks, "cg": cg,
           "graph_replay": graph, "guided_search": guided, "with_values": with_values,
           "tune_reference": "oracle" if drefs else "library reference kernel", "sm_count": info.sm_count, "l2_bytes": info.l2_bytes,
           "device": info.device_name.decode()}
    for h in handles:
        h.close()
    return res, probs[0]


def bench_banded(args, torch, binding, W, device):
    """Extra line: a banded matrix with unstructured columns inside the band (2^21 rows, 24
    entries per row within +-2000 of the diagonal: ~4000 distinct diagonals, DIA refuses it).  Tuned twice: over
    everything, and over the 32-bit-index families only; both winners are checked against the oracle."""
    A = W.banded_random(1 << 21, 24, 2000)
    x = W.uniform(90, A.cols)
    prob = W.Problem("banded-random 2^21 rows, 24/row within +-2000", A, x, None, 1.0, 0.0)
    nb = W.algorithmic_bytes(A.rows, A.cols, A.nnz, 0.0)
    S = binding.SpMV.from_csr(A, device=device)
    dx = torch.from_numpy(x).to(device)
    dy = torch.zeros(A.rows, dtype=torch.float64, device=device)
    out = {"workload": prob.name, "rows": A.rows, "nnz": A.nnz, "bytes_algorithmic": nb}
    for key, flt in (("idx32_only", "csr_scalar,csr_vector,sell:,sell_tma,ell,merge"), ("all", None)):
        rep = S.tune(alpha=1.0, beta=0.0, use_cache=2, variant_filter=flt, seed=7)
        S.apply(1.0, dx, 0.0, dy)
        torch.cuda.synchronize()
        chk = oracle_check(prob, dy.cpu().numpy())
        if not chk["ok"]:
            raise SystemExit(f"bench: banded {rep['winner']} FAILED the oracle check: {chk}")
        fb = int(S.info().format_bytes)
        out[key] = {"variant": rep["winner"], "us": rep["winner_us"], "eff_gbs": nb / rep["winner_us"] / 1e3,
                    "format_bytes": fb, "actual_gbs": (fb + 16 * A.rows) / rep["winner_us"] / 1e3,
                    "max_err_over_scale": chk["max_err_over_scale"], "tune_seconds": rep["tune_seconds"]}
    out["speedup_16bit_over_32bit"] = out["idx32_only"]["us"] / out["all"]["us"]
    out["timing"] = "spmv_tune's own protocol: median of 5 batches of back-to-back applies (603 MB CSR: warm = streaming)"
    S.close()
    return out


def bench_sharded(args, torch, binding, W, dist_max, device, world, rank):
    """--sharded: ONE matrix row-sharded over the N GPUs (strong scaling), instead of the default
    N independent replicas.  Every rank builds the same seeded matrix and keeps its nnz-balanced row block; a step
    is one sharded apply: halo exchange (torch.distributed point-to-point over NCCL) overlapped with the interior
    rows, then the boundary rows.  Time: CUDA events on the launching stream, barrier on both sides, max over ranks."""
    from paper_1309_1894_b200 import sharded
    cfg = int(args.configs.split(",")[0])
    prob = W.config(cfg)
    A = prob.A
    transport = sharded.TorchDistTransport() if world > 1 else sharded.LoopbackTransport(1).view(0)
    align = 768 if cfg == 4 else 512
    sh = sharded.ShardedSpMV(A, transport, device=device, align=align)
    sh.finish_setup()
    l2 = torch.cuda.get_device_properties(device).L2_cache_size
    rep = sh.tune(alpha=prob.alpha, beta=prob.beta, use_cache=2, seed=cfg,
                  flush_l2=(12 * sh.nnz_local + 24 * sh.rows_local < 4 * l2))
    sh.x_owned.copy_(torch.from_numpy(prob.x[sh.lo:sh.hi]))
    y0 = prob.y0 if prob.y0 is not None else np.zeros(A.rows)
    y = torch.from_numpy(y0[sh.lo:sh.hi].copy()).to(device)
    for _ in range(args.warmup):
        sh.apply(prob.alpha, prob.beta, y)
    torch.cuda.synchronize()
    dist_max(0.0)
    ts = []
    while sum(ts) * args.steps * 1e3 < args.min_ms and len(ts) < 400 or not ts:
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(args.steps):
            sh.apply(prob.alpha, prob.beta, y)
        b.record()
        torch.cuda.synchronize()
        ts.append(dist_max(a.elapsed_time(b) * 1e-3 / args.steps))
    t = float(np.median(ts))
    # parity of this rank's block against the oracle on sampled rows (one apply from y0)
    y.copy_(torch.from_numpy(y0[sh.lo:sh.hi]))
    sh.apply(prob.alpha, prob.beta, y)
    torch.cuda.synchronize()
    sub = W.CSR(sh.rows_local, A.cols, (A.row_ptr[sh.lo:sh.hi + 1].astype(np.int64) - int(A.row_ptr[sh.lo])).astype(np.int32),
                A.col_idx[int(A.row_ptr[sh.lo]):int(A.row_ptr[sh.hi])], A.val[int(A.row_ptr[sh.lo]):int(A.row_ptr[sh.hi])])
    chk = oracle_check(W.Problem(prob.name, sub, prob.x, None if prob.y0 is None else y0[sh.lo:sh.hi], prob.alpha, prob.beta),
                       y.cpu().numpy())
    if not chk["ok"]:
        raise SystemExit(f"bench --sharded: rank {rank} FAILED the oracle check: {chk}")
    nbytes = W.algorithmic_bytes(A.rows, A.cols, A.nnz, prob.beta)
    line = {"metric": METRIC, "value": nbytes / t / 1e9, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": headline_config(W, cfg, A.rows, A.nnz),
            "selection": {"variant_rank0": rep["winner"], "parallelism": f"rows sharded over {world} GPUs, halo exchange + interior overlap",
                          "rows_rank0": sh.rows_local, "halo_bytes_rank0": sh.halo.bytes_received(),
                          "interior_split_rank0": sh.split},
            "gpu_launches": args.steps * len(ts) * (1 if sh.split is None else 3), "parity": chk,
            "timed_batches": len(ts), "gflops": 2.0 * A.nnz / t / 1e9}
    if rank == 0:
        print(json.dumps(line))
    sh.close()


def config_roofline(r, peak, ceil):
    """What bounds this config's winner and the fraction of that bound."""
    if r["cfg"] == 1:       # 0.1 MB per apply: launch-latency-bound
        return {"bound": "launch", "achieved": r["t_step_us"], "peak": ceil["empty_launch_us"],
                "unit": "us (lower is better; cold apply vs empty-kernel launch)",
                "frac": ceil["empty_launch_us"] / r["t_step_us"],
                "actual_gbs": r["actual_gbs"], "frac_hbm_actual": r["frac_actual_of_measured"]}
    if r["cfg"] == 3:       # unstructured columns: every x gather is its own L1->XBAR request
        g = r["gathers_per_s"] / 1e9
        return {"bound": "l1-xbar gather requests", "achieved": g, "peak": ceil["random_gather_G_per_s_32MiB_table"],
                "unit": "G gathers/s", "frac": g / ceil["random_gather_G_per_s_32MiB_table"],
                "actual_gbs": r["actual_gbs"], "frac_hbm_actual": r["frac_actual_of_measured"],
                "traffic": ncu_traffic(r["variant"], r["cfg"])}
    return {"bound": "hbm", "achieved": r["actual_gbs"], "peak": peak, "unit": "GB/s",
            "frac": r["frac_actual_of_measured"], "bytes_per_launch": r["bytes_actual"],
            "effective_gbs": r["eff_gbs"], "frac_effective": r["frac_effective_of_measured"],
            "traffic": ncu_traffic(r["variant"], r["cfg"]),
            "note": "achieved = bytes the winning format must move (its arrays + x + y) / time; effective_* uses the "
                    "CSR byte model of the metric and exceeds 1 when the format streams fewer bytes than CSR"}


COMPACT_LIMIT = 2048      # bytes: the LAST stdout line must stay a short, driver-parseable JSON object


def _r(v, nd=4):
    """Round floats for the compact line (significant digits, not decimals)."""
    if isinstance(v, float):
        return float(f"{v:.{nd + 2}g}")
    return v


def compact_line(full: dict, detail_path: str | None) -> dict:
    """The one JSON line of the contract: headline fields of the first config, the roofline / cpu_baseline / e2e
    objects, and a one-entry-per-config summary.  Everything else (tune reports, ceilings, solver loops, the banded
    extra) goes to the detail file.  Kept under COMPACT_LIMIT bytes (tests/test_bench_line_cpu.py)."""
    out = {k: _r(full.get(k)) for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step",
                                        "higher_is_better", "scaling", "vs_baseline", "dtype", "data")}
    out["config"] = dict(full["config"])
    rf = full.get("roofline") or {}
    out["roofline"] = {k: _r(rf.get(k)) for k in ("bound", "achieved", "peak", "unit", "frac", "traffic",
                                                  "bytes_per_launch", "effective_gbs", "kernel") if k in rf}
    cb = full.get("cpu_baseline")
    if cb:
        out["cpu_baseline"] = {"value": _r(cb["value"]), "unit": cb["unit"], "cores": cb["cores"], "kind": cb["kind"],
                               "sample": str(cb.get("sample", ""))[:64]}
    e = full["e2e"]
    out["e2e"] = {k: _r(e[k]) for k in ("value", "unit", "ms_per_step", "h2d_bytes_per_step", "d2h_bytes_per_step")}
    out["gpu_launches"] = full["gpu_launches"]
    ck = full.get("clocks") or {}
    out["clocks"] = {"sm_mhz": ck.get("sm_mhz"), "sm_max_mhz": ck.get("sm_max_mhz"), "reasons": ck.get("reasons", [])}
    par = full.get("parity") or {}
    out["parity"] = {k: _r(par.get(k)) for k in ("ok", "rows_checked", "rows", "max_err_over_scale", "tolerance")}
    out["deterministic"] = full.get("deterministic")
    out["speedup_vs_default"] = _r(full.get("speedup_vs_default"))
    g = full.get("guided_search") or {}
    out["tune"] = {"reference": full.get("tune_reference"), "exhaustive_s": _r(g.get("exhaustive_tune_seconds"), 2),
                   "guided_s": _r(g.get("tune_seconds"), 2), "exhaustive_us": _r(g.get("exhaustive_winner_us")),
                   "guided_us": _r(g.get("winner_us"))}
    rows = []
    for r in full.get("per_config", []):
        rr = r.get("roofline") or {}
        row = {"cfg": r["cfg"], "variant": r["variant"], "us": _r(r["t_step_us"], 2), "frac": _r(rr.get("frac"), 1)}
        wv = r.get("with_values")
        if wv and wv["frac_actual_of_measured"] > 0.05:    # (not for launch-bound sizes)
                  # the best variant that still streams the matrix values: [descriptor, us, fraction of the HBM peak]
            row["with_values"] = [wv["variant"], _r(wv["t_us"], 2), _r(wv["frac_actual_of_measured"], 1)]
        rows.append(row)
    out["detail"] = detail_path
    # never let the summary break the contract line: drop its optional parts until it fits
    for drop in ((), ("with_values",), ("with_values", "variant")):
        out["per_config"] = [{k: v for k, v in row.items() if k not in drop} for row in rows]
        if len(json.dumps(out, separators=(",", ":"))) < COMPACT_LIMIT - 100:
            break
    return out


def write_detail(full: dict) -> str | None:
    """The full record (per-config tune reports, ceilings, solver loops, banded extra) as a side file."""
    for d in (os.path.join(ROOT, "gpurun_out"), tempfile.gettempdir()):
        try:
            os.makedirs(d, exist_ok=True)
            path = os.path.join(d, "bench_detail.json")
            with open(path, "w") as f:
                json.dump(full, f, indent=1)
            return os.path.relpath(path, ROOT) if path.startswith(ROOT) else path
        except OSError:
            continue
    return None


def relaunch_under_torchrun(args) -> None:
    """`python bench.py --gpus N` with N > 1 and no launcher around it: start N ranks ourselves (one process per GPU,
    torch.distributed.run on 127.0.0.1) -- the same launch the driver uses -- and become that launcher."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    sys.stdout.flush()
    os.execv(sys.executable, cmd)


def rendezvous_only(args) -> None:
    """--rendezvous-only: every rank joins the process group (nccl with a GPU per rank, else gloo), one all-reduce
    counts them, rank 0 prints {"ranks_joined": N}.  The launch-readiness check of `--gpus N` (no SpMV work)."""
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    n = 1
    if world > 1:
        use_nccl = torch.cuda.is_available() and torch.cuda.device_count() >= world
        if use_nccl:
            torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
        dist.init_process_group("nccl" if use_nccl else "gloo")
        t = torch.ones(1, device="cuda" if use_nccl else "cpu")
        dist.all_reduce(t)
        n = int(t.item())
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"ranks_joined": n, "n_gpus": args.gpus, "world_size": world}))


def profile_one(args, torch, binding, W):
    """A few applies of one variant on one config: the command the ncu captures under profiles/ run."""
    cfg = args.profile_one
    if cfg == 6:        # the banded extra workload of bench_banded
        A6 = W.banded_random(1 << 21, 24, 2000)
        prob = W.Problem("banded-random 2^21 rows, 24/row within +-2000", A6, W.uniform(90, A6.cols), None, 1.0, 0.0)
    else:
        prob = W.config(cfg)
    A = prob.A
    S = binding.SpMV.from_csr(A)
    x = torch.from_numpy(prob.x).cuda()
    y = torch.from_numpy(prob.y0 if prob.y0 is not None else np.zeros(A.rows)).cuda()
    if args.variant in (None, "tuned"):
        rep = S.tune(alpha=prob.alpha, beta=prob.beta, use_cache=2, flush_l2=True, variant_filter=args.variant_filter)
        print("tuned:", rep["winner"], f"{rep['winner_us']:.2f} us; default {rep['default_us']:.2f} us")
    else:
        S.select(args.variant)
    flush = torch.empty(int(2 * S.info().l2_bytes // 8), dtype=torch.float64, device="cuda")
    ts = []
    for _ in range(args.iters):
        flush.fill_(1.0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        S.apply(prob.alpha, x, prob.beta, y)
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1) * 1e3)
    nb = W.algorithmic_bytes(A.rows, A.cols, A.nnz, prob.beta)
    t = float(np.median(ts))
    print(f"{prob.name} | {S.variant} | {t:.2f} us/apply (cold, single launches) | {nb / t / 1e3:.1f} GB/s effective | "
          f"format bytes {S.info().format_bytes}")
    S.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--configs", default=DEFAULT_CONFIGS, help="comma list; the first is the headline (default cfg4)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--min-ms", type=float, default=50.0, help="batches of --steps repeat until the timed region lasts this long")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-oracle-check", action="store_true")
    ap.add_argument("--sharded", action="store_true",
                    help="N > 1: row-shard ONE matrix (the first of --configs) over the GPUs instead of N replicas")
    ap.add_argument("--no-extras", action="store_true", help="skip the extras: the banded-matrix line, the guided-search comparison, the value-streaming "
                                                              "runner-up (profiling runs: only the tuned variant's launches)")
    ap.add_argument("--variant-filter", default=None,
                    help="comma list of descriptor prefixes the tuner may use (spmv_tune variant_filter), e.g. "
                         "'csr_scalar,csr_vector,sell:,sell_tma,ell,merge,bcsr3,dia:,dia_tma' = everything that still "
                         "reads the matrix values (no constant-coefficient elision)")
    ap.add_argument("--tune-cache", default=None,
                    help="file persisting tuning winners (spmv_tune cache_path); a second run then skips the search")
    ap.add_argument("--profile-one", type=int, default=0, metavar="CFG", help="ncu / sanitizer driver: a few cold applies of one variant (6 = the banded extra workload)")
    ap.add_argument("--variant", default=None, help="--profile-one: descriptor to force ('tuned' or absent: tune)")
    ap.add_argument("--iters", type=int, default=5)
    ap.add_argument("--ceilings", action="store_true", help="run only the library's ceiling kernels (spmv_measure_ceiling) and print them")
    ap.add_argument("--rendezvous-only", action="store_true", help="join the N ranks, count them, print, exit (launch check)")
    args = ap.parse_args()
    args.warmup = max(3, args.warmup)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and not args.profile_one:
        relaunch_under_torchrun(args)           # does not return
    if args.rendezvous_only:
        rendezvous_only(args)
        return

    from paper_1309_1894_b200 import workloads as W
    if args.impl == "reference":
        run_reference(args, W)
        return

    import torch
    from paper_1309_1894_b200 import binding
    binding.lib()                               # fail loudly if the CUDA library is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    if args.profile_one:
        profile_one(args, torch, binding, W)
        return
    if args.ceilings:          # the library's ceiling kernels alone (the command the ceiling captures in profiles/ run)
        torch.cuda.set_device(0)
        print(json.dumps({"copy_gbs_1GiB": binding.measure_ceiling(0, 1 << 30, 5),
                          "read_gbs_1GiB": binding.measure_ceiling(1, 1 << 30, 5),
                          "read_gbs_1777MB": binding.measure_ceiling(1, 1777136820, 5),
                          "blockrow_read_gbs_1684MB": binding.measure_ceiling(4, 1684343232, 7),
                          "empty_launch_us": binding.measure_ceiling(2, 0, 200),
                          "random_gather_G_per_s_32MiB_table": binding.measure_ceiling(3, 1 << 25, 3)}))
        return
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus and rank == 0:
        print(f"bench: --gpus {args.gpus} but the launcher started {world} rank(s); n_gpus = {world}", file=sys.stderr)
    torch.cuda.set_device(local)
    device = f"cuda:{local}"
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(device))
    from paper_1309_1894_b200.dist import make_dist_max
    dist_max = make_dist_max(torch, world, device)

    if args.sharded:
        bench_sharded(args, torch, binding, W, dist_max, device, world, rank)
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return
    cfgs = [int(c) for c in args.configs.split(",")]
    results = []
    for cfg in cfgs:
        res, prob = bench_config(cfg, args, torch, binding, W, dist_max, device, primary=(rank == 0))
        if rank == 0 and not args.no_cpu_baseline:
            res["cpu_baseline"] = cpu_baseline(prob, W)
            if res["members"] > 1:
                res["cpu_baseline"]["sample"] += f" (first of the {res['members']} matrices; GB/s per matrix is the batch's GB/s)"
        results.append(res)
        del prob
    head = results[0]
    peak, peak_src = measured_peak()
    line = {
        "metric": METRIC, "value": head["eff_gbs"] * world, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": head["t_step_us"] * 1e-3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": headline_config(W, head["cfg"], head["rows"], head["nnz"]),
        "guided_search": head["guided_search"], "tune_reference": head["tune_reference"],
        "selection": {"variant": head["variant"], "nstreams": head["nstreams"], "variant_filter": args.variant_filter,
                      "l2": head["timing"],
                      "parallelism": "replicas only (no data-path collective)" if world > 1 else "1 GPU"},
        "timed_batches": head["t_batches_us"]["n"], "timed_region_ms": head["timed_region_ms"],
        "gpu_launches": head["gpu_launches"],
        "clocks": head["clocks"],
        "e2e": {"value": head["e2e"]["value"] * world, "unit": "GB/s",
                "h2d_bytes_per_step": head["e2e"]["h2d_bytes_per_step"],
                "d2h_bytes_per_step": head["e2e"]["d2h_bytes_per_step"],
                "ms_per_step": head["e2e"]["ms_per_step"]},
        "gflops": head["gflops"] * world, "speedup_vs_default": head["speedup_vs_default"],
        "tune_seconds": head["tune_seconds"], "deterministic": head["deterministic"], "parity": head["parity"],
        "host_us_per_apply": head["host_us_per_apply"],
        "per_config": results,
    }
    if rank == 0:
        # ceilings measured in the same run with the library's own kernels
        torch.cuda.synchronize()
        ceil = {"copy_gbs_1GiB": binding.measure_ceiling(0, 1 << 30, 5),
                "read_gbs_1GiB": binding.measure_ceiling(1, 1 << 30, 5),
                "empty_launch_us": binding.measure_ceiling(2, 0, 200),
                "random_gather_G_per_s_32MiB_table": binding.measure_ceiling(3, 1 << 25, 3),
                "bcsr3_value_loads_only_gbs": binding.measure_ceiling(4, 1684343232, 5)}
        line["ceilings"] = ceil
        try:
            cpu_model = [l.split(":", 1)[1].strip() for l in open("/proc/cpuinfo") if l.startswith("model name")][0]
        except Exception:
            cpu_model = "unknown"
        line["host"] = {"cpu_model": cpu_model, "cores": os.cpu_count(), "cuda": torch.version.cuda,
                        "gpu": torch.cuda.get_device_properties(device).name, "torch": torch.__version__}
        for r in results:
            r["roofline"] = config_roofline(r, peak, ceil)
            r["roofline"]["peak_source"] = peak_src if r["roofline"]["bound"] == "hbm" else "measured in this run (spmv_measure_ceiling)"
        line["roofline"] = dict(head["roofline"], kernel=head["variant"])
        line["cpu_baseline"] = head.get("cpu_baseline")
        line["cg"] = next((r["cg"] for r in results if r["cg"]), None)
        if not args.no_extras:
            line["banded"] = bench_banded(args, torch, binding, W, device)
        detail = write_detail(line)
        sys.stdout.flush()
        print(json.dumps(compact_line(line, detail), separators=(",", ":")), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

"""bench.py's output contract, checked without a GPU: the last stdout line is a compact JSON object (the driver
could not parse round 2's 22 KB line), both arms print the same `config`, and `--gpus N` starts N ranks."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _canned(n_cfg=5):
    per = []
    for c in range(1, n_cfg + 1):
        per.append({"cfg": c, "variant": "sell16_tma:b288:c512:s8192:l128:r2:u16:i6:x3:h4096:g8:co100", "t_step_us": 275.94876543,
                    "eff_gbs": 9348.123456, "parity": {"ok": True},
                    "roofline": {"bound": "l1-xbar gather requests", "frac": 0.98123456},
                    "with_values": {"variant": "dia_tma:b288:c256:r1:u8:i3:x0:g2", "t_us": 34.123456, "frac_actual_of_measured": 0.91234},
                    "tune_reports": [{"log": "x" * 5000}]})
    return {"metric": bench.METRIC, "value": 9348.123456789, "unit": "GB/s", "n_gpus": 1, "steps": 50, "warmup": 10,
            "ms_per_step": 0.27594876, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": "cfg4: FEM 27-pt x 3x3 blocks, 96^3 nodes, alpha=1 beta=0",
                                            "rows": 2654208, "nnz": 210542904, "l2": "inputs >= 4x L2 (126 MB): every step streams from HBM, no flush"},
            "roofline": {"bound": "hbm", "achieved": 6440.123, "peak": 6542.7, "unit": "GB/s", "frac": 0.98432,
                         "traffic": 1763600000, "bytes_per_launch": 1777136820, "effective_gbs": 9348.1,
                         "kernel": "bcsr3:b128:w16:u2:i16:x0:g8", "note": "n" * 400, "peak_source": "p" * 80},
            "cpu_baseline": {"value": 111.8, "unit": "GB/s", "cores": 16, "kind": "oracle", "sample": "s" * 300,
                             "parallel_seconds": 0.023},
            "e2e": {"value": 3821.0, "unit": "GB/s", "ms_per_step": 0.675, "h2d_bytes_per_step": 21233664,
                    "d2h_bytes_per_step": 21233664, "steps": 50},
            "gpu_launches": 9000, "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 2100.0, "reasons": ["sw_power_cap"], "samples": 107},
            "parity": {"ok": True, "rows_checked": 2654208, "rows": 2654208, "max_err_over_scale": 4.02e-16, "tolerance": 1e-12,
                       "what": "w" * 100},
            "deterministic": True, "gflops": 1525.9, "speedup_vs_default": 3.9, "tune_reference": "oracle",
            "guided_search": {"tune_seconds": 0.61, "winner": "bcsr3:b128:w16:u2:i16:x0:g8", "winner_us": 277.1,
                              "exhaustive_tune_seconds": 4.1, "exhaustive_winner_us": 276.0},
            "per_config": per, "ceilings": {"x": 1.0}, "cg": {"y": "z" * 2000}, "banded": {"b": "b" * 3000}}


def test_compact_line_is_short_and_round_trips():
    full = _canned()
    line = json.dumps(bench.compact_line(full, "gpurun_out/bench_detail.json"), separators=(",", ":"))
    assert len(line) < bench.COMPACT_LIMIT, len(line)
    assert "\n" not in line
    back = json.loads(line)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches"):
        assert k in back, k
    assert back["value"] > 0 and back["config"]["workload"].startswith("cfg4")
    assert set(back["roofline"]) >= {"bound", "achieved", "peak", "unit", "frac", "traffic"}
    assert set(back["e2e"]) >= {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"}
    assert set(back["cpu_baseline"]) >= {"value", "unit", "cores", "kind", "sample"}
    assert back["parity"]["rows_checked"] == back["parity"]["rows"]
    assert back["tune"]["reference"] == "oracle" and back["tune"]["guided_s"] < back["tune"]["exhaustive_s"]
    assert [r["cfg"] for r in back["per_config"]] == [1, 2, 3, 4, 5]
    assert "tune_reports" not in line and "banded" not in back


def test_compact_line_degrades_instead_of_overflowing():
    full = _canned(5)
    for r in full["per_config"]:
        r["variant"] = r["variant"] * 4
        r["with_values"]["variant"] *= 4
    out = bench.compact_line(full, None)
    assert len(json.dumps(out, separators=(",", ":"))) < bench.COMPACT_LIMIT


def test_both_arms_print_the_same_config():
    from paper_1309_1894_b200 import workloads as W
    a = bench.headline_config(W, 4, 2654208, 210542904)
    assert set(a) == {"workload", "rows", "nnz", "l2"} and "no flush" in a["l2"]
    assert "cold" in bench.headline_config(W, 1, 4096, 20224)["l2"]


def test_gpus_n_without_a_launcher_starts_n_ranks():
    """`python bench.py --gpus 2` with WORLD_SIZE unset re-executes itself under torch.distributed.run: two ranks
    join (gloo here, nccl on a GPU box) and rank 0 reports the count."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--rendezvous-only"],
                       capture_output=True, text=True, env=env, timeout=240)
    assert r.returncode == 0, r.stderr[-2000:]
    last = [l for l in r.stdout.splitlines() if l.startswith("{")][-1]
    rec = json.loads(last)
    assert rec == {"ranks_joined": 2, "n_gpus": 2, "world_size": 2}


def test_reference_arm_under_n_ranks_prints_one_line_with_n_gpus():
    """`bench.py --impl reference --gpus 2` (no launcher): two ranks are started, rank 0 alone runs the oracle and prints
    ONE line whose n_gpus and config agree with what the product arm would print for the same workload."""
    from paper_1309_1894_b200 import workloads as W
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2",
                        "--warmup", "3", "--configs", "1"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, lines
    rec = json.loads(lines[0])
    assert rec["impl"] == "reference" and rec["n_gpus"] == 2 and rec["value"] > 0
    assert rec["config"] == bench.headline_config(W, 1, 4096, 20224)
    assert rec["cpu_baseline"]["kind"] == "oracle" and rec["e2e"]["h2d_bytes_per_step"] == 0

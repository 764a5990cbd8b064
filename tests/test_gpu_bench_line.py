"""bench.py prints ONE JSON line with the keys the driver reads (metric, value, roofline, cpu_baseline, e2e, clocks,
gpu_launches, per_config ...): checked here on the smallest workload so that a broken bench shows up in the test run."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]
    d = json.loads(lines[0])
    d["_line_bytes"] = len(lines[0])
    return d


def test_bench_line_has_the_contracted_keys():
    d = run_bench("--workload", "C1", "--steps", "4", "--warmup", "3", "--config-steps", "3", "--e2e-steps", "2")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline", "per_config"):
        assert k in d, k
    assert d["value"] > 0 and d["gpu_launches"] > 0 and d["vs_baseline"] is None and "workload" in d["config"]
    r = d["roofline"]
    for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic", "traffic_source", "phases", "sweep_only", "kernel_ms"):
        assert k in r, k
    assert r["bound"] == "alu" and 0 < r["frac"] < 1
    assert set(r["phases"]["ns_per_spin"]) == {"metropolis", "houdayer", "exchange", "rest"}
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["one_core"]["cores"] == 1
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0 and e["packed_boundary"]["value"] > 0
    assert set(d["per_config"]) == {"C1", "C2", "C3", "C4", "C5"}
    for name in ("C2", "C3", "C4", "C5"):
        pc = d["per_config"][name]
        assert pc["value"] > 100 and 0 < pc["frac"] < 1 and pc["sm_mhz"] is not None and pc["from_mcs0"] > 0
        st = pc["ms_step_stats"]
        assert 0 < st["min"] <= st["median"] <= st["max"]
    # SURVEY 8(d) timing protocol: per-step statistics, the steady-state window and the run from MCS 0
    assert 0 < d["ms_step_stats"]["min"] <= d["ms_step_stats"]["median"] <= d["ms_step_stats"]["max"]
    assert d["timed_window_mcs"][0] >= 128 and d["from_mcs0"]["mcs"][0] == 0 and d["from_mcs0"]["value"] > 0
    # the driver keeps the TAIL of the line: every config's figures sit in `summary`, the last key, and the line is short
    assert list(d)[-2] == "summary" and d["_line_bytes"] < 6144, d["_line_bytes"]
    assert set(d["summary"]) == {"C1", "C2", "C3", "C4", "C5", "G2", "G5"}
    for name, (value, frac, whole) in d["summary"].items():
        assert value > 0 and 0 < whole < 1 and (frac is None or 0 < frac < 1), name


def test_reference_arm_prints_the_oracle_line():
    d = run_bench("--impl", "reference", "--workload", "C1", "--steps", "3", "--warmup", "1")
    assert d["impl"] == "reference" and d["value"] > 0 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0

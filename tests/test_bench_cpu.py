"""bench.py's reference arm (`--impl reference`: the CPU oracle, as it stands, on a bounded sample) runs without a GPU and
prints the contract's JSON line.  The GPU arm is exercised by the driver and by tests/test_multirank_cpu.py (its aggregation)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_reference(extra_env=None):
    env = dict(os.environ)
    env.pop("RANK", None)
    env.update(extra_env or {})
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--steps", "2",
                          "--warmup", "1", "--ref-cols", "2"], cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    return [ln for ln in out.stdout.splitlines() if ln.startswith("{")]


def test_reference_arm_prints_one_contract_line():
    lines = run_reference()
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "chebyshev_filter_throughput"
    assert d["unit"] == "complex_DoF*vectors*degree/s" and d["higher_is_better"] is True
    assert d["steps"] == 2 and d["warmup"] == 1 and d["value"] > 0 and d["ms_per_step"] > 0
    assert d["dtype"] == "f64" and d["data"] == "synthetic" and d["gpu_launches"] == 0
    assert "configs[0]" in d["config"]["workload"] and "sample" in d["config"]
    cb = d["cpu_baseline"]
    assert cb["kind"].startswith("oracle") and cb["cores"] >= 1 and cb["value"] == d["value"] and cb["sample"]
    e2e = d["e2e"]
    assert e2e["value"] == d["value"] and e2e["unit"] == d["unit"]
    assert e2e["h2d_bytes_per_step"] == 0 and e2e["d2h_bytes_per_step"] == 0


def test_reference_arm_only_rank_zero_works():
    # under torchrun the other ranks exit 0 without work and without a line
    assert run_reference({"RANK": "1", "WORLD_SIZE": "2"}) == []

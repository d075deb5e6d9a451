"""bench.py's reference arm runs on the CPU box (it times the oracle): check the JSON line it prints against the
contract (keys, units, the reference-arm additions).  The GPU arm is exercised by the driver on the GPU box."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*extra):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", *extra], capture_output=True, text=True, cwd=ROOT, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    return json.loads(lines[0])


def check_common(d):
    assert d["impl"] == "reference" and d["higher_is_better"] is True and d["unit"] == "planes/s"
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["steps"] == 1 and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["gpu_launches"] == 0 and "workload" in d["config"]


def test_reference_arm_flux_tube_config0():
    d = run_bench("--config", "0")
    check_common(d)
    assert d["metric"] == "ExB nonlinearity planes/s" and d["vs_baseline"] is None


def test_reference_arm_xglobal():
    d = run_bench("--xglobal")
    check_common(d)
    assert "x-global" in d["metric"] and abs(d["vs_baseline"] - d["value"] / 197e3) < 1e-9

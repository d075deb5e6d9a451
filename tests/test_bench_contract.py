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


def test_measured_traffic_rows_are_tied_to_the_cuda_sources(tmp_path, monkeypatch):
    """profiles/dram_traffic.csv rows count only while their src_sha16 equals the hash of the CUDA sources being timed
    ("stamp the CSV row with the hash it was captured at and refuse a mismatch")."""
    sys.path.insert(0, ROOT)
    import bench
    sha = bench.source_sha16()
    assert len(sha) == 16
    prof = tmp_path / "profiles"
    prof.mkdir()
    (prof / "dram_traffic.csv").write_text(
        "workload,kernel,dram_bytes_per_launch,planes_per_launch,src_sha16,source\n"
        f"wl_a,k_plane_fused,1000,10,{sha},x\n"
        "wl_b,k_plane_fused,2000,10,0123456789abcdef,x\n")
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    monkeypatch.setattr(bench, "source_sha16", lambda: sha)
    rows, why = bench.measured_traffic("wl_a")
    assert why is None and rows == {"k_plane_fused": (1000.0, 10.0)}
    rows, why = bench.measured_traffic("wl_b")
    assert rows == {} and "predates" in why
    rows, why = bench.measured_traffic("wl_c")
    assert rows == {} and "no ncu capture" in why

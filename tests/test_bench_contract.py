"""bench.py prints ONE JSON line with the keys the driver reads (tiny custom shape; GPU box only)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*extra):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "2", "--warmup", "3", *extra],
                         capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1, out.stdout
    return json.loads(lines[0])


@pytest.mark.gpu
def test_bench_line_has_the_contract_keys():
    d = _run("--shape", "d,700,64,600", "--e2e-steps", "1")
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "roofline", "clocks", "e2e", "gpu_launches", "cpu_baseline"):
        assert key in d, key
    assert d["dtype"] == "f64" and d["n_gpus"] == 1 and d["steps"] == 2 and d["vs_baseline"] is None
    assert d["gpu_launches"] >= 2 * 2 and d["value"] > 0
    r = d["roofline"]
    assert r["bound"] == "tensor" and r["unit"] == "TFLOP/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0
    assert d["checks"]["max_rel_column_norm_drift_after_all_steps"] < 1e-12


@pytest.mark.gpu
def test_bench_chase_line():
    d = _run("--chase", "--shape", "d,700,64,8", "--no-cpu-baseline")
    assert d["metric"].startswith("bulge chase") and d["value"] > 0 and d["gpu_launches"] >= 2
    assert d["checks"]["relative_trace_error"] < 1e-13


def test_bench_reference_arm_runs_on_cpu():
    d = _run("--impl", "reference", "--shape", "d,300,32,64", "--steps", "1", "--warmup", "0")
    assert d["impl"] == "reference" and d["value"] > 0 and d["gpu_launches"] == 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["cpu_baseline"]["kind"] == "oracle"


@pytest.mark.gpu
def test_bench_default_line_times_chase_reflectors():
    d = _run("--shape", "d,700,64,600", "--e2e-steps", "0", "--no-cpu-baseline")
    assert d["config"]["reflectors"].startswith("GPU bulge chase")
    d = _run("--shape", "d,700,64,600", "--e2e-steps", "0", "--no-cpu-baseline", "--reflectors", "synthetic")
    assert d["config"]["reflectors"].startswith("synthetic")


@pytest.mark.gpu
def test_bench_other_lines():
    d = _run("--dtype", "f32", "--shape", "z,500,64,300", "--e2e-steps", "1")
    assert d["dtype"] == "f32" and d["roofline"]["bound"] == "alu" and d["gpu_launches"] >= 2 and "FP32" in d["metric"]
    assert d["checks"]["max_rel_column_norm_drift_after_all_steps"] < 1e-4
    d = _run("--step", "6e", "--shape", "z,600,64,300", "--e2e-steps", "1")
    assert d["metric"].startswith("band->full") and d["roofline"]["kernel"].startswith("bt_b2fz_kernel")
    d = _run("--row-pipeline", "3", "--shape", "d,900,64,200")
    assert d["scaling"] == "strong" and d["config"]["halo_messages_per_step"] > 0 and d["value"] > 0

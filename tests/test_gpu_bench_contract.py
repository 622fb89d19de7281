"""`-m gpu`: `python bench.py` prints ONE JSON line with the keys the measurement contract names (metric, value, unit,
n_gpus, steps, warmup, ms_per_step, higher_is_better, scaling, vs_baseline, dtype, data, config.workload, clocks, e2e with
its byte counts, gpu_launches > 0, roofline with bound / achieved / peak / frac / traffic, cpu_baseline with kind =
"oracle"), and the numbers in it hang together.  Run on configs[1] (9,000 atoms) so that the test takes seconds."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*extra):
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "1", "--steps", "40", "--warmup", "3", *extra],
                         capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-3000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


def test_bench_line_has_the_contracts_keys_and_consistent_numbers():
    d = _run("--no-scan")
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert key in d, key
    assert d["metric"] == "pair_interactions_per_s" and d["unit"] == "pair interactions/s" and d["higher_is_better"] is True
    assert d["n_gpus"] == 1 and d["steps"] == 40 and d["warmup"] >= 3 and d["scaling"] == "weak" and d["vs_baseline"] is None
    assert d["dtype"] == "f32" and d["data"] == "synthetic" and "configs[1]" in d["config"]["workload"]
    assert "model" not in d["config"]
    # value = in-cutoff pairs x steps / time
    assert d["value"] == pytest.approx(d["config"]["pairs_in_cutoff"] / (d["ms_per_step"] * 1e-3), rel=1e-6)
    assert d["gpu_launches"] >= 4 * d["steps"]  # trigger, gather, pair kernel, finalize per step at least
    c = d["clocks"]
    assert c["sm_mhz"] > 0 and c["sm_max_mhz"] >= c["sm_mhz"] and isinstance(c["reasons"], list)
    e = d["e2e"]
    n = d["config"]["n_atoms"]
    assert e["h2d_bytes_per_step"] >= 12 * n and e["d2h_bytes_per_step"] >= 12 * n and e["unit"] == d["unit"]
    assert 0 < e["value"] < d["value"]  # host copies inside the timed region cannot make it faster
    r = d["roofline"]
    assert r["bound"] in ("alu", "hbm", "tensor") and r["unit"] in ("TFLOP/s", "GB/s")
    assert r["frac"] == pytest.approx(r["achieved"] / r["peak"], rel=1e-9) and 0 < r["frac"] < 1
    assert r["achieved"] == pytest.approx(r["flops_per_launch"] / (r["kernel_ms"] * 1e-3) * 1e-12, rel=1e-6)
    assert r["kernel"] == "pair_force_f32x2_kernel" and r["kernel_launches_timed"] + r["kernel_launches_skipped_on_device"] >= d["steps"]
    assert d["last_step_check"]["max_dF_over_rms"] < 2e-4 and d["last_step_check"]["dE_over_E"] < 1e-5  # the loop's last forces are real
    b = d["cpu_baseline"]
    assert b["kind"] == "oracle" and b["cores"] >= 1 and b["value"] > 0 and b["unit"] == d["unit"] and b["same_config"] is True
    assert b["value"] < d["value"]


def test_reference_arm_prints_the_oracle_line():
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--steps", "3", "--warmup", "1"],
                         capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-3000:]
    d = json.loads([ln for ln in res.stdout.splitlines() if ln.strip()][-1])
    assert d["impl"] == "reference" and d["metric"] == "pair_interactions_per_s" and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["e2e"]["value"] == d["value"] and d["dtype"] == "f64"

"""bench.py prints ONE JSON line with the keys the measurement contract names, for the CUDA arm
(GPU) and for the reference arm (the oracle, CPU only), on the small configs[0] workload."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                         cwd=ROOT, timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, out.stdout
    return json.loads(lines[0])


def test_reference_arm_line():
    d = run_bench("--impl", "reference", "--config", "0", "--steps", "1", "--warmup", "0", "--cpu-seconds", "1")
    assert d["impl"] == "reference" and d["metric"] == "motor_cell_updates_per_s" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"].startswith("configs[0]") and d["vs_baseline"] is None


@pytest.mark.gpu
def test_cuda_arm_line_and_option_legs():
    d = run_bench("--config", "0", "--steps", "2", "--warmup", "3", "--cpu-seconds", "1", "--spread", "--free")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "roofline_hbm", "cpu_baseline"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 2 and d["scaling"] == "weak" and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["gpu_launches"] > 0 and d["value"] > 0 and d["e2e"]["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    r, h = d["roofline"], d["roofline_hbm"]
    # the fused kernel is bound by FMA issue: peak = the FMA probe of the same run; the HBM side has its own object
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-3
    assert 0 < r["frac"] < 1 and 0.5 * r["peak_nominal"] < r["peak"] < 1.1 * r["peak_nominal"] and "traffic" in r
    assert r["kernel"].startswith("tm<") and r["flops_per_cell_update"] == 12
    assert 0.5 * r["peak"] < r["peak_three_fresh_operands"] < 0.95 * r["peak"]
    assert abs(r["frac_three_fresh_operands"] - r["achieved"] / r["peak_three_fresh_operands"]) < 1e-3
    assert h["bound"] == "hbm" and h["unit"] == "GB/s" and abs(h["frac"] - h["achieved"] / h["peak"]) < 1e-3
    for k in ("frac_nominal_8tbs", "effective_gbs", "effective_frac", "t1_gbs", "t1_frac", "t1_frac_nominal_8tbs"):
        assert k in h, k
    assert abs(h["effective_gbs"] / h["achieved"] - r["fuse_T"]) < 0.6          # a pass carries fuse_T substeps
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
    one = d["cpu_baseline"]["one_thread_configs0"]
    assert one["cores"] == 1 and 0 < one["value"] <= 1.5 * d["cpu_baseline"]["value"]
    assert "per_config" not in d                                                # only the default (no --config) run adds it
    assert d["spread_force"]["ms_per_call"] > 0
    assert d["free_motors"]["update_ms_per_call"] > 0 and d["free_motors"]["coupled_substep_kernel"].startswith("tm_mf<")
    d = run_bench("--config", "0", "--steps", "1", "--warmup", "1", "--no-cpu", "--no-t1", "--scheme", "rk2")
    assert d["roofline"]["kernel"].startswith("rk2_fused<") and d["config"]["workload"].endswith("+rk2_superbee")
    d = run_bench("--config", "0", "--steps", "1", "--warmup", "1", "--no-cpu", "--local-dt")
    assert d["roofline"]["kernel"].startswith("tm_local<") and d["local_dt"]["n_c_max"] >= d["local_dt"]["n_c_min"] >= 1
    d = run_bench("--config", "0", "--steps", "1", "--warmup", "1", "--no-cpu", "--no-t1", "--kernel", "4")
    assert d["roofline"]["kernel"].startswith("coef<")

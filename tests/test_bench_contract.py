"""The JSON line `bench.py` prints: keys and types of the measurement contract, on the small
config so that it runs in seconds.  The reference arm (the oracle on the host cores) needs no GPU; the arm of the
CUDA path is a gpu test."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

COMMON = {"metric": str, "value": float, "unit": str, "n_gpus": int, "steps": int, "warmup": int, "ms_per_step": float,
          "higher_is_better": bool, "scaling": str, "dtype": str, "data": str, "config": dict, "e2e": dict, "cpu_baseline": dict,
          "gpu_launches": int}


def run_bench(*args):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]           # ONE JSON line
    return json.loads(lines[0])


def check_common(d):
    for k, t in COMMON.items():
        assert k in d, k
        assert isinstance(d[k], t) or (t is float and isinstance(d[k], int)), (k, d[k])
    assert d["vs_baseline"] is None                    # the paper prints nothing for this metric on this workload
    assert "workload" in d["config"] and "model" not in d["config"]
    for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"):
        assert k in d["e2e"], k
    for k in ("value", "unit", "cores", "kind", "sample"):
        assert k in d["cpu_baseline"], k
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1


def test_reference_arm_line():
    d = run_bench("--impl", "reference", "--config", "1", "--steps", "2", "--warmup", "1")
    check_common(d)
    assert d["impl"] == "reference" and d["dtype"] == "f64" and d["gpu_launches"] == 0
    assert d["steps"] == 2 and d["warmup"] == 1 and d["value"] > 0
    assert d["e2e"]["value"] == d["value"] and d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["cpu_baseline"]["value"] == d["value"]
    assert d["config"]["workload"].startswith("config 1")


@pytest.mark.gpu
def test_cuda_arm_line():
    d = run_bench("--config", "1", "--steps", "3", "--warmup", "3", "--cpu-baseline-seconds", "0.5")
    check_common(d)
    assert "impl" not in d or d["impl"] != "reference"
    assert d["dtype"] == "f32" and d["gpu_launches"] > 0 and d["value"] > 0
    n = d["config"]["n"]
    assert d["e2e"]["h2d_bytes_per_step"] == 16 * n and d["e2e"]["d2h_bytes_per_step"] == 16 * n and d["e2e"]["value"] > 0
    roof = d["roofline"]
    assert roof["bound"] == "alu" and roof["unit"] == "TFLOP/s" and roof["kernel"] == "mwf::k_force"
    assert abs(roof["frac"] - roof["achieved"] / roof["peak"]) < 1e-12 and 0 < roof["frac"] < 1
    assert "traffic" in roof
    assert "traffic_source" in roof and roof["kernel_ms_min"] <= roof["kernel_ms_median"]
    clk = d["clocks"]
    assert set(("sm_mhz", "sm_max_mhz", "reasons", "samples", "source")) <= set(clk)
    assert d["ms_per_step_min"] <= d["ms_per_step_median"]
    par = d["parity"]                                   # the oracle pass of the cpu_baseline leg, compared with the GPU's result
    assert par["ok"] and par["acc_max"] <= 1e-4 and par["acc_rms"] <= 2e-5 and par["pot_rms"] <= 1e-5 and par["particles"] > 0

"""bench.py's JSON line: the keys the measurement contract asks for.  The reference
arm (the oracle on the host cores) runs without a GPU; the CUDA arm is checked on a small config (-m gpu)."""
import json
import os
import subprocess
import sys

import pytest

from conftest import ROOT

BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
             "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "cpu_baseline"}


def run_bench(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                         cwd=ROOT, timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]
    return json.loads(lines[0])


def test_reference_arm_line():
    d = run_bench("--impl", "reference", "--config", "0", "--steps", "1", "--warmup", "0")
    assert BASE_KEYS <= set(d) and d["impl"] == "reference"
    assert d["unit"] == "pair interactions/s" and d["value"] > 0 and d["higher_is_better"] is True
    assert d["vs_baseline"] is None and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["config"]["workload"] == "c0_tiny_disc" and "model" not in d["config"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and cb["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["gpu_launches"] == 0


@pytest.mark.gpu
def test_cuda_arm_line_small_config():
    d = run_bench("--config", "0", "--steps", "5", "--warmup", "3")
    assert BASE_KEYS | {"roofline", "clocks", "precisions", "alu_probe"} <= set(d)
    assert "impl" not in d and d["n_gpus"] == 1 and d["steps"] == 5 and d["warmup"] == 3
    assert d["dtype"] == "f32" and d["scaling"] == "weak" and d["vs_baseline"] is None
    assert d["config"]["workload"] == "c0_tiny_disc" and "l2" in d["config"]
    r = d["roofline"]
    # frac = 18 (25) flop x ordered pairs / kernel time / peak: the symmetric kernels need fewer executed flops than this
    # convention counts, so it is not bounded by 1 in principle (it is far below at this small N)
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and 0 < r["frac"] < 1.5 and r["peak"] > 70
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and "traffic" in r and r["traffic_source"]
    assert r["peak_measured"] > 60 and abs(r["frac_of_measured"] - r["achieved"] / r["peak_measured"]) < 1e-12
    assert r["fp64"]["peak"] > 35 and 0 < r["fp64"]["frac"] < 1.5 and r["fp64"]["peak_measured"] > 30
    assert r["kernel"] in ("kick32_kernel", "kick32_sym_kernel")
    # the per-config table and the N sweep ride in the same line, every row with its own clock record
    assert [row["config"] for row in d["configs"]] == [0, 1, 2, 3]
    assert [row["N"] for row in d["sweep"]] == [1 << k for k in range(10, 18)]
    for row in d["configs"] + d["sweep"]:
        assert row["clocks"]["sm_max_mhz"] and isinstance(row["clocks"]["rejected"], bool)
        for name in ("fp32", "fp64"):
            assert row[name]["ms_per_step"] > 0 and 0 < row[name]["step_frac_of_peak"] < 1.5 and row[name]["kernel_variant"]
    for row in d["configs"]:
        assert abs(row["fp64"]["dE_over_E"]) < 1e-4 and abs(row["fp64"]["dL_over_L"]) < 1e-11
        assert abs(row["fp32"]["dL_over_L"]) < 1e-8
    e = d["e2e"]
    assert e["e2e_over_device"] > 1.0
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 2048 * 8 * 7 and e["d2h_bytes_per_step"] == 2048 * 8 * 6
    assert e["value"] < d["value"]                                    # copies are inside the timed region
    assert d["gpu_launches"] >= 3 * d["steps"]                        # onbody + all-pairs + near field per step
    c = d["clocks"]
    assert c["sm_max_mhz"] and isinstance(c["reasons"], list)
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] > 0 and cb["sample"]
    for name in ("fp32", "fp64"):
        p = d["precisions"][name]
        assert p["pair_interactions_per_s"] > 0 and p["kernel_ms"]["kick"] > 0
        assert abs(p["dE_over_E"]) < 1e-6 and abs(p["dL_over_L"]) < 1e-8

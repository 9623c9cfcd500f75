"""The bench.py output contract (one JSON line with the keys the driver reads), checked without a GPU:
the reference arm runs here on the CPU oracle; the GPU arm is run for real by the gpu-marked test."""
import json
import os
import subprocess
import sys

import pytest

from conftest import ROOT

BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
             "vs_baseline", "dtype", "data", "config", "e2e", "cpu_baseline", "gpu_launches"}


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--config", "1"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and BASE_KEYS <= set(d)
    assert d["metric"] == "spin_configs_evaluated_per_s" and d["unit"] == "configs/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert "workload" in d["config"] and d["vs_baseline"] is None


@pytest.mark.gpu
def test_gpu_arm_prints_the_contract_keys():
    """The GPU arm, run for real on a 2^38-state prefix of cfg5 (large enough for the tensor-core screen to take the
    bulk): one JSON line with the driver's keys, a self-consistent tensor roofline, live clocks, an e2e leg with
    declared copies and the CPU-oracle baseline. (Full-size numbers are the driver's; this pins the code, not a file.)"""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "0",
                          "--range-log2", "38", "--no-int32"], capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert BASE_KEYS | {"roofline", "clocks", "time_to_S_lowest_s", "evaluated", "value_int32"} <= set(d)
    assert d["metric"] == "spin_configs_evaluated_per_s" and d["unit"] == "configs/s" and d["value"] > 1e12
    r = d["roofline"]
    assert {"bound", "achieved", "peak", "unit", "frac", "traffic"} <= set(r)
    assert r["bound"] == "tensor" and r["unit"] == "TFLOP/s" and r["kernel"] == "ising::zwalk_kernel"
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and 0 < r["frac"] < 1.2
    # the GEMM work of the screen is 2 flop per configuration, counted over the kernel's own launches
    assert abs(r["achieved"] - 2.0 * r["configs_per_s_in_kernel"] * 1e-12) < 1e-6 * r["achieved"]
    assert r["launches"] == 2 and r["blocks_screened"] > 0
    assert d["n_gpus"] == 1 and d["steps"] == 1 and d["gpu_launches"] > 0 and d["config"]["kernel_variant"] == 128
    assert "N=48" in d["config"]["workload"] and "2^38" in d["config"]["workload"]
    assert d["e2e"]["h2d_bytes_per_step"] == (48 * 48 + 48) * 8 and d["e2e"]["d2h_bytes_per_step"] == 100 * 16
    assert d["e2e"]["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert "sm_mhz" in d["clocks"] and "reasons" in d["clocks"]
    assert "bf16" in d["evaluated"] and d["value_int32"] is None          # --no-int32: the int32 pass was skipped

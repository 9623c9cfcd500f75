"""The bench.py output contract (one JSON line with the keys the driver reads), checked without a GPU:
the reference arm runs here on the CPU oracle; the GPU arm's line is checked on the copy stored under profiles/."""
import json
import os
import subprocess
import sys

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


def test_stored_gpu_bench_line_has_the_contract_keys():
    path = os.path.join(ROOT, "profiles", "r02_bench_full.txt")
    line = [l for l in open(path) if l.startswith("{")][-1]
    d = json.loads(line)
    assert BASE_KEYS | {"roofline", "roofline_packed16", "roofline_int32", "clocks", "time_to_S_lowest_s",
                        "per_config"} <= set(d)
    r = d["roofline"]
    assert {"bound", "achieved", "peak", "unit", "frac", "traffic"} <= set(r)
    assert r["bound"] == "tensor" and r["unit"] == "TFLOP/s" and r["kernel"] == "ising::zwalk_kernel"
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and 0 < r["frac"] < 1.2
    # the GEMM work of the screen is 2 flop per configuration, counted over the kernel's own launches
    assert abs(r["achieved"] - 2.0 * r["configs_per_s_in_kernel"] * 1e-12) < 1e-6 * r["achieved"]
    for key in ("roofline_packed16", "roofline_int32"):
        a = d[key]
        assert a["bound"] == "alu" and abs(a["frac"] - a["achieved"] / a["peak"]) < 1e-12 and 0 < a["frac"] < 1
        assert a["same_list_as_default_path"] is True
    assert d["n_gpus"] == 1 and d["steps"] >= 1 and d["warmup"] >= 3 and d["gpu_launches"] > 0
    assert d["clocks"]["reasons"] == [] or set(d["clocks"]["reasons"]) <= {"sw_power_cap"}
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    assert "N=48" in d["config"]["workload"] and len(d["per_config"]) == 5

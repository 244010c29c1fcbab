"""bench.py keeps the driver's JSON contract: one line on stdout with the required keys, for the CUDA arm (gpu) and the
oracle reference arm (CPU)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline", "dtype",
             "data", "config", "e2e", "gpu_launches"}


def _run(args):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True,
                       cwd=ROOT, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1, r.stdout
    return json.loads(lines[0])


def test_reference_arm_line():
    d = _run(["--impl", "reference", "--workload", "C1s", "--steps", "1", "--warmup", "0"])
    assert BASE_KEYS <= set(d) and d["impl"] == "reference"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["value"] > 0 and d["vs_baseline"] is None and d["config"]["workload"] == "C1s"


@pytest.mark.gpu
def test_cuda_arm_line():
    d = _run(["--workload", "C1s", "--steps", "3", "--warmup", "3", "--cpu-seconds", "1"])
    assert BASE_KEYS | {"roofline", "cpu_baseline", "clocks"} <= set(d)
    assert d["value"] > 0 and d["steps"] == 3 and d["n_gpus"] == 1 and d["scaling"] == "weak" and d["dtype"] == "f32"
    rf = d["roofline"]
    assert rf["bound"] in ("hbm", "alu") and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-9
    if rf["bound"] == "alu":      # the fused kernel is instruction-bound: its HBM figures ride along
        hb = d["hbm_roofline"]
        assert hb["bound"] == "hbm" and hb["unit"] == "GB/s" and abs(hb["frac"] - hb["achieved"] / hb["peak"]) < 1e-9
    d2 = _run(["--workload", "C1s", "--steps", "3", "--warmup", "3", "--no-cpu-baseline", "--mode", "onthefly"])
    assert d2["roofline"]["bound"] == "hbm" and d2["roofline"]["unit"] == "GB/s"
    assert d["gpu_launches"] > 0 and d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and "workload" in d["config"]


@pytest.mark.gpu
def test_dense_tp_side_bench_line():
    """bench.py --dense-tp: the dense per-path mix alone on a workload's graph (l_max = 3 runs the paths-outer FMA kernels)"""
    d = _run(["--workload", "C3s", "--dense-tp", "--steps", "2", "--warmup", "3"])
    assert BASE_KEYS | {"roofline", "clocks", "calls"} <= set(d)
    assert d["value"] > 0 and d["gpu_launches"] >= 4 and d["roofline"]["bound"] == "alu"
    assert set(d["calls"]) == {"tp_forward_dense", "tp_backward_dense"} and "l_max=3" in d["config"]["workload"]

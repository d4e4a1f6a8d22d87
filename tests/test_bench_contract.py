"""bench.py's contract on a box without a GPU: the reference arm (the CPU oracle on a bounded sample)
prints one JSON line with the keys the driver reads; the clock sampler parses nvidia-smi rows."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "C2",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["higher_is_better"] is False and d["unit"] == "ms"
    assert d["value"] > 0 and d["n_gpus"] == 1 and d["steps"] == 1
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in d["config"] and "model" not in d["config"]


def test_reference_arm_other_ranks_do_nothing():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                         capture_output=True, text=True, timeout=300, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_clock_sampler_summary():
    sys.path.insert(0, ROOT)
    import bench
    c = bench.ClockSampler(0)
    c.rows = [["1965", "1965", "612.3", "Not Active", "Not Active", "Not Active", "Active"],
              ["1800", "1965", "990.1", "Not Active", "Not Active", "Not Active", "Not Active"],
              ["1950", "1965", "700.0", "Not Active", "Not Active", "Not Active", "Not Active"],
              ["garbage"]]
    s = c.summary()
    assert s["sm_mhz"] == 1950.0 and s["sm_max_mhz"] == 1965.0 and s["reasons"] == ["sw_power_cap"] and s["samples"] == 3


@pytest.mark.gpu
def test_default_arm_line_is_reproducible_by_hand():
    """bench.py on the GPU (configs[0], a few steps): one JSON line with the contract's keys, and a roofline object whose
    numbers follow from each other the way DESIGN.md section 7 says (achieved = algorithmic bytes / kernel time, frac = achieved / peak)."""
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "C1", "--steps", "3", "--warmup", "3",
                          "--no-library-baseline"], capture_output=True, text=True, timeout=600)
    assert res.returncode == 0, res.stderr[-2000:]
    line = json.loads(res.stdout.strip().splitlines()[-1])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "e2e", "gpu_launches", "clocks", "roofline", "cpu_baseline"):
        assert key in line, key
    assert line["config"]["workload"].startswith("C1") and line["higher_is_better"] is False and line["vs_baseline"] is None
    rf = line["roofline"]
    assert rf["bound"] == "hbm" and rf["unit"] == "GB/s"
    assert abs(rf["achieved"] - rf["algorithmic_bytes_per_launch"] / (rf["ms_per_launch"] * 1e-3) / 1e9) <= 1e-6 * rf["achieved"]
    assert abs(rf["frac"] - rf["achieved"] / rf["peak"]) <= 1e-9
    w_bytes = 33 * 4 * 64 * 16 + (32 * 64 + 32 * 4) * 8          # |Fhat| (N_t + 1 frequencies, complex128) + |m| + |d|
    assert rf["algorithmic_bytes_per_launch"] == w_bytes
    assert line["gpu_launches"] == 7 * line["steps"]             # C1 is far below the size where F^T d runs B3 beside B2 (8 kernels)
    assert line["e2e"]["h2d_bytes_per_step"] == (32 * 64 + 32 * 4) * 8
    cb = line["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and "sample" in cb

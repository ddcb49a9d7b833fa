"""The measurement contract of bench.py: both arms print ONE JSON line with the identical `config`, the reference arm
runs only the oracle (CPU), and the product line's roofline arithmetic is consistent (GPU)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
from paper_2205_00856_b200 import workloads as W  # noqa: E402


def run(args, timeout=900):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                         timeout=timeout, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


def test_reference_arm_line():
    line = run(["--impl", "reference", "--steps", "1", "--warmup", "0"])
    cfg = W.CONFIGS["C2dense"]
    assert line["impl"] == "reference" and line["metric"] == bench.METRIC and line["unit"] == bench.UNIT
    assert line["config"] == bench.bench_config(cfg, cfg.P, 1)     # what the product arm prints for the same launch
    assert line["higher_is_better"] is True and line["vs_baseline"] is None and line["gpu_launches"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1
    assert line["cpu_baseline"]["value"] == line["value"] == line["e2e"]["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0


@pytest.mark.gpu
def test_product_arm_line():
    line = run(["--steps", "2", "--warmup", "3", "--cn-per-step", "10", "--no-cpu-baseline", "--no-per-config"])
    cfg = W.CONFIGS["C2dense"]
    assert "impl" not in line and line["metric"] == bench.METRIC and line["n_gpus"] == 1 and line["steps"] == 2
    assert line["config"] == bench.bench_config(cfg, cfg.P, 1)
    assert line["dtype"] == "f64" and line["data"] == "synthetic" and line["scaling"] == "weak"
    r = line["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["traffic_source"]
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert abs(r["achieved"] - r["algorithmic_bytes_per_launch"] / (r["kernel_ms"] * 1e-3) / 1e9) < 1e-6 * r["achieved"]
    assert r["algorithmic_bytes_per_launch"] == 56 * cfg.N
    cn = line["launch"]["cn_steps_per_bench_step"]
    assert r["kernel_ms"] * cn <= line["ms_per_step"] * 1.02      # the dominant kernel fits inside the step it is part of
    # `frac` is on the 56 B per point SURVEY 8d declares; the fused pass moves 48 (it recovers gamma from q), so it is the
    # fraction on the bytes MOVED that a roofline bounds by 1
    assert r["bytes_per_point"] == {"declared_minimum_SURVEY_8d": 56.0, "moved_by_this_formulation": 48.0}
    assert abs(r["frac_on_bytes_moved"] - r["frac"] * 48.0 / 56.0) < 1e-12
    assert 0.3 < r["frac_on_bytes_moved"] < 1.0 and r["whole_step_GBps"] * 48.0 / 56.0 < r["peak"]
    assert abs(line["value"] - cfg.N * cn / (line["ms_per_step"] * 1e-3) / 1e9) < 1e-6 * line["value"]
    assert line["gpu_launches"] >= 2 * (3 * cn - 1)                # pass + reduce + substitute per CN step, two bench steps
    e = line["e2e"]
    assert e["h2d_bytes_per_step"] == e["d2h_bytes_per_step"] == 16 * cfg.N and 0 < e["value"] <= line["value"] * 1.02
    assert "sm_mhz" in line["clocks"] and "reasons" in line["clocks"]

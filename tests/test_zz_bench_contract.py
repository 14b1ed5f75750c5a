"""bench.py prints ONE JSON line with the keys the driver reads (metric, value, unit, e2e, roofline, cpu_baseline, ...).

(Named to run last: it starts bench.py in a subprocess, and pinning tens of GB right after another CUDA process has exited is
what fails transiently on the boxes -- the full-size tests should not follow it.)"""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
             "dtype", "data", "config", "e2e", "gpu_launches"}


def run_bench(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]
    return json.loads(lines[0])


def test_both_arms_print_the_same_metric_and_pick_the_same_workload():
    """The driver divides the two arms' values only when metric and workload agree: one METRIC string serves both, and the
    default (`auto`) workload is a function of the host's MemTotal alone -- the largest configuration it can pin."""
    sys.path.insert(0, ROOT)
    import bench
    name, wl = bench.pick_workload("auto")
    assert (name, wl) == bench.pick_workload("auto")
    total = bench.wl_bytes(wl)
    assert total <= bench.meminfo("MemTotal") - 14 * (1 << 30) or name == "cfg1"
    if name == "cfg5s":
        assert wl["M"] == wl["N"] and wl["M"] % 2048 == 0 and 65536 < wl["M"] <= 163840 and wl["K"] == 8192 and wl["budget"] == 0
    # per rank under torchrun: a smaller share of the host
    n8, w8 = bench.pick_workload("auto", 8)
    assert bench.wl_bytes(w8) <= bench.meminfo("MemTotal") // 8 or n8 == "cfg1"
    d = run_bench("--impl", "reference", "--workload", "cfg1", "--steps", "1", "--warmup", "0")
    assert d["metric"] == bench.METRIC and d["config"]["workload"].startswith("cfg1: ")
    rows, cols = bench.oracle_sample_shape(bench.cfg5_scaled(), 1.5e11)
    assert rows == 512 and cols % 128 == 0 and 1.0e11 < 2.0 * rows * cols * 8192 <= 1.5e11


def test_reference_arm_times_the_oracle_on_the_host_cores():
    """`--impl reference`: the oracle, as it stands, on a bounded sample of the same workload (no GPU needed)."""
    d = run_bench("--impl", "reference", "--workload", "cfg1", "--steps", "2", "--warmup", "1", "--ref-rows", "256")
    assert BASE_KEYS <= set(d) and d["impl"] == "reference"
    assert d["unit"] == "TFLOP/s" and d["value"] > 0 and d["dtype"] == "f64" and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"] and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in d["config"] and "model" not in d["config"] and d["gpu_launches"] == 0


@pytest.mark.gpu
def test_our_arm_carries_roofline_e2e_clocks_and_launch_count():
    d = run_bench("--workload", "cfg1", "--steps", "5", "--warmup", "3", "--cpu-flops", "1e8")
    assert BASE_KEYS | {"roofline", "cpu_baseline", "clocks"} <= set(d) and "impl" not in d
    assert d["n_gpus"] == 1 and d["steps"] == 5 and d["warmup"] >= 3 and d["higher_is_better"] is True and d["scaling"] == "weak"
    assert d["dtype"] == "f64" and d["data"] == "synthetic" and d["vs_baseline"] is None and d["gpu_launches"] > 0
    e = d["e2e"]
    assert e["unit"] == "TFLOP/s" and 0 < e["value"] and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] == 8 * 512 * 512
    assert 0 < e["frac_of_roofline"] <= 1.0 and e["bound"] in ("link", "fp64") and e["link_peaks"]["h2d_GBps"] > 10
    r = d["roofline"]
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and r["peak"] == 37.2 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert "traffic" in r and 0 < r["frac"] <= 1.0 and 30.0 < r["peak_measured"] < 40.0 and "solo_step" in r and "streamk" in r
    assert abs(d["value"] - e["value"]) < 0.05 * e["value"] and d["in_core"]["value"] > 0
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["value"] > 0 and c["cores"] >= 1 and "sample" in c
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"} and not set(d["clocks"]["reasons"]) & {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}
    assert d["config"]["workload"].startswith("cfg1") and "model" not in d["config"]

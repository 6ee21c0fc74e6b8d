"""bench.py's GPU arm on a B200: the JSON contract and the timing protocol (whole sort periods, starting on a sort step),
on the small configurations so that the test takes seconds."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench(*args):
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=900)
    assert p.returncode == 0, p.stderr[-3000:]
    lines = [l for l in p.stdout.strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1, p.stdout[-2000:]
    return json.loads(lines[0])


def test_gpu_arm_line_and_sort_aligned_timed_region():
    d = _bench("--config", "C2", "--steps", "20", "--warmup", "5", "--cpu-particles", "40000", "--cpu-steps", "2", "--e2e-steps", "2")
    assert d["metric"] == "mpcd_particle_steps_per_s" and d["unit"] == "particle-steps/s" and d["higher_is_better"] is True
    assert d["n_gpus"] == 1 and d["scaling"] == "weak" and d["vs_baseline"] is None and d["data"] == "synthetic"
    # the driver's arguments cannot produce a sort-free window: 25 steps timed after 25, one sort inside
    assert d["steps"] == 20 and d["steps_timed"] == 25 and d["warmup"] == 5 and d["warmup_run"] == 25
    assert d["check"]["sorts_in_timed_region"] == 1 and d["check"]["sort_period"] == 25
    w = d["windows"]                                       # >= 5 windows of 25 steps each, the median one reported
    assert w["count"] >= 5 and w["steps_each"] == 25 and w["ms_min"] <= w["ms_median"] <= w["ms_max"]
    assert abs(w["ms_median"] / 25 - d["ms_per_step"]) < 1e-9
    assert abs(d["value"] - d["config"]["particles_per_gpu"] * 25 / (d["ms_per_step"] * 25e-3)) / d["value"] < 1e-9
    assert d["config"]["workload"].startswith("C2") and "model" not in d["config"]
    assert d["gpu_launches"] >= 25 and d["dtype"].startswith("f32")
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["peak"] > 1000 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    # the target's own figure: N * 96 B per step (two-pass model B2) over the whole step, against 8 TB/s and the measured peak
    assert r["b2_bytes_per_step"] == d["config"]["particles_per_gpu"] * 96 and "LSU" in r["limiter"]
    assert abs(r["b2_frac_of_8tbs"] - r["b2_bytes_per_step"] / (d["ms_per_step"] * 1e-3) / 8e12) < 1e-9
    assert abs(r["b2_frac_of_measured"] * r["peak"] - r["b2_frac_of_8tbs"] * 8000.0) < 1e-6
    assert r["kernel_ms"] > 0 and r["kernel_ms"] < d["ms_per_step"] and (r["traffic"] is None or r["traffic"] > 0) and r["traffic_source"]
    e = d["e2e"]
    assert e["unit"] == d["unit"] and e["value"] > 0 and e["value"] < d["value"]
    assert e["h2d_bytes_per_step"] == e["d2h_bytes_per_step"] == d["config"]["particles_per_gpu"] * 36
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] == len(os.sched_getaffinity(0)) and c["value"] == c["all_cores"] > 0 and c["single_thread"] > 0
    assert "sub-box" in c["sample"]
    k = d["clocks"]
    assert k["samples"] >= 1 and k["sm_max_mhz"] >= k["sm_mhz"] > 0 and isinstance(k["reasons"], list)
    assert abs(d["check"]["kT"] - 1.0) < 0.01


def test_gpu_arm_rounds_longer_requests_up_and_honours_the_sort_period():
    d = _bench("--config", "C1", "--steps", "60", "--warmup", "30", "--sort-period", "10", "--no-e2e", "--no-cpu-baseline")
    assert d["steps"] == 60 and d["steps_timed"] == 60 and d["warmup_run"] == 30 and d["check"]["sorts_in_timed_region"] == 6
    d = _bench("--config", "C1", "--steps", "26", "--warmup", "3", "--no-e2e", "--no-cpu-baseline")
    assert d["steps"] == 26 and d["steps_timed"] == 50 and d["warmup_run"] == 25 and d["check"]["sorts_in_timed_region"] == 2
    assert d["e2e"] is None and d["cpu_baseline"] is None

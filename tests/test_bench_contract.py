"""bench.py's reference arm (the CPU oracle on the host cores) and its JSON contract, runnable without a GPU."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args, env=None):
    e = dict(os.environ)
    e.update(env or {})
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=600, env=e)
    assert p.returncode == 0, p.stderr[-2000:]
    return p.stdout.strip().splitlines()


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    lines = _run("--impl", "reference", "--steps", "2", "--warmup", "3", "--ref-particles", "20000")
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "mpcd_particle_steps_per_s" and d["unit"] == "particle-steps/s"
    assert d["higher_is_better"] is True and d["scaling"] == "weak" and d["vs_baseline"] is None and d["data"] == "synthetic"
    assert d["steps"] == 2 and d["warmup"] == 3 and d["n_gpus"] == 1 and d["value"] > 0 and d["ms_per_step"] > 0
    assert d["steps_timed"] == 25 and d["warmup_run"] == 25                      # whole sort periods, as the GPU arm times them
    assert d["config"]["workload"].startswith("C3") and "model" not in d["config"]
    # the line says what ran: a sub-box of the workload, with its size
    side = d["config"]["sample_cells"]
    assert side[0] == side[1] == side[2] and d["config"]["sample_particles"] == side[0] ** 3 * 10 and "sub-box" in d["config"]["sample"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] == 1 and cb["value"] == d["value"] and "sub-box" in cb["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_reference_arm_other_ranks_exit_quietly_and_configs_are_selectable():
    assert _run("--impl", "reference", "--steps", "1", "--warmup", "3", "--ref-particles", "5000", env={"RANK": "1", "WORLD_SIZE": "2"}) == []
    for cfg, word in (("C4", "MPCD-AT"), ("C5", "chains of 50 beads")):
        d = json.loads(_run("--impl", "reference", "--config", cfg, "--steps", "1", "--warmup", "3", "--ref-particles", "20000")[0])
        assert d["config"]["workload"].startswith(cfg) and word in d["config"]["workload"]


def test_all_core_oracle_timing_runs_one_process_per_core():
    sys.path.insert(0, ROOT)
    import bench
    cfg = bench.synth.CONFIGS["C3"]
    value, cores, n_each = bench.oracle_all_cores(cfg, "mixed", 2, 1, (8, 8, 8))
    assert cores == len(os.sched_getaffinity(0)) and value > 0 and n_each == 8 * 8 * 8 * cfg["M"]


def test_ncu_traffic_is_only_quoted_for_the_kernel_sources_it_was_taken_on():
    sys.path.insert(0, ROOT)
    import bench
    assert len(bench.csrc_hash()) == 16
    for row in open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")).read().splitlines()[1:]:
        w = [x.strip() for x in row.split(",")]
        value, lsu, note = bench.ncu_traffic(w[0], w[1], int(w[2]))
        assert (value is not None) == (w[4] == bench.csrc_hash(int(w[2]))) == (lsu is not None), note
        assert lsu is None or 0.0 < lsu <= 1.0
    assert bench.ncu_traffic("C1", "mixed", 0) == (None, None, "no ncu capture committed for this workload")


def test_whole_sort_periods_and_the_b2_byte_model():
    """Both arms round --steps / --warmup up to whole sort periods; the target's byte model is SURVEY.md 8d's B2."""
    sys.path.insert(0, ROOT)
    import bench
    assert [bench.whole_periods(k, 25) for k in (0, 1, 20, 25, 26, 100)] == [25, 25, 25, 25, 50, 100]
    assert bench.whole_periods(7, 0) == 7 and bench.whole_periods(0, 0) == 1 and bench.whole_periods(60, 10) == 60
    assert bench.b2_bytes_per_particle("mixed", "srd") == 96 and bench.b2_bytes_per_particle("fp64", "srd") == 192
    assert bench.b2_bytes_per_particle("mixed", "at") == 100
    # C3 mixed: N * B2 = 7.68 GB, so 70 % of 8 TB/s is 1.37 ms per step = 58 G particle-steps/s
    N = 80_000_000
    t = N * bench.b2_bytes_per_particle("mixed", "srd") / (0.70 * bench.NOMINAL_HBM_GBS * 1e9)
    assert abs(t * 1e3 - 1.371) < 1e-3 and abs(N / t / 1e9 - 58.3) < 0.1
    assert bench.algorithmic_bytes_per_particle("mixed", 10) == 72 and bench.algorithmic_bytes_per_particle("fp64", 10) == 136

#!/usr/bin/env python
"""bench.py -- MPCD particle-steps/s and roofline fraction on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--precision mixed|fp64]
    python bench.py --impl reference ...          # the CPU oracle on the host cores (tier framing (4))
    torchrun --nproc-per-node N bench.py --gpus N # N independent replicas (weak scaling)

A "step" is one full MPCD step (stream, shift, bin, cell sums, [sort every 25], SRD collision) of
the named workload; the default workload is BASELINE config 3 (C3: L = 200, density 10, 80 M
particles, mixed precision) -- the configuration the north-star target is quoted on.  Inputs are
seeded and synthetic (paper recipe) and far larger than L2 (6.4 GB of particle
state vs 126 MB), so no L2 flush is needed between iterations.

Timing protocol ("whole multiples of the sort period so the sort is amortised in"; the sort and
its period are PAPER.md:173, :177-179): the untimed warm-up runs at least --warmup steps and ends on a step
with t % sort_period == 0; the timed region is ONE mpcd_step call of ceil(--steps / sort_period) * sort_period
steps, so it always contains one sort per period whatever --steps says.  The line reports both counts
(`steps` = as requested, `steps_timed` = what the timed call ran and what `ms_per_step` and `value` are computed over,
`warmup` = requested, `warmup_run`) and `check.sorts_in_timed_region`.  The reference arm rounds the same way, so both
arms time the same number of steps.

Prints ONE JSON line (rank 0).  `value` = particle-steps/s with the state resident in HBM, timed
with CUDA events on the library's stream around that mpcd_step call, max over ranks (workloads below 10 M particles: >= 5 such windows,
about one second in all, the median window reported -- `windows`).  `e2e` = the same
metric through the C ABI with HOST buffers: every step copies the state from pinned host memory
(mpcd_set_state), steps, and copies it back (mpcd_get_state).  `roofline` = algorithmic bytes of
the steady-state fused kernel / its live-measured duration, against the measured HBM copy peak.
`cpu_baseline` = the oracle, as it stands, on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads as synth  # noqa: E402
from paper_1801_10187_b200 import replicas  # noqa: E402

METRIC = "mpcd_particle_steps_per_s"
UNIT = "particle-steps/s"

# Algorithmic bytes per particle-step of the steady-state (fused, single-pass) kernel, DESIGN.md
# "Roofline": B1 = read pos, vel + write pos, vel as 16-byte vectors (SURVEY.md 8d "single-pass lower
# bound") + the cell arrays the method must write and read once per step (40 B sums + 40 B u/axis per
# cell) / M.  The cached cell index, the sort and all re-reads are NOT counted.
def algorithmic_bytes_per_particle(precision: str, M: float) -> float:
    vec = 16 if precision == "mixed" else 32
    return 4 * vec + 80.0 / M


# SURVEY.md 8d's headline model: two passes over the particles per step, B2 = 96 B (mixed) / 192 B (fp64) per particle-step
# (read r, v; write r; write + read the cached cell index through v; read v; write v), + 4 B tag read for the AT rule.
# The target sentence of BASELINE.md ("70 % of the HBM roofline") is N * B2 / t_step over 8 TB/s; the fused single-pass
# kernel here moves less than B2, so this figure is a rate of useful work, not of bytes moved.
def b2_bytes_per_particle(precision: str, rule: str) -> float:
    return (96.0 if precision == "mixed" else 192.0) + (4.0 if rule == "at" else 0.0)


NOMINAL_HBM_GBS = 8000.0   # BASELINE.json / SURVEY.md 8d "8 TB/s"


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def csrc_hash(brick: int = 0) -> str:
    """sha256 (first 16 hex digits) over the sources of the step kernel, in name order: what an ncu capture is stamped with
    (the per-particle kernel lives in mpcd_device.cuh, mpcd_embedded.cuh and mpcd_kernels.cuh; the brick kernel adds mpcd_brick.cuh)."""
    import hashlib
    d = os.path.join(ROOT, "paper_1801_10187_b200", "csrc")
    h = hashlib.sha256()
    for name in ["mpcd_brick.cuh"] * int(bool(brick)) + ["mpcd_device.cuh", "mpcd_embedded.cuh", "mpcd_kernels.cuh"]:
        h.update(name.encode())
        with open(os.path.join(d, name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def ncu_traffic(workload: str, precision: str, brick: int):
    """DRAM bytes per launch of the step kernel (dram__bytes_read.sum + dram__bytes_write.sum) and the busy fraction of its
    actual limiter, the SM's LSU data pipe (l1tex__data_pipe_lsu_wavefronts, % of peak), from the committed `ncu --set full`
    summary profiles/ncu_traffic.csv (workload,precision,brick,bytes,csrc_hash,lsu_pipe_pct,source).  A capture is only
    quoted for the kernel sources it was taken on: returns (bytes or None, lsu pipe fraction or None, note)."""
    found = None
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            for line in f:
                w = [x.strip() for x in line.split(",")]
                if len(w) >= 6 and w[0] == workload and w[1] == precision and w[2] == str(int(brick)):
                    found = (float(w[3]), w[4], float(w[5]) / 100.0)
    except Exception:
        pass
    if found is None:
        return None, None, "no ncu capture committed for this workload"
    if found[1] != csrc_hash(brick):
        return None, None, f"ncu capture is of kernel sources {found[1]}, the tree is {csrc_hash(brick)}: not quoted"
    return found[0], found[2], f"ncu --set full capture of kernel sources {found[1]} (profiles/ncu_traffic.csv)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the GPU arm (B200_PROFILING.md recipe), sampled every 10 ms from
    before the warm-up to after the per-kernel timing leg (all of it back-to-back GPU work around the timed region).
    `sm_mhz` is the median over the samples taken under load (utilization.gpu >= 50 %, which nvidia-smi averages over its own
    window and so lags, or power.draw >= 250 W)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,utilization.gpu,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, None

    def __enter__(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "10"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
            t0 = time.time()                      # the first sample arrives once nvidia-smi has attached to the device
            while time.time() - t0 < 3.0 and os.path.getsize(self.path) == 0:
                time.sleep(0.01)
        except Exception:
            self.proc = None
        return self

    def __exit__(self, *exc):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()

    def summary(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0, "samples_under_load": 0}
        if not self.path:
            return out
        rows, reasons = [], set()
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    rows.append((float(f[1]), float(f[2]), float(f[3]), float(f[4])))
                except ValueError:
                    continue
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if rows:
            load = [r for r in rows if r[3] >= 50.0 or r[2] >= 250.0] or rows
            out.update(sm_mhz=float(np.median([r[0] for r in load])), sm_max_mhz=float(max(r[1] for r in rows)), reasons=sorted(reasons),
                       samples=len(rows), samples_under_load=len([r for r in rows if r[3] >= 50.0 or r[2] >= 250.0]), power_w_max=float(max(r[2] for r in rows)))
        return out


def oracle_sample(cfg, precision, steps, warmup, n_sample, barrier=None):
    """The oracle, as it stands, on a bounded sample of the workload: the same recipe (density, rule,
    parameters, sort period) in a smaller box.  Returns (particle-steps/s, seconds per step, N)."""
    from oracle import oracle as O
    dtype = np.float32 if precision == "mixed" else np.float64
    pos, vel, tag = synth.solvent(n_sample, cfg["M"], seed=cfg["seed"], dtype=dtype)
    o = O.OracleMPCD([float(x) for x in n_sample], pos.shape[0], seed=cfg["seed"], dtype=dtype, init=False,
                     rule=1 if cfg["rule"] == "at" else 0, sort_period=25)
    o.set_state(pos, vel, tag)
    if "chains" in cfg:      # the same bead : solvent ratio in the sample box
        ch = cfg["chains"]
        nch = max(1, round(ch["n_chains"] * pos.shape[0] / (cfg["n"][0] * cfg["n"][1] * cfg["n"][2] * cfg["M"])))
        bp, bv, bm = synth.chains(n_sample, nch, ch["chain_len"], seed=cfg["seed"] + 1, mass=ch["mass"], r0=ch["r0"])
        o.set_embedded(bp, bv, bm, ch["chain_len"], ch["k"], ch["r0"], ch["md_substeps"])
    for _ in range(warmup):
        o.step()
    if barrier is not None:
        barrier.wait()
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step()
    dt = time.perf_counter() - t0
    return pos.shape[0] * steps / dt, dt / steps, pos.shape[0]


def _oracle_worker(cfg, precision, steps, warmup, n_sample, seed_offset, barrier, queue):
    """One process of the all-core timing: its own box (own seed), the oracle as it stands; all processes leave the
    barrier together, so the boxes are stepped at the same time and share the host's memory bandwidth."""
    cfg = dict(cfg, seed=cfg["seed"] + seed_offset)
    try:
        queue.put(oracle_sample(cfg, precision, steps, warmup, n_sample, barrier=barrier))
    except Exception as e:                                   # a worker that dies must not hang the others at the barrier
        try:
            barrier.abort()
        except Exception:
            pass
        queue.put(("error", repr(e), 0))


def oracle_all_cores(cfg, precision, steps, warmup, n_sample):
    """The oracle on ALL host cores (SURVEY.md 8d "Oracle timing beside it" (b); the paper's own CPU runs are one MPI rank
    per core, each with its own sub-domain): one process per core, each stepping an independent
    sub-box of the workload -- the unmodified single-threaded oracle, replicated, with no communication at all, which is
    an upper bound for a domain-decomposed CPU run.  Returns (aggregate particle-steps/s, cores, particles per process)."""
    import multiprocessing as mp
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    ctx = mp.get_context("spawn")                            # never fork a process that holds a CUDA context
    barrier, queue = ctx.Barrier(cores), ctx.Queue()
    procs = [ctx.Process(target=_oracle_worker, args=(cfg, precision, steps, warmup, n_sample, 1000 + k, barrier, queue)) for k in range(cores)]
    for p in procs:
        p.start()
    res = [queue.get() for _ in procs]
    for p in procs:
        p.join()
    bad = [r for r in res if r[0] == "error"]
    if bad:
        raise RuntimeError(f"all-core oracle timing failed: {bad[0][1]}")
    slowest = max(r[1] for r in res)                         # seconds per step of the slowest process
    return sum(r[2] for r in res) / slowest, cores, res[0][2]


def whole_periods(steps: int, period: int) -> int:
    """max(steps, 1) rounded up to whole sort periods (period 0 = no sort: unchanged)."""
    steps = max(int(steps), 1)
    return -(-steps // period) * period if period > 0 else steps


def sample_box(cfg, target_particles):
    """Cubic sub-box of about target_particles at the workload's density."""
    side = max(4, int(round((target_particles / cfg["M"]) ** (1.0 / 3.0))))
    side = min(side, min(cfg["n"]))
    return (side, side, side)


def run_reference(args, cfg, rank, world):
    if rank != 0:
        return 0
    n_sample = sample_box(cfg, args.ref_particles)
    warm_run, timed = whole_periods(args.warmup, 25), whole_periods(args.steps, 25)      # as the GPU arm: both arms time the same number of steps
    value, sec_per_step, Ns = oracle_sample(cfg, args.precision, timed, warm_run, n_sample)
    sample = f"{n_sample[0]}^3-cell sub-box of {args.config} at the same density ({Ns} particles), {timed} steps after {warm_run} warm-up, sort every 25"
    config = workload_config(args, cfg)
    config.update({"sample": "each step advances a sub-box of the workload, not the whole box (tier framing: bounded sample)",
                   "sample_cells": [int(x) for x in n_sample], "sample_particles": int(Ns)})
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "steps_timed": timed,
        "warmup": args.warmup, "warmup_run": warm_run, "ms_per_step": sec_per_step * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32 state / f64 cell sums + collision" if args.precision == "mixed" else "f64",
        "data": "synthetic", "config": config,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_config(args, cfg):
    n = cfg["n"]
    solute = ""
    if "chains" in cfg:
        ch = cfg["chains"]
        solute = (f" + {ch['n_chains']} chains of {ch['chain_len']} beads (mass {ch['mass']:g}, harmonic bonds k={ch['k']:g}, r0={ch['r0']:g}, "
                  f"{ch['md_substeps']} velocity-Verlet substeps per collision) joining the collisions")
    return {"workload": f"{args.config}: MPCD-{cfg['rule'].upper()} solvent{solute}, {n[0]}x{n[1]}x{n[2]} cells (a=1), density {cfg['M']}, "
                        f"{n[0] * n[1] * n[2] * cfg['M']} particles, alpha=130deg, dt=0.1, random grid shift, sort every 25, {args.precision} precision",
            "particles_per_gpu": n[0] * n[1] * n[2] * cfg["M"], "cells_per_gpu": n[0] * n[1] * n[2],
            "precision": args.precision, "cell_energy": bool(args.cell_energy), "thermostat": bool(args.thermostat),
            "parallelism": f"replicas x{args.gpus} (one GPU per box, no data-path collective)",
            "l2_policy": "working set (6.4 GB mixed / 11.5 GB fp64 at C3) >> 126 MB L2; no flush needed"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=25)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C3", choices=sorted(synth.CONFIGS))
    ap.add_argument("--precision", default="mixed", choices=["mixed", "fp64"])
    ap.add_argument("--cell-energy", type=int, default=1)
    ap.add_argument("--sort-period", type=int, default=25)
    ap.add_argument("--brick", type=int, default=0, help="1: brick-major sort order + the brick-tiled step kernel")
    ap.add_argument("--thermostat", type=int, default=0, help="1: Maxwell-Boltzmann cell thermostat on (SRD rule; for profiling cell_thermostat and the kThermo kernels)")
    ap.add_argument("--min-ms", type=float, default=None,
                    help="repeat the timed window until the windows add up to this many ms (then at least 5 windows, the median reported); "
                         "default: 1000 for workloads below 10 M particles, whose single window is too short for the 10 ms clock sampler, "
                         "0 (one window of exactly the whole sort periods asked for, as in rounds 1-2) for the large ones")
    ap.add_argument("--max-windows", type=int, default=400)
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-particles", type=int, default=8_000_000, help="cpu_baseline sample size (particles)")
    ap.add_argument("--cpu-steps", type=int, default=40)
    ap.add_argument("--ref-particles", type=int, default=2_000_000, help="--impl reference sample size per step")
    args = ap.parse_args()
    cfg = synth.CONFIGS[args.config]
    if args.min_ms is None:
        args.min_ms = 1000.0 if cfg["n"][0] * cfg["n"][1] * cfg["n"][2] * cfg["M"] < 10_000_000 else 0.0
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        return run_reference(args, cfg, rank, world)

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    from paper_1801_10187_b200 import MPCD

    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        replicas.barrier(dist if world > 1 else None)
        torch.cuda.synchronize(dev)

    dtype = np.float32 if args.precision == "mixed" else np.float64
    n, M = cfg["n"], cfg["M"]
    seed = replicas.replica_seed(cfg["seed"], rank)
    pos, vel, tag = synth.solvent(n, M, seed=seed, dtype=dtype)
    N = pos.shape[0]
    sim = MPCD([float(x) for x in n], N, seed=seed, precision=args.precision, rule=cfg["rule"], sort_period=args.sort_period,
               cell_energy=bool(args.cell_energy), init_state=False, brick=bool(args.brick), thermostat=bool(args.thermostat), device=f"cuda:{local_rank}")
    sim.set_state(pos, vel, tag)
    if "chains" in cfg:
        ch = cfg["chains"]
        bp, bv, bm = synth.chains(n, ch["n_chains"], ch["chain_len"], seed=seed + 1, mass=ch["mass"], r0=ch["r0"])
        sim.set_embedded(bp, bv, bm, ch["chain_len"], ch["k"], ch["r0"], ch["md_substeps"])

    # ---- device-resident throughput: whole sort periods, starting on a sort step ----
    P = max(args.sort_period, 0)
    warm_run, timed = whole_periods(args.warmup, P), whole_periods(args.steps, P)
    if warm_run < 3:
        raise SystemExit("bench.py: at least 3 warm-up steps are required (timing rules); give --warmup >= 3")
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local_rank) as clocks:
        sim.step(warm_run)                                    # ends on t % P == 0: the timed call starts with a sort step
        barrier()
        st0 = sim.stats()
        barrier()
        ev0.record()
        sim.step(timed)
        ev1.record()
        barrier()
        ms = ev0.elapsed_time(ev1)
        st1 = sim.stats()
        # SURVEY.md 8d "median of >= 5 windows", for the small configurations (--min-ms): the same timed call repeated (every window
        # again whole sort periods starting on a sort step) until the windows add up to about a second, so that a workload whose
        # window is a few ms is timed over a stretch in which the 10 ms clock sampler sees the GPU under load.  All ranks run the
        # same number of windows.  The large configurations keep ONE window of exactly the steps asked for.
        _, ms_first = replicas.whole_job_throughput(float(N) * timed, ms, dist if world > 1 else None, dev)
        windows = [ms]
        nwin = min(max(int(math.ceil(args.min_ms / max(ms_first, 1e-3))), 5), args.max_windows) if args.min_ms > 0 else 1
        for _ in range(nwin - 1):
            barrier()
            ev0.record()
            sim.step(timed)
            ev1.record()
            barrier()
            windows.append(ev0.elapsed_time(ev1))
        ms = float(np.median(windows))
        # ---- per-kernel durations, live, CUDA events on the library's stream, over one more whole sort period ----
        sim.set_profiling(True)
        sim.step(max(P, 1) + 1)
        prof = sim.get_profile()
        sim.set_profiling(False)
    launches = st1["kernel_launches"] - st0["kernel_launches"]
    sorts_timed = st1["sorts"] - st0["sorts"]
    value, ms_max = replicas.whole_job_throughput(float(N) * timed, ms, dist if world > 1 else None, dev)

    fused_ms = prof["fused"][0] / max(prof["fused"][1], 1)
    per_step_ms = {k: (v[0] / max(v[1], 1), v[1]) for k, v in prof.items() if v[1]}
    peak, peak_src = measured_peak()
    algo = algorithmic_bytes_per_particle(args.precision, M) * N
    achieved = algo / (fused_ms * 1e-3) / 1e9 if fused_ms > 0 else 0.0
    traffic, lsu_frac, traffic_note = ncu_traffic(args.config, args.precision, args.brick)
    kernel = "brick_pass" if args.brick else "particle_pass"
    step_s = ms_max / timed * 1e-3
    b2 = b2_bytes_per_particle(args.precision, cfg["rule"]) * N
    lsu_note = f"ncu: l1tex__data_pipe_lsu_wavefronts {100 * lsu_frac:.0f} % busy" if lsu_frac else "no ncu capture of this workload on these kernel sources"
    roofline = {"bound": "hbm", "limiter": f"HBM is the roofline the fraction is taken against; what the kernel actually saturates first is the SM's LSU data pipe ({lsu_note}; DESIGN.md 5.1)",
                "kernel": f"{kernel}<collide+stream+bin+accumulate> (steady-state fused step)",
                "achieved": achieved, "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": traffic_note, "lsu_data_pipe_busy_frac_ncu": lsu_frac, "algorithmic_bytes_per_launch": algo,
                "kernel_ms": fused_ms, "kernel_share_of_step": fused_ms / (ms_max / timed),
                "stage_ms_per_launch": {k: round(v[0], 4) for k, v in per_step_ms.items()},
                "whole_step_frac": algo / step_s / 1e9 / peak,
                # the target's own figure: N * B2 / t_step, sort included, against 8 TB/s and against the measured copy peak
                "b2_bytes_per_step": b2, "b2_gbs": b2 / step_s / 1e9, "b2_frac_of_8tbs": b2 / step_s / 1e9 / NOMINAL_HBM_GBS,
                "b2_frac_of_measured": b2 / step_s / 1e9 / peak}

    # ---- end to end through the C ABI with host buffers ----
    e2e = None
    if not args.no_e2e:
        st = sim.get_state(cell=False)
        bufs = []
        for _ in range(2):                                    # two sets of pinned host buffers: a step's output set is the next step's input set
            bufs.append({"pos": torch.empty((N, 4), dtype=torch.float32 if dtype == np.float32 else torch.float64).pin_memory(),
                         "vel": torch.empty((N, 4), dtype=torch.float32 if dtype == np.float32 else torch.float64).pin_memory(),
                         "tag": torch.empty(N, dtype=torch.int32).pin_memory()})
        bufs[0]["pos"].copy_(torch.from_numpy(st["pos"])); bufs[0]["vel"].copy_(torch.from_numpy(st["vel"]))
        bufs[0]["tag"].copy_(torch.from_numpy(st["tag"].view(np.int32)))
        step0 = st["step"]
        del st

        def one(k):
            src, dst = bufs[k & 1], bufs[(k & 1) ^ 1]
            sim.set_state(src["pos"], src["vel"], src["tag"], step=step0 + k)   # H2D from pinned host memory
            sim.step(1)
            sim.get_state(out=dst)                                              # D2H of the step's result (tags travel: a sort step permutes them)
        one(0)
        barrier()
        t0 = time.perf_counter()
        for k in range(args.e2e_steps):
            one(1 + k)
        barrier()
        wall = time.perf_counter() - t0
        t = torch.tensor([wall], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        nbytes = int(sum(bufs[0][k].numel() * bufs[0][k].element_size() for k in ("pos", "vel", "tag")))
        e2e = {"value": world * N * args.e2e_steps / float(t.item()), "unit": UNIT,
               "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
               "steps": args.e2e_steps, "ms_per_step": float(t.item()) / args.e2e_steps * 1e3,
               "note": "mpcd_set_state(pinned host) + mpcd_step(1) + mpcd_get_state(pinned host) per step; the output buffers of a step are the input buffers of the next"}
        del bufs

    Pm, KE, kT = sim.get_thermo()
    stats = sim.stats()
    sim.close()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n_sample = sample_box(cfg, args.cpu_particles)
        v1, sps, Ns = oracle_sample(cfg, args.precision, args.cpu_steps, 1, n_sample)
        n_each = sample_box(cfg, max(args.cpu_particles // 4, 1))
        vall, cores, Ne = oracle_all_cores(cfg, args.precision, args.cpu_steps, 1, n_each)
        cpu = {"value": vall, "unit": UNIT, "cores": cores, "kind": "oracle", "single_thread": v1, "all_cores": vall,
               "sample": f"single_thread: {n_sample[0]}^3-cell sub-box of {args.config} at the same density ({Ns} particles), {args.cpu_steps} steps after 1 warm-up, "
                         f"{sps * args.cpu_steps:.1f} s of CPU work; all_cores: {cores} processes (one per host core), each the unmodified oracle on its own "
                         f"{n_each[0]}^3-cell sub-box ({Ne} particles), {args.cpu_steps} steps started together, aggregate = particles of all boxes / slowest process's time per step"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "steps_timed": timed,
            "warmup": args.warmup, "warmup_run": warm_run, "ms_per_step": ms_max / timed, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "windows": {"count": len(windows), "steps_each": timed, "ms_min": float(min(windows)), "ms_median": float(np.median(windows)), "ms_max": float(max(windows)),
                        "note": "value and ms_per_step are over the median window of this rank, max over ranks; gpu_launches counts one window"},
            "dtype": "f32 state / f64 cell sums + collision" if args.precision == "mixed" else "f64",
            "data": "synthetic", "config": workload_config(args, cfg),
            "clocks": clocks.summary(), "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "cpu_baseline": cpu,
            "check": {"kT": kT, "momentum_per_particle": float(np.max(np.abs(Pm)) / N), "sorts": stats["sorts"], "sorts_in_timed_region": int(sorts_timed), "sort_period": P, "max_occupancy": stats["max_occupancy"]},
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())

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

Prints ONE JSON line (rank 0).  `value` = particle-steps/s with the state resident in HBM, timed
with CUDA events on the library's stream around mpcd_step(K), max over ranks.  `e2e` = the same
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


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(workload: str, precision: str):
    """DRAM bytes per launch of the fused kernel (dram__bytes_read.sum + dram__bytes_write.sum) from the
    committed `ncu --set full` summary profiles/ncu_traffic.csv (workload,precision,bytes,source), if any."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            for line in f:
                w = [x.strip() for x in line.split(",")]
                if len(w) >= 3 and w[0] == workload and w[1] == precision:
                    return float(w[2])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, None

    def __enter__(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
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
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if not self.path:
            return out
        sm, mx, reasons, power = [], [], set(), []
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    sm.append(float(f[1])); mx.append(float(f[2])); power.append(float(f[3]))
                except ValueError:
                    continue
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=float(max(power)))
        return out


def oracle_sample(cfg, precision, steps, warmup, n_sample):
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
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step()
    dt = time.perf_counter() - t0
    return pos.shape[0] * steps / dt, dt / steps, pos.shape[0]


def sample_box(cfg, target_particles):
    """Cubic sub-box of about target_particles at the workload's density."""
    side = max(4, int(round((target_particles / cfg["M"]) ** (1.0 / 3.0))))
    side = min(side, min(cfg["n"]))
    return (side, side, side)


def run_reference(args, cfg, rank, world):
    if rank != 0:
        return 0
    n_sample = sample_box(cfg, args.ref_particles)
    value, sec_per_step, Ns = oracle_sample(cfg, args.precision, args.steps, args.warmup, n_sample)
    sample = f"{n_sample[0]}^3-cell sub-box of {args.config} at the same density ({Ns} particles), {args.steps} steps after {args.warmup} warm-up, sort every 25"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec_per_step * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32 state / f64 cell sums + collision" if args.precision == "mixed" else "f64",
        "data": "synthetic", "config": workload_config(args, cfg),
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
            "precision": args.precision, "cell_energy": bool(args.cell_energy),
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
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-particles", type=int, default=8_000_000, help="cpu_baseline sample size (particles)")
    ap.add_argument("--cpu-steps", type=int, default=40)
    ap.add_argument("--ref-particles", type=int, default=2_000_000, help="--impl reference sample size per step")
    args = ap.parse_args()
    cfg = synth.CONFIGS[args.config]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.warmup < 3:
        args.warmup = 3

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
               cell_energy=bool(args.cell_energy), init_state=False, device=f"cuda:{local_rank}")
    sim.set_state(pos, vel, tag)
    if "chains" in cfg:
        ch = cfg["chains"]
        bp, bv, bm = synth.chains(n, ch["n_chains"], ch["chain_len"], seed=seed + 1, mass=ch["mass"], r0=ch["r0"])
        sim.set_embedded(bp, bv, bm, ch["chain_len"], ch["k"], ch["r0"], ch["md_substeps"])

    # ---- device-resident throughput ----
    sim.step(args.warmup)
    barrier()
    l0 = sim.stats()["kernel_launches"]
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local_rank) as clocks:
        barrier()
        ev0.record()
        sim.step(args.steps)
        ev1.record()
        barrier()
    ms = ev0.elapsed_time(ev1)
    launches = sim.stats()["kernel_launches"] - l0
    value, ms_max = replicas.whole_job_throughput(float(N) * args.steps, ms, dist if world > 1 else None, dev)

    # ---- per-kernel durations, live, CUDA events on the library's stream ----
    sim.set_profiling(True)
    sim.step(max(args.sort_period, 1) + 1)
    prof = sim.get_profile()
    sim.set_profiling(False)
    fused_ms = prof["fused"][0] / max(prof["fused"][1], 1)
    per_step_ms = {k: (v[0] / max(v[1], 1), v[1]) for k, v in prof.items() if v[1]}
    peak, peak_src = measured_peak()
    algo = algorithmic_bytes_per_particle(args.precision, M) * N
    achieved = algo / (fused_ms * 1e-3) / 1e9 if fused_ms > 0 else 0.0
    roofline = {"bound": "hbm", "kernel": "particle_pass<collide+stream+bin+accumulate> (steady-state fused step)",
                "achieved": achieved, "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak,
                "traffic": ncu_traffic(args.config, args.precision), "algorithmic_bytes_per_launch": algo,
                "kernel_ms": fused_ms, "kernel_share_of_step": fused_ms / (ms_max / args.steps),
                "stage_ms_per_launch": {k: round(v[0], 4) for k, v in per_step_ms.items()},
                "whole_step_frac": algo / (ms_max / args.steps * 1e-3) / 1e9 / peak}

    # ---- end to end through the C ABI with host buffers ----
    e2e = None
    if not args.no_e2e:
        st = sim.get_state(cell=False)
        hp = torch.from_numpy(st["pos"]).pin_memory()
        hv = torch.from_numpy(st["vel"]).pin_memory()
        ht = torch.from_numpy(st["tag"].view(np.int32)).pin_memory()
        out = {"pos": torch.empty_like(hp).pin_memory(), "vel": torch.empty_like(hv).pin_memory()}
        step0 = st["step"]
        del st

        def one(k):
            sim.set_state(hp, hv, ht, step=step0 + k)         # H2D from pinned host memory
            sim.step(1)
            sim.get_state(out=out)                            # D2H of the step's result
            hp.copy_(out["pos"]); hv.copy_(out["vel"])        # the next step's input is this step's output
        one(0)
        barrier()
        t0 = time.perf_counter()
        ev0.record()
        for k in range(args.e2e_steps):
            one(1 + k)
        ev1.record()
        barrier()
        wall = time.perf_counter() - t0
        t = torch.tensor([wall], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e = {"value": world * N * args.e2e_steps / float(t.item()), "unit": UNIT,
               "h2d_bytes_per_step": int(hp.numel() * hp.element_size() + hv.numel() * hv.element_size() + ht.numel() * 4),
               "d2h_bytes_per_step": int(hp.numel() * hp.element_size() + hv.numel() * hv.element_size()),
               "steps": args.e2e_steps, "ms_per_step": float(t.item()) / args.e2e_steps * 1e3,
               "note": "mpcd_set_state(pinned host) + mpcd_step(1) + mpcd_get_state(pinned host) per step; includes a host-side copy of the result into the next input"}
        del hp, hv, ht, out

    P, KE, kT = sim.get_thermo()
    stats = sim.stats()
    sim.close()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n_sample = sample_box(cfg, args.cpu_particles)
        v, sps, Ns = oracle_sample(cfg, args.precision, args.cpu_steps, 1, n_sample)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{n_sample[0]}^3-cell sub-box of {args.config} at the same density ({Ns} particles), {args.cpu_steps} steps after 1 warm-up, "
                         f"{sps * args.cpu_steps:.1f} s of CPU work; host has {os.cpu_count()} cores, the oracle is single-threaded"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 state / f64 cell sums + collision" if args.precision == "mixed" else "f64",
            "data": "synthetic", "config": workload_config(args, cfg),
            "clocks": clocks.summary(), "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "cpu_baseline": cpu,
            "check": {"kT": kT, "momentum_per_particle": float(np.max(np.abs(P)) / N), "sorts": stats["sorts"], "max_occupancy": stats["max_occupancy"]},
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())

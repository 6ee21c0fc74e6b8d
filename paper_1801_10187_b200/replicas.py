"""Host-side logic of the multi-GPU launch: independent replicas, one process per GPU.

north_star: "It runs on one GPU".  The paper's multi-GPU path is spatial domain decomposition with
MPI particle migration and halo-cell exchange; it is out of scope here
(DESIGN.md "Multi-GPU"), so `bench.py --gpus N` runs N independent boxes (weak scaling)
and there is NO data-path collective.  What the ranks share is only bookkeeping: a distinct seed per
rank, a barrier around the timed region, and the whole-job throughput = units all ranks processed /
the slowest rank's time.  This module holds that bookkeeping so that it can be tested with the gloo
backend on CPU (tests/test_replicas_gloo.py).  It contains none of the method's arithmetic.
"""
from __future__ import annotations


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of rank's box: replicas must not simulate the same fluid."""
    return int(base_seed) + int(rank)


def whole_job_throughput(units_local: float, ms_local: float, dist=None, device=None):
    """(units/s over all ranks, max-over-ranks ms).  `dist` is torch.distributed when the process
    group is initialised, else None (single process)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return units_local / (ms_local * 1e-3), ms_local
    import torch
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(u.item()) / (float(t.item()) * 1e-3), float(t.item())


def barrier(dist=None):
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()

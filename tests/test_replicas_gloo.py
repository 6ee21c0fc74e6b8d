"""The N > 1 path of bench.py is "replicas only": this covers its host logic
with two gloo ranks on CPU -- distinct seeds, barrier, whole-job throughput = sum of units / max time."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1801_10187_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        seed = replicas.replica_seed(180110187, rank)
        replicas.barrier(dist)
        # rank 0 "takes" 2 ms for 1000 units, rank 1 4 ms for 3000 units
        value, ms = replicas.whole_job_throughput(1000.0 * (1 + 2 * rank), 2.0 * (1 + rank), dist)
        replicas.barrier(dist)
        q.put((rank, seed, value, ms))
    finally:
        dist.destroy_process_group()


def test_two_replicas_over_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, v0, m0), (r1, s1, v1, m1) = out
    assert (r0, r1) == (0, 1) and s0 != s1 and s0 == 180110187 and s1 == 180110188
    assert m0 == m1 == 4.0                      # max over ranks
    assert v0 == v1 == 4000.0 / 4.0e-3          # all units / slowest rank's time


def test_single_process_needs_no_process_group():
    v, ms = replicas.whole_job_throughput(500.0, 2.0, None)
    assert v == 250000.0 and ms == 2.0
    replicas.barrier(None)

"""Seeded synthetic inputs shared by the tests, bench.py and smoke() -- a module of its own, outside both the product
package and the oracle.

Holds none of the method's arithmetic: only numpy's own generators producing the
paper's workload recipe: positions i.i.d. uniform in the box,
velocity components i.i.d. N(0, kT/m) with the mean velocity removed, tags 0..N-1.
Both the CPU oracle and the CUDA library are fed the arrays made here through their
own set_state calls.
"""
from __future__ import annotations

import numpy as np

# BASELINE.json configs: name -> parameters
CONFIGS = {
    "C1": dict(n=(8, 8, 8), M=5, seed=1801, rule="srd", steps=100),
    "C2": dict(n=(64, 64, 64), M=10, seed=10187, rule="srd", steps=1000),
    "C3": dict(n=(200, 200, 200), M=10, seed=180110187, rule="srd", steps=500),
    "C4": dict(n=(256, 256, 128), M=5, seed=42, rule="at", steps=500),
    # polymer solution: + 1000 chains of 50 beads (mass 5, harmonic bonds k = 1000, r0 = 0.5), 10 MD substeps per collision
    "C5": dict(n=(100, 100, 100), M=5, seed=5, rule="srd", steps=500,
               chains=dict(n_chains=1000, chain_len=50, mass=5.0, k=1000.0, r0=0.5, md_substeps=10)),
}


def solvent(n, M, seed, *, a=1.0, kT=1.0, m=1.0, dtype=np.float32, N=None):
    """Return (pos4, vel4, tag) for a box of n = (nx, ny, nz) cells of edge a at mean
    occupancy M (or an explicit particle count N).  pos4 / vel4 are N x 4 with w = 0."""
    n = tuple(int(x) for x in n)
    if N is None:
        N = n[0] * n[1] * n[2] * int(M)
    rng = np.random.default_rng(seed)
    L = np.array(n, dtype=np.float64) * a
    pos4 = np.zeros((N, 4), dtype=dtype)
    vel4 = np.zeros((N, 4), dtype=dtype)
    chunk = 1 << 22
    mean = np.zeros(3)
    for lo in range(0, N, chunk):
        hi = min(N, lo + chunk)
        p = (rng.random((hi - lo, 3)) * L).astype(dtype)
        for d in range(3):                      # a cast that rounds up to L goes to 0
            p[p[:, d] >= np.asarray(L[d]).astype(dtype), d] = 0
        pos4[lo:hi, :3] = p
        v = rng.standard_normal((hi - lo, 3)) * np.sqrt(kT / m)
        mean += v.sum(axis=0)
        vel4[lo:hi, :3] = v.astype(dtype)
    mean /= N
    for lo in range(0, N, chunk):
        hi = min(N, lo + chunk)
        vel4[lo:hi, :3] = (vel4[lo:hi, :3].astype(np.float64) - mean).astype(dtype)
    tag = np.arange(N, dtype=np.uint32)
    return pos4, vel4, tag


def chains(n, n_chains, chain_len, seed, *, a=1.0, kT=1.0, mass=5.0, r0=0.5):
    """Seeded beads of linear chains for BASELINE config 5: every chain is a random walk of step r0 from a uniform
    random start (wrapped into the box), velocities N(0, kT/mass).  Returns (pos3, vel3, mass) as float64 arrays."""
    rng = np.random.default_rng(seed)
    L = np.array([int(x) for x in n], dtype=np.float64) * a
    start = rng.random((n_chains, 1, 3)) * L
    step = rng.standard_normal((n_chains, chain_len, 3))
    step *= r0 / np.linalg.norm(step, axis=2, keepdims=True)
    step[:, 0, :] = 0.0
    pos = np.mod(start + np.cumsum(step, axis=1), L).reshape(-1, 3)
    pos[pos >= L] = 0.0
    vel = rng.standard_normal((n_chains * chain_len, 3)) * np.sqrt(kT / mass)
    return np.ascontiguousarray(pos), np.ascontiguousarray(vel), np.full(n_chains * chain_len, float(mass))

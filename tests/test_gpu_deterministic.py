"""Deterministic accumulation (PAPER.md:124-126 names fixed-point sums as the alternative to
double): parity with the oracle within the mixed-model tolerance, and the property the mode exists for -- the
trajectory does not depend on the order of particles in memory, of warps or of atomics."""
import math

import numpy as np
import pytest

import workloads as synth

pytestmark = pytest.mark.gpu


def _by_tag(s):
    o = np.argsort(s["tag"], kind="stable")
    return {k: (v[o] if isinstance(v, np.ndarray) else v) for k, v in s.items()}


def test_cell_sums_and_one_step_match_the_oracle(oracle):
    from paper_1801_10187_b200 import MPCD
    n, M = (11, 9, 8), 10
    pos, vel, tag = synth.solvent(n, M, seed=14, dtype=np.float32)
    box = [float(x) for x in n]
    g = MPCD(box, pos.shape[0], seed=14, init_state=False, deterministic=True)
    o = oracle.OracleMPCD(box, pos.shape[0], seed=14, dtype=np.float32, init=False)
    g.set_state(pos, vel, tag); o.set_state(pos, vel, tag)
    g.stream(); o.stream(); g.shift_and_bin(); o.shift_and_bin()
    c = g.get_cells()
    assert np.array_equal(c["count"], o.count) and g.stats()["max_occupancy"] == o.count.max()
    np.testing.assert_allclose(c["sumv"], o.sumv, rtol=0, atol=o.count.max() * 2.0 ** -41)   # exact up to 2^-41 per particle with |v| < 2^-17
    np.testing.assert_allclose(c["ke"], o.ke, rtol=0, atol=o.count.max() * 2.0 ** -41)
    np.testing.assert_allclose(c["u"], o.u, rtol=0, atol=1e-12)
    P, KE, kT = g.get_thermo()
    assert abs(KE - o.ke.sum()) / KE < 1e-12
    g.collide_srd(math.radians(130.0)); o.collide_srd(math.radians(130.0))
    assert np.max(np.abs(g.get_state()["vel"][:, :3].astype(np.float64) - o.vel[:, :3])) <= 1e-5
    g.step(3); o.step(3)                                                   # fused kernels, with a sort
    s = _by_tag(g.get_state()); b = np.argsort(o.tag)
    assert np.max(np.abs(s["vel"][:, :3].astype(np.float64) - o.vel[b][:, :3])) <= 4e-5
    g.close()


@pytest.mark.parametrize("thermostat", [False, True])
def test_trajectory_is_bit_identical_whatever_the_order_in_memory(thermostat):
    """Same fluid, three handles: particles given in creation order with the paper's sort period, in a random order
    with sorts every 2 steps, and in reversed order without sorting.  After 40 steps every tagged particle must have
    bit-identical position and velocity.  (With double accumulators the three differ after a few steps.)"""
    from paper_1801_10187_b200 import MPCD
    n, M = (12, 12, 10), 10
    pos, vel, tag = synth.solvent(n, M, seed=15, dtype=np.float32)
    N = pos.shape[0]
    rng = np.random.default_rng(1)
    orders = [(np.arange(N), 25), (rng.permutation(N), 2), (np.arange(N)[::-1].copy(), 0)]
    states = []
    for perm, sp in orders:
        g = MPCD([float(x) for x in n], N, seed=15, init_state=False, deterministic=True, sort_period=sp, thermostat=thermostat)
        g.set_state(pos[perm], vel[perm], tag[perm])
        g.step(17); g.step(23)
        states.append(_by_tag(g.get_state()))
        g.close()
    for s in states[1:]:
        assert np.array_equal(s["pos"], states[0]["pos"])
        assert np.array_equal(s["vel"][:, :3], states[0]["vel"][:, :3])
        assert np.array_equal(s["cell"], states[0]["cell"])


def test_default_accumulation_is_order_dependent_but_within_tolerance():
    """The contrast: double accumulators give trajectories that agree only within the tolerance at first."""
    from paper_1801_10187_b200 import MPCD
    n, M = (12, 12, 10), 10
    pos, vel, tag = synth.solvent(n, M, seed=15, dtype=np.float32)
    N = pos.shape[0]
    perm = np.random.default_rng(1).permutation(N)
    out = []
    for p in (np.arange(N), perm):
        g = MPCD([float(x) for x in n], N, seed=15, init_state=False, sort_period=0)
        g.set_state(pos[p], vel[p], tag[p]); g.step(2)
        out.append(_by_tag(g.get_state())); g.close()
    assert np.max(np.abs(out[0]["vel"][:, :3] - out[1]["vel"][:, :3])) <= 2e-5


def test_deterministic_needs_mixed_srd_and_no_beads():
    from paper_1801_10187_b200 import MPCD, MPCDError
    for kw in (dict(precision="fp64"), dict(rule="at")):
        with pytest.raises(MPCDError) as e:
            MPCD([4.0] * 3, 100, deterministic=True, **kw)
        assert e.value.code == -1
    g = MPCD([4.0] * 3, 320, seed=1, deterministic=True)
    bp, bv, bm = synth.chains((4, 4, 4), 2, 5, seed=1)
    with pytest.raises(MPCDError):
        g.set_embedded(bp, bv, bm, 5, 1000.0, 0.5, 10)
    g.close()

"""GPU parity for the brick-tiled step kernel (opt.brick = 1; csrc/mpcd_brick.cuh): brick-major sort order, one CTA per
brick, cell means / axes and the next step's sums in shared memory.  Against the oracle element by element, against the per-particle kernel bit for bit with deterministic
accumulation, and on the edge cases of the tiling: boxes smaller than a window, ragged last bricks, a brick that holds
more particles than one chunk, particles that leave the window between two sorts."""
import math

import numpy as np
import pytest

import workloads as synth
from parity_explain import explained_compare

pytestmark = pytest.mark.gpu


def _pair(oracle, n, M, seed, dtype, N=None, kT=1.0, **kw):
    from paper_1801_10187_b200 import MPCD
    pos, vel, tag = synth.solvent(n, M, seed=seed, dtype=dtype, N=N, kT=kT)
    box = [float(x) for x in n]
    g = MPCD(box, pos.shape[0], seed=seed, precision="fp64" if dtype == np.float64 else "mixed", init_state=False, brick=True, **kw)
    g.set_state(pos, vel, tag)
    okw = {k: v for k, v in kw.items() if k in ("dt", "alpha", "sort_period", "thermostat")}
    o = oracle.OracleMPCD(box, pos.shape[0], seed=seed, dtype=dtype, init=False, **okw)
    o.set_state(pos, vel, tag)
    return g, o


def _check(g, o, box, dtype, tol_scale=1.0):
    s = g.get_state()
    a, b = np.argsort(s["tag"], kind="stable"), np.argsort(o.tag, kind="stable")
    assert np.array_equal(s["tag"][a], o.tag[b])
    tol = (1e-12 if dtype == np.float64 else 1e-5) * tol_scale
    return explained_compare(s["pos"][a], s["vel"][a], s["cell"][a], o.pos[b], o.vel[b], o.cell[b], g.get_shift(), 1.0, box, tol, dtype,
                             pos_ulps=2 if dtype == np.float32 else 300)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("n", [(16, 12, 10), (9, 6, 11), (4, 4, 4), (3, 5, 2), (21, 4, 7)])
def test_brick_steps_teacher_forced_against_the_oracle(oracle, dtype, n):
    """Every two steps the oracle restarts from the GPU's state (the GPU handle itself is left alone: mpcd_set_state would
    declare its order arbitrary and switch the brick kernel off until the next sort) and must land on the GPU's state two
    steps later, every mismatch explained.  mpcd_step(2) = one launch of the fused kernel; with a sort every 3 steps the
    launches right after a sort, later ones, and the ones that sort on their way out are all covered."""
    g, o = _pair(oracle, n, 10, 7, dtype, sort_period=3)
    assert g.stats()["brick"][0] > 0
    box = [float(x) for x in n]
    g.step(1)                                           # step 0 sorts: from here on the arrays are in brick order
    for t in range(1, 13, 2):
        st = g.get_state()
        o.set_state(st["pos"], st["vel"], st["tag"], step=t)
        g.step(2); o.step(2)
        r = _check(g, o, box, dtype)
        assert r["bad_cell"] <= (1 if dtype == np.float32 else 0), (t, r)
    assert g.stats()["sorts"] == 5
    g.close()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_brick_fused_steps_match_the_oracle(oracle, dtype):
    """mpcd_step(3) from a common state (two launches of the brick kernel after the sort of step 0), every mismatch explained."""
    n = (16, 12, 10)
    g, o = _pair(oracle, n, 10, 5, dtype, sort_period=25)
    g.step(3); o.step(3)
    r = _check(g, o, [float(x) for x in n], dtype, tol_scale=3.0)
    assert r["bad_cell"] <= (2 if dtype == np.float32 else 0), r
    g.close()


def test_brick_and_per_particle_kernels_give_bit_identical_trajectories():
    """With deterministic accumulation (64-bit fixed-point sums) the trajectory does not depend on which kernel processed a
    particle, in which order, or how the sums were combined: brick = 1 and brick = 0 agree bit for bit over 30 steps
    (two sorts), with and without the cell thermostat."""
    from paper_1801_10187_b200 import MPCD
    n, M = (13, 9, 10), 10
    pos, vel, tag = synth.solvent(n, M, seed=11, dtype=np.float32)
    for thermostat in (False, True):
        out = []
        for brick in (False, True):
            g = MPCD([float(x) for x in n], pos.shape[0], seed=11, init_state=False, deterministic=True, brick=brick, thermostat=thermostat)
            g.set_state(pos, vel, tag)
            g.step(7); g.step(23)
            s = g.get_state()
            i = np.argsort(s["tag"], kind="stable")
            out.append((s["pos"][i], s["vel"][i][:, :3], s["cell"][i]))
            g.close()
        for x, y in zip(*out):
            assert np.array_equal(x, y)


def test_a_brick_with_more_particles_than_one_chunk(oracle):
    """3000 particles in a box of one brick (4 x 4 x 4 cells): more additions per window cell than the fixed-point headroom
    of the shared-memory partial sums allows between two flushes."""
    n = (4, 4, 4)
    g, o = _pair(oracle, n, None, 3, np.float32, N=3000, sort_period=25)
    g.step(3); o.step(3)
    r = _check(g, o, [4.0] * 3, np.float32, tol_scale=3.0)
    assert r["bad_cell"] <= 2
    c = g.stats()
    assert c["max_occupancy"] >= 47
    g.close()


def test_particles_that_leave_the_window_take_the_global_route(oracle):
    """A hot fluid (kT = 25: 0.5 a per step) with a long sort period drifts far outside the halo of its brick's window: the
    result must not depend on it.  Teacher-forced (oracle side only) after 12 unsorted steps, two more steps through the
    brick kernel; tolerance 1e-5 sqrt(kT/m)."""
    n = (12, 12, 12)
    g, o = _pair(oracle, n, 8, 19, np.float32, kT=25.0, sort_period=40)
    g.step(12)
    for t in (12, 14):
        st = g.get_state()
        o.set_state(st["pos"], st["vel"], st["tag"], step=t)
        g.step(2); o.step(2)
        r = _check(g, o, [12.0] * 3, np.float32, tol_scale=5.0)
        assert r["bad_cell"] <= 2, r
    s = g.get_state()
    assert np.max(np.abs(s["vel"][:, :3].astype(np.float64).sum(axis=0))) / s["tag"].size <= 1e-5
    g.shift_and_bin()
    assert np.array_equal(g.get_cells()["count"], np.bincount(g.get_state()["cell"], minlength=12 ** 3))
    g.close()


def test_brick_kernel_with_embedded_beads(oracle):
    from paper_1801_10187_b200 import MPCD
    n = (10, 9, 8)
    pos, vel, tag = synth.solvent(n, 5, seed=41, dtype=np.float32)
    bp, bv, bm = synth.chains(n, 10, 20, seed=42, mass=5.0, r0=0.5)
    box = [float(x) for x in n]
    g = MPCD(box, pos.shape[0], seed=41, init_state=False, brick=True, sort_period=25)
    g.set_state(pos, vel, tag); g.set_embedded(bp, bv, bm, 20, 1000.0, 0.5, 10)
    o = oracle.OracleMPCD(box, pos.shape[0], seed=41, dtype=np.float32, init=False, sort_period=25)
    o.set_state(pos, vel, tag); o.set_embedded(bp, bv, bm, 20, 1000.0, 0.5, 10)
    g.step(3); o.step(3)
    e = g.get_embedded()
    assert np.max(np.abs(e["vel"] - o.emb["vel"])) <= 3e-5 and np.max(np.abs(e["pos"] - o.emb["pos"])) <= 3e-5
    assert np.array_equal(e["cell"], o.emb["cell"])
    _check(g, o, box, np.float32, tol_scale=3.0)
    g.close()


def test_brick_thermostat_steps_match_the_oracle(oracle):
    n = (10, 10, 8)
    g, o = _pair(oracle, n, 10, 8, np.float32, sort_period=25, thermostat=True)
    g.step(3); o.step(3)
    _check(g, o, [float(x) for x in n], np.float32, tol_scale=3.0)
    g.close()


def test_brick_kernel_keeps_the_invariants_over_many_sort_periods():
    """BASELINE config 2 (64^3 cells, 2.6 M particles, sort every 25) for 300 steps through the brick kernel: total-momentum
    drift <= 1e-6 (reading A25), kinetic energy conserved to fp32 store rounding (SRD conserves energy), no
    particle lost or duplicated by 12 brick-major sorts, positions inside the box."""
    from paper_1801_10187_b200 import MPCD
    cfg = synth.CONFIGS["C2"]
    pos, vel, tag = synth.solvent(cfg["n"], cfg["M"], seed=cfg["seed"], dtype=np.float32)
    N = pos.shape[0]
    g = MPCD([float(x) for x in cfg["n"]], N, seed=cfg["seed"], sort_period=25, init_state=False, brick=True)
    g.set_state(pos, vel, tag)
    P0, KE0, kT0 = g.get_thermo()
    drift, KEs = 0.0, []
    for _ in range(6):
        g.step(50)
        P, KE, kT = g.get_thermo()
        drift = max(drift, float(np.max(np.abs(np.asarray(P) - np.asarray(P0)))) / N)
        KEs.append(KE)
    assert g.stats()["step"] == 300 and g.stats()["sorts"] == 12
    assert drift <= 1e-6, drift
    assert max(abs(k - KE0) for k in KEs) / KE0 <= 2e-5, KEs
    s = g.get_state()
    assert np.array_equal(np.sort(s["tag"]), tag)
    assert np.all((s["pos"][:, :3] >= 0) & (s["pos"][:, :3] < 64.0))
    g.close()


@pytest.mark.parametrize("kT_state", [1.0, 150.0])
def test_fp64_brick_sums_stay_within_their_stated_quantisation(kT_state):
    """include/mpcd.h, opt.brick: in the fp64 model the brick kernel's block-local sums round a velocity component to
    2^-49 unit (unit = the power of two >= sqrt(kT/m) of the handle) -- coarser than the per-particle kernel's fp64 atomics,
    so "same up to summation order" does not quite hold.  The stated bound: a cell mean moves by <= 2^-50 unit, a velocity
    after the collision by < 1e-13 unit.  Checked brick = 1 against brick = 0 on the same fluid over one sort and two
    brick launches.  Second case: a state at 150x the handle's kT, where most particles have a component above 8 unit,
    do not fit the fixed-point headroom and take the direct fp64 route: same agreement (scaled by |v| ~ 12 unit)."""
    from paper_1801_10187_b200 import MPCD
    n, M = (16, 12, 10), 10
    pos, vel, tag = synth.solvent(n, M, seed=23, dtype=np.float64, kT=kT_state)
    if kT_state > 64.0:
        assert np.mean(np.max(np.abs(vel[:, :3]), axis=1) >= 8.0) > 0.5
    out = []
    for brick in (True, False):
        g = MPCD([float(x) for x in n], pos.shape[0], kT=1.0, seed=23, precision="fp64", init_state=False, brick=brick, sort_period=25,
                 dt=0.1 if kT_state == 1.0 else 0.02)
        g.set_state(pos, vel, tag)
        g.step(3)                     # step 0 sorts; the collisions of steps 0 and 1 run in the step kernel under test
        assert (g.stats()["brick"][0] > 0) == brick
        s = g.get_state()
        o = np.argsort(s["tag"], kind="stable")
        out.append((s["pos"][o][:, :3], s["vel"][o][:, :3], s["cell"][o]))
        g.close()
    scale = math.sqrt(kT_state)
    assert np.array_equal(out[0][2], out[1][2])
    assert np.max(np.abs(out[0][1] - out[1][1])) < 1e-13 * scale * 3       # three collisions
    assert np.max(np.abs(out[0][0] - out[1][0])) < 1e-13 * scale

"""GPU parity for the small-system path (csrc/mpcd_small.cuh): a system that fits on the chip as one resident wave runs
the steps between two sorts in ONE cooperative launch (BASELINE config 1 is bound by launches, not bandwidth).  The
kernel is reached by mpcd_step(k) with k >= 3; mpcd_step(1) never uses it."""
import numpy as np
import pytest

import workloads as synth
from parity_explain import explained_compare

pytestmark = pytest.mark.gpu


def _gpu(n, M, seed, dtype, **kw):
    from paper_1801_10187_b200 import MPCD
    pos, vel, tag = synth.solvent(n, M, seed=seed, dtype=dtype)
    g = MPCD([float(x) for x in n], pos.shape[0], seed=seed, precision="fp64" if dtype == np.float64 else "mixed", init_state=False, **kw)
    g.set_state(pos, vel, tag)
    return g, (pos, vel, tag)


def test_config1_hundred_steps_in_one_call_equal_a_hundred_calls():
    """BASELINE config 1 (8^3 cells, 2560 particles, sort every 25, 100 steps) with deterministic sums: mpcd_step(100) -- four
    cooperative launches of 24 steps between the sort steps -- lands bit for bit on mpcd_step(1) x 100 (ordinary kernels only)."""
    cfg = synth.CONFIGS["C1"]
    ga, _ = _gpu(cfg["n"], cfg["M"], cfg["seed"], np.float32, deterministic=True)
    gb, _ = _gpu(cfg["n"], cfg["M"], cfg["seed"], np.float32, deterministic=True)
    la = ga.stats()["kernel_launches"]
    ga.step(100)
    assert ga.stats()["kernel_launches"] - la < 60          # not two launches per step
    for _ in range(100):
        gb.step(1)
    a, b = ga.get_state(), gb.get_state()
    ia, ib = np.argsort(a["tag"]), np.argsort(b["tag"])
    for k in ("pos", "vel", "cell"):
        assert np.array_equal(a[k][ia], b[k][ib]), k
    assert a["step"] == b["step"] == 100 and ga.stats()["sorts"] == gb.stats()["sorts"] == 4
    assert np.array_equal(ga.get_shift(), gb.get_shift())
    ga.close(); gb.close()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("cell_energy", [True, False])
def test_small_system_steps_teacher_forced_against_the_oracle(oracle, dtype, cell_energy):
    """Every four steps (three phases of the cooperative kernel) the oracle restarts from the GPU's state and must land on
    the GPU's next state, every mismatch explained; the cell arrays left behind are those of the last bin."""
    n, M = (9, 7, 8), 6
    g, (pos, vel, tag) = _gpu(n, M, 13, dtype, sort_period=7, cell_energy=cell_energy)
    box = [float(x) for x in n]
    o = oracle.OracleMPCD(box, pos.shape[0], seed=13, dtype=dtype, init=False, sort_period=7)
    tol = 1e-12 if dtype == np.float64 else 1e-5
    for t in range(0, 24, 4):
        st = g.get_state()
        o.set_state(st["pos"], st["vel"], st["tag"], step=t)
        g.step(4); o.step(4)
        s = g.get_state()
        a, b = np.argsort(s["tag"]), np.argsort(o.tag)
        r = explained_compare(s["pos"][a], s["vel"][a], s["cell"][a], o.pos[b], o.vel[b], o.cell[b], g.get_shift(), 1.0, box, 10 * tol, dtype,
                              pos_ulps=4 if dtype == np.float32 else 300)
        assert r["bad_cell"] <= 1, (t, r)
        np.testing.assert_allclose(g.get_shift(), o.shift.astype(dtype).astype(np.float64), rtol=0, atol=0)
    # the sums the last phase left behind serve the next bin-dependent call
    g.shift_and_bin()
    c = g.get_cells()
    assert np.array_equal(c["count"], np.bincount(g.get_state()["cell"], minlength=n[0] * n[1] * n[2]))
    P, KE, kT = g.get_thermo()
    assert abs(kT - 1.0) < 0.1 and np.max(np.abs(P)) / pos.shape[0] < 1e-6
    g.close()


def test_small_path_is_left_alone_by_other_rules_and_options(oracle):
    """AT rule, thermostat and the brick order keep their ordinary kernels; results still match the oracle."""
    from paper_1801_10187_b200 import MPCD
    n, M = (8, 8, 8), 5
    pos, vel, tag = synth.solvent(n, M, seed=3, dtype=np.float32)
    for kw in (dict(rule="at"), dict(thermostat=True), dict(brick=True)):
        g = MPCD([8.0] * 3, pos.shape[0], seed=3, init_state=False, **kw)
        g.set_state(pos, vel, tag)
        okw = dict(rule=1) if kw.get("rule") == "at" else {k: v for k, v in kw.items() if k == "thermostat"}
        o = oracle.OracleMPCD([8.0] * 3, pos.shape[0], seed=3, dtype=np.float32, init=False, **okw)
        o.set_state(pos, vel, tag)
        g.step(4); o.step(4)
        s = g.get_state()
        a, b = np.argsort(s["tag"]), np.argsort(o.tag)
        explained_compare(s["pos"][a], s["vel"][a], s["cell"][a], o.pos[b], o.vel[b], o.cell[b], g.get_shift(), 1.0, [8.0] * 3, 1e-4, np.float32, pos_ulps=4)
        g.close()


def test_config1_thousand_steps_keep_momentum_and_energy():
    """BASELINE config 1 for 1000 steps, 40 cooperative launches: momentum drift <= 1e-6 (A25), energy to fp32 store rounding."""
    cfg = synth.CONFIGS["C1"]
    g, (pos, vel, tag) = _gpu(cfg["n"], cfg["M"], cfg["seed"], np.float32)
    N = pos.shape[0]
    P0, KE0, _ = g.get_thermo()
    g.step(1000)
    P, KE, kT = g.get_thermo()
    assert g.stats()["step"] == 1000 and g.stats()["sorts"] == 40 and g.stats()["kernel_launches"] < 400
    assert float(np.max(np.abs(np.asarray(P) - np.asarray(P0)))) / N <= 1e-6
    assert abs(KE - KE0) / KE0 <= 1e-4
    s = g.get_state()
    assert np.array_equal(np.sort(s["tag"]), tag) and np.all((s["pos"][:, :3] >= 0) & (s["pos"][:, :3] < 8.0))
    g.close()

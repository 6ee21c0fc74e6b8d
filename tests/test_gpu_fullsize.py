"""GPU parity and invariants at BASELINE.json's full sizes, in the launch configuration bench.py
times (mpcd_step: the fused one-pass-per-step pipeline, sort every 25).

C3 / C4 (80 M / 42 M particles): the C oracle still finishes one step in seconds, so the first
steps are compared ELEMENT BY ELEMENT (positions and cell indices bit-exact, velocities within the
north_star tolerance), plus the size-independent properties: counts sum to N, momentum conserved.
C2 (2.6 M particles, 1000 steps): the multi-step invariants of north_star -- total-momentum drift
<= 1e-6 relative (reading A25) and temperature within statistical error (SRD conserves energy,
PAPER.md:45)."""
import numpy as np
import pytest

import workloads as synth

pytestmark = pytest.mark.gpu


def _pair(oracle, cfgname, dtype, sort_period=25):
    from paper_1801_10187_b200 import MPCD
    cfg = synth.CONFIGS[cfgname]
    pos, vel, tag = synth.solvent(cfg["n"], cfg["M"], seed=cfg["seed"], dtype=dtype)
    box = [float(x) for x in cfg["n"]]
    g = MPCD(box, pos.shape[0], seed=cfg["seed"], precision="fp64" if dtype == np.float64 else "mixed", rule=cfg["rule"],
             sort_period=sort_period, init_state=False)
    g.set_state(pos, vel, tag)
    o = oracle.OracleMPCD(box, pos.shape[0], seed=cfg["seed"], dtype=dtype, init=False, rule=1 if cfg["rule"] == "at" else 0,
                          sort_period=sort_period)
    o.set_state(pos, vel, tag)
    return g, o, pos.shape[0]


def _compare(g, o, tol):
    """One step from an identical state: positions and cells bit-exact, velocities within tol."""
    s = g.get_state()
    a, b = np.argsort(s["tag"], kind="stable"), np.argsort(o.tag, kind="stable")
    assert np.array_equal(s["tag"][a], o.tag[b])
    assert np.array_equal(s["pos"][a][:, :3], o.pos[b][:, :3]), "positions are not bit-exact"
    assert np.array_equal(s["cell"][a], o.cell[b]), "cell indices are not bit-exact"
    err = 0.0
    for lo in range(0, a.size, 1 << 24):     # chunked: keeps the fp64 temporaries small
        sl = slice(lo, lo + (1 << 24))
        err = max(err, float(np.max(np.abs(s["vel"][a[sl]][:, :3].astype(np.float64) - o.vel[b[sl]][:, :3].astype(np.float64)))))
    assert err <= tol, err
    return err


def _compare_multistep(g, o, box, tol):
    """Several steps from an identical state.  A velocity that differs by one fp32 ulp after the first step
    (fp64 summation order, allowed by the tolerance) moves the next position by ulp * dt, and at 10^8
    particles a handful of those land on the other side of a cell boundary, which changes the mean of two
    cells.  So: positions within 2 ulp of the box length (minimum image), and all but a 1e-5 fraction of
    cell indices / velocities in agreement."""
    s = g.get_state()
    a, b = np.argsort(s["tag"], kind="stable"), np.argsort(o.tag, kind="stable")
    assert np.array_equal(s["tag"][a], o.tag[b])
    N = a.size
    L = np.asarray(box, dtype=np.float64)
    bad_cell = bad_vel = 0
    worst_pos = 0.0
    for lo in range(0, N, 1 << 24):
        sl = slice(lo, lo + (1 << 24))
        d = np.abs(s["pos"][a[sl]][:, :3].astype(np.float64) - o.pos[b[sl]][:, :3].astype(np.float64))
        d = np.minimum(d, L - d)
        worst_pos = max(worst_pos, float(d.max()))
        bad_cell += int(np.count_nonzero(s["cell"][a[sl]] != o.cell[b[sl]]))
        dv = np.abs(s["vel"][a[sl]][:, :3].astype(np.float64) - o.vel[b[sl]][:, :3].astype(np.float64)).max(axis=1)
        bad_vel += int(np.count_nonzero(dv > tol))
    assert worst_pos <= 2 * np.spacing(np.float32(L.max())), worst_pos
    assert bad_cell <= 1e-5 * N, bad_cell
    assert bad_vel <= 1e-4 * N, bad_vel
    return bad_cell, bad_vel


def test_config3_full_size_first_steps_match_the_oracle(oracle):
    """C3: 200^3 cells, 80 M particles, mixed precision, SRD.  Step 0 sorts (t % 25 == 0)."""
    g, o, N = _pair(oracle, "C3", np.float32)
    g.step(1); o.step(1)
    _compare(g, o, 1e-5)
    # the bin of the next step through the unfused ABI calls: counts bit-exact, sums to rounding.
    # Teacher-forced: the oracle continues from the GPU's state (a velocity that differs by one fp32 ulp
    # would otherwise show up in the sums at 1e-8).
    st = g.get_state(cell=False)
    o.set_state(st["pos"], st["vel"], st["tag"], step=1)
    del st
    g.stream(); g.shift_and_bin()
    o.stream(); o.shift_and_bin()
    c = g.get_cells()
    assert int(c["count"].sum()) == N
    assert np.array_equal(c["count"], o.count)
    assert np.max(np.abs(c["sumv"] - o.sumv)) <= 1e-11
    assert np.max(np.abs(c["ke"] - o.ke)) <= 1e-10 * max(1.0, float(np.max(o.ke)))
    assert np.max(np.abs(c["u"] - o.u)) <= 1e-12
    assert np.max(np.abs(c["axis"] - o.axis)) <= 4e-15
    assert g.stats()["max_occupancy"] == int(o.count.max())
    # a second, fused step (collide(t) + stream + bin(t+1) in one kernel) from the same state
    st = g.get_state()
    P0 = st["vel"][:, :3].astype(np.float64).sum(axis=0)
    g.step(2); o.step(2)
    _compare_multistep(g, o, [200.0] * 3, 1e-5)
    P1 = g.get_state(pos=False, tag=False, cell=False)["vel"][:, :3].astype(np.float64).sum(axis=0)
    assert np.max(np.abs(P1 - P0)) / N <= 1e-8
    g.close()


def test_config4_full_size_andersen_thermostat_step(oracle):
    """C4: 256 x 256 x 128 cells, density 5, 42 M particles, AT collision keyed by (seed, step, tag)."""
    g, o, N = _pair(oracle, "C4", np.float32)
    g.step(1); o.step(1)
    _compare(g, o, 1e-5)
    g.step(2); o.step(2)                 # the fused AT kernel (apply(t) + stream + bin + draw(t+1))
    _compare_multistep(g, o, [256.0, 256.0, 128.0], 1e-5)
    P, KE, kT = g.get_thermo()
    assert abs(kT - 1.0) < 5e-3          # one AT collision thermalises to kT (statistical error ~ 3e-4 here)
    assert np.max(np.abs(P)) / N <= 1e-7
    g.close()


def test_config3_fp64_mode_sampled_cells(oracle):
    """C3 in the all-fp64 model: one fused step, checked on sampled cells the oracle computes one by
    one (its per-cell definition written out in numpy fp64) and on the global invariants."""
    from paper_1801_10187_b200 import MPCD
    cfg = synth.CONFIGS["C3"]
    pos, vel, tag = synth.solvent(cfg["n"], cfg["M"], seed=cfg["seed"], dtype=np.float64)
    N = pos.shape[0]
    box = [float(x) for x in cfg["n"]]
    g = MPCD(box, N, seed=cfg["seed"], precision="fp64", sort_period=0, init_state=False)
    g.set_state(pos, vel, tag)
    g.stream(); g.shift_and_bin()
    s = g.get_state()
    shift = g.get_shift()
    cell_o = oracle.bin_cells(s["pos"], shift, 1.0, cfg["n"])
    assert np.array_equal(s["cell"], cell_o)
    c = g.get_cells()
    assert int(c["count"].sum()) == N
    rng = np.random.default_rng(1)
    sample = rng.choice(c["count"].size, size=64, replace=False)
    members = {int(k): np.flatnonzero(cell_o == k) for k in sample}
    axis = oracle.draw_axis(cfg["seed"], 0, c["count"].size)
    g.collide_srd(np.deg2rad(130.0))
    v1 = g.get_state(pos=False, tag=False, cell=False)["vel"]
    ca, sa = np.cos(np.deg2rad(130.0)), np.sin(np.deg2rad(130.0))
    for k, idx in members.items():
        assert c["count"][k] == idx.size
        if idx.size == 0:
            continue
        v = s["vel"][idx, :3]
        u = v.sum(axis=0) / idx.size
        np.testing.assert_allclose(c["u"][k], u, rtol=0, atol=1e-13)
        n = axis[k]
        w = v - u
        wr = w * ca + np.cross(n, w) * sa + np.outer(w @ n, n) * (1.0 - ca)
        np.testing.assert_allclose(v1[idx, :3], u + wr, rtol=0, atol=1e-12)
    P0 = s["vel"][:, :3].sum(axis=0); P1 = v1[:, :3].sum(axis=0)
    assert np.max(np.abs(P1 - P0)) / N <= 1e-15
    K0 = (s["vel"][:, :3] ** 2).sum(); K1 = (v1[:, :3] ** 2).sum()
    assert abs(K1 - K0) / K0 <= 1e-13          # SRD conserves energy
    g.close()


def test_config2_thousand_steps_momentum_drift_and_temperature():
    """C2: 64^3 cells, 2.6 M particles, mixed precision, sort every 25, 1000 steps (north_star invariants)."""
    from paper_1801_10187_b200 import MPCD
    cfg = synth.CONFIGS["C2"]
    pos, vel, tag = synth.solvent(cfg["n"], cfg["M"], seed=cfg["seed"], dtype=np.float32)
    N = pos.shape[0]
    g = MPCD([float(x) for x in cfg["n"]], N, seed=cfg["seed"], sort_period=25, init_state=False)
    g.set_state(pos, vel, tag)
    P0, KE0, kT0 = g.get_thermo()
    drift, kTs, KEs = 0.0, [kT0], [KE0]
    for _ in range(20):
        g.step(50)
        P, KE, kT = g.get_thermo()
        drift = max(drift, float(np.max(np.abs(np.asarray(P) - np.asarray(P0)))) / N)   # / (N m sigma), m = sigma = 1 (A25)
        kTs.append(kT); KEs.append(KE)
    assert g.stats()["step"] == 1000 and g.stats()["sorts"] == 40
    assert drift <= 1e-6, drift
    # SRD conserves energy: the total kinetic energy moves only by fp32 store rounding
    assert max(abs(k - KE0) for k in KEs) / KE0 <= 2e-5, KEs
    # temperature within statistical error: the pooled estimator (A11) measures KE relative to the cell means of
    # one particular binning, whose share (~1/M of KE) fluctuates by sqrt(2 / (3 N_c)) from bin to bin: sigma ~ 2e-4
    sigma_bin = np.sqrt(2.0 / (3.0 * 64 ** 3)) / cfg["M"]
    assert max(abs(k - kT0) for k in kTs) <= 6 * sigma_bin, (kTs, sigma_bin)
    assert abs(kT0 - 1.0) <= 5 * np.sqrt(2.0 / (3.0 * N))      # the initial draw itself
    s = g.get_state()
    assert np.array_equal(np.sort(s["tag"]), tag)               # no particle lost or duplicated by 40 sorts
    assert np.all((s["pos"][:, :3] >= 0) & (s["pos"][:, :3] < 64.0))
    g.close()

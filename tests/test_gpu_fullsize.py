"""GPU parity and invariants at BASELINE.json's full sizes, in the launch configuration bench.py
times (mpcd_step: the fused one-pass-per-step pipeline, sort every 25).

C3 / C4 / C5 (80 M / 42 M / 5 M + 50 000 beads): the C oracle still finishes one step in seconds, so the
first steps are compared ELEMENT BY ELEMENT (positions and cell indices bit-exact, velocities within the
north_star tolerance; over two steps every mismatch must be explained, tests/parity_explain.py), in both
precision models, plus the size-independent properties: counts sum to N, momentum conserved.
C2 (2.6 M particles, 1000 steps): the multi-step invariants of north_star -- total-momentum drift
<= 1e-6 relative (reading A25) and temperature within statistical error (SRD conserves energy,
PAPER.md:45)."""
import numpy as np
import pytest

import workloads as synth
from parity_explain import explained_compare

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


def _compare_multistep(g, o, box, tol, dtype=np.float32):
    """Two steps from an identical state: every mismatch must be explained by the only legitimate chain (a velocity
    differing in its last bit -> a position differing by an ulp -> a particle on a cell face binned next door ->
    another mean for the members of the two cells); see tests/parity_explain.py.  Anything else fails."""
    s = g.get_state()
    a, b = np.argsort(s["tag"], kind="stable"), np.argsort(o.tag, kind="stable")
    assert np.array_equal(s["tag"][a], o.tag[b])
    N = a.size
    r = explained_compare(s["pos"][a], s["vel"][a], s["cell"][a], o.pos[b], o.vel[b], o.cell[b], g.get_shift(), 1.0, box, tol, dtype)
    assert r["bad_cell"] <= 1e-5 * N and r["bad_vel"] <= 40 * max(r["touched_cells"], 1), r
    return r


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
    del c
    # two more steps from this common state: the steady-state kernel bench.py times (collide(t) + stream + bin(t+1) in one
    # launch, particle_pass<float, kSRD|kStream|kBin|kEnergy>), every mismatch explained
    P0 = g.get_state(pos=False, tag=False, cell=False)["vel"][:, :3].astype(np.float64).sum(axis=0)
    g.step(2); o.step(2)
    _compare_multistep(g, o, [200.0] * 3, 1e-5)
    P1 = g.get_state(pos=False, tag=False, cell=False)["vel"][:, :3].astype(np.float64).sum(axis=0)
    assert np.max(np.abs(P1 - P0)) / N <= 1e-8
    g.close()


def test_config3_full_size_fused_kernel_teacher_forced(oracle):
    """The fused steady-state kernel at full size, ELEMENT BY ELEMENT.  With deterministic accumulation (64-bit fixed-point
    cell sums) a trajectory does not depend on how the steps are split over calls, so mpcd_step(1) x 2 (unfused kernels
    only) and mpcd_step(2) (the fused kernel in the middle, the sort on its way out: kSortOut) must agree bit for bit; and
    the oracle, started from the state after the first step, must land on the second: positions and cells bit-exact,
    velocities within the north_star tolerance."""
    from paper_1801_10187_b200 import MPCD
    cfg = synth.CONFIGS["C3"]
    pos, vel, tag = synth.solvent(cfg["n"], cfg["M"], seed=cfg["seed"], dtype=np.float32)
    box = [float(x) for x in cfg["n"]]
    N = pos.shape[0]
    ga = MPCD(box, N, seed=cfg["seed"], deterministic=True, init_state=False)
    ga.set_state(pos, vel, tag)
    ga.step(1)
    s1 = ga.get_state(cell=False)
    o = oracle.OracleMPCD(box, N, seed=cfg["seed"], dtype=np.float32, init=False)
    o.set_state(s1["pos"], s1["vel"], s1["tag"], step=1)
    del s1
    ga.step(1)
    gb = MPCD(box, N, seed=cfg["seed"], deterministic=True, init_state=False)
    gb.set_state(pos, vel, tag)
    del pos, vel
    gb.step(2)
    sa, sb = ga.get_state(), gb.get_state()
    ga.close()
    ia, ib = np.argsort(sa["tag"], kind="stable"), np.argsort(sb["tag"], kind="stable")
    for k in ("pos", "vel", "cell"):
        assert np.array_equal(sa[k][ia], sb[k][ib]), f"{k}: mpcd_step(1) x 2 and mpcd_step(2) differ"
    del sa, sb, ia, ib
    o.step(1)
    _compare(gb, o, 1e-5)
    gb.close()


def test_config4_full_size_andersen_thermostat_step(oracle):
    """C4: 256 x 256 x 128 cells, density 5, 42 M particles, AT collision keyed by (seed, step, tag)."""
    g, o, N = _pair(oracle, "C4", np.float32)
    g.step(1); o.step(1)
    _compare(g, o, 1e-5)
    st = g.get_state(cell=False)                      # teacher-force, then two steps through the fused AT kernel
    o.set_state(st["pos"], st["vel"], st["tag"], step=1)
    del st
    g.step(2); o.step(2)                 # apply(t) + stream + bin + draw(t+1) in one launch
    _compare_multistep(g, o, [256.0, 256.0, 128.0], 1e-5)
    P, KE, kT = g.get_thermo()
    assert abs(kT - 1.0) < 5e-3          # one AT collision thermalises to kT (statistical error ~ 3e-4 here)
    assert np.max(np.abs(P)) / N <= 1e-7
    g.close()


def test_config3_fp64_model_full_size_through_mpcd_step(oracle):
    """C3 in the all-fp64 model, element by element against the oracle, through mpcd_step: two steps from t = 0 run
    particle_pass<double, ...|kSortOut> (the sort of step 0 on the fused kernel's way out), two more the plain fused kernel
    particle_pass<double, kSRD|kStream|kBin|kEnergy>.  In double a last-bit difference never reaches a cell face, so the
    comparison is strict: positions 1e-12, cells bit-exact, velocities 1e-12."""
    g, o, N = _pair(oracle, "C3", np.float64)
    P0 = o.vel[:, :3].sum(axis=0)
    K0 = float((o.vel[:, :3] ** 2).sum())
    for _ in range(2):
        g.step(2); o.step(2)
        s = g.get_state()
        a, b = np.argsort(s["tag"], kind="stable"), np.argsort(o.tag, kind="stable")
        assert np.array_equal(s["cell"][a], o.cell[b]), "cell indices are not bit-exact"
        for k, ref in (("pos", o.pos), ("vel", o.vel)):
            err = 0.0
            for lo in range(0, N, 1 << 23):
                sl = slice(lo, lo + (1 << 23))
                err = max(err, float(np.max(np.abs(s[k][a[sl]][:, :3] - ref[b[sl]][:, :3]))))
            assert err <= 1e-12, (k, err)
        P1 = s["vel"][:, :3].sum(axis=0)
        K1 = float((s["vel"][:, :3] ** 2).sum())
        del s, a, b
        assert np.max(np.abs(P1 - P0)) / N <= 1e-15
        assert abs(K1 - K0) / K0 <= 1e-13          # SRD conserves energy
    assert g.stats()["sorts"] == 1 and g.stats()["step"] == 4
    g.close()


def test_config5_full_size_polymer_solution(oracle):
    """BASELINE config 5 at full size: 100^3 cells, 5 M solvent particles + 1000 chains of 50 beads (mass 5, k = 1000,
    r0 = 0.5, 10 velocity-Verlet substeps per collision), mixed precision, two steps through mpcd_step (the fused
    solvent kernel with kEmbedded beside the bead kernel): beads to 1e-11, bead cells bit-exact, solvent within the
    north_star tolerance with every mismatch explained."""
    from paper_1801_10187_b200 import MPCD
    cfg = synth.CONFIGS["C5"]
    ch = cfg["chains"]
    pos, vel, tag = synth.solvent(cfg["n"], cfg["M"], seed=cfg["seed"], dtype=np.float32)
    bp, bv, bm = synth.chains(cfg["n"], ch["n_chains"], ch["chain_len"], seed=cfg["seed"] + 1, mass=ch["mass"], r0=ch["r0"])
    box = [float(x) for x in cfg["n"]]
    N = pos.shape[0]
    assert N == 5_000_000 and bm.size == 50_000
    g = MPCD(box, N, seed=cfg["seed"], init_state=False)
    g.set_state(pos, vel, tag); g.set_embedded(bp, bv, bm, ch["chain_len"], ch["k"], ch["r0"], ch["md_substeps"])
    o = oracle.OracleMPCD(box, N, seed=cfg["seed"], dtype=np.float32, init=False)
    o.set_state(pos, vel, tag); o.set_embedded(bp, bv, bm, ch["chain_len"], ch["k"], ch["r0"], ch["md_substeps"])
    P0 = vel[:, :3].astype(np.float64).sum(axis=0) + (bm[:, None] * bv).sum(axis=0)
    g.step(2); o.step(2)
    e = g.get_embedded()
    assert np.max(np.abs(e["pos"] - o.emb["pos"])) <= 1e-11
    assert np.max(np.abs(e["vel"] - o.emb["vel"])) <= 1e-11
    assert np.array_equal(e["cell"], o.emb["cell"])
    _compare_multistep(g, o, box, 1e-5)
    s = g.get_state(pos=False, tag=False, cell=False)
    P1 = s["vel"][:, :3].astype(np.float64).sum(axis=0) + (bm[:, None] * e["vel"]).sum(axis=0)
    assert np.max(np.abs(P1 - P0)) / (N + ch["mass"] * bm.size) <= 1e-8        # total momentum incl. the beads
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

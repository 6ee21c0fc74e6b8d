"""GPU parity for the embedded solute (BASELINE config 5) through the C ABI:
MD of the beads, mass-weighted cell means, the collision of beads and solvent against the oracle, and the invariants
of a config-5-like run (total momentum, bond lengths, equipartition)."""
import math

import numpy as np
import pytest

import workloads as synth

pytestmark = pytest.mark.gpu
K, R0, NSUB, MB = 1000.0, 0.5, 10, 5.0


def _pair(oracle, n, M, seed, dtype, n_chains, chain_len, **kw):
    from paper_1801_10187_b200 import MPCD
    pos, vel, tag = synth.solvent(n, M, seed=seed, dtype=dtype)
    bp, bv, bm = synth.chains(n, n_chains, chain_len, seed=seed + 1, mass=MB, r0=R0)
    box = [float(x) for x in n]
    g = MPCD(box, pos.shape[0], seed=seed, precision="fp64" if dtype == np.float64 else "mixed", init_state=False, **kw)
    g.set_state(pos, vel, tag); g.set_embedded(bp, bv, bm, chain_len, K, R0, NSUB)
    o = oracle.OracleMPCD(box, pos.shape[0], seed=seed, dtype=dtype, init=False, **kw)
    o.set_state(pos, vel, tag); o.set_embedded(bp, bv, bm, chain_len, K, R0, NSUB)
    return g, o, bm


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_md_bin_and_collision_with_beads_match_the_oracle(oracle, dtype):
    g, o, bm = _pair(oracle, (9, 8, 7), 5, 40, dtype, 14, 12)
    for _ in range(2):
        g.stream(); o.stream()
        e = g.get_embedded()
        np.testing.assert_allclose(e["pos"], o.emb["pos"], rtol=0, atol=1e-12)      # velocity Verlet, 10 substeps
        np.testing.assert_allclose(e["vel"], o.emb["vel"], rtol=0, atol=1e-11)
        g.shift_and_bin(); o.shift_and_bin()
        assert np.array_equal(g.get_embedded()["cell"], o.emb["cell"])              # bead cells bit-exact
        assert np.array_equal(g.get_state()["cell"], o.cell)
        g.collide_srd(math.radians(130.0)); o.collide_srd(math.radians(130.0))
        np.testing.assert_allclose(g.get_embedded()["vel"], o.emb["vel"], rtol=0, atol=1e-11)
        err = np.max(np.abs(g.get_state()["vel"][:, :3].astype(np.float64) - o.vel[:, :3].astype(np.float64)))
        assert err <= (1e-12 if dtype == np.float64 else 1e-5), err
        st = g.get_state()                                                          # teacher-force the next round
        o.set_state(st["pos"], st["vel"], st["tag"], step=st["step"] + 1)
        g.set_state(st["pos"], st["vel"], st["tag"], step=st["step"] + 1)
        e = g.get_embedded(); o.emb["pos"][:] = e["pos"]; o.emb["vel"][:] = e["vel"]


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_fused_steps_with_beads_match_the_oracle(oracle, dtype):
    g, o, bm = _pair(oracle, (10, 9, 8), 5, 41, dtype, 10, 20, sort_period=2)
    g.step(3); o.step(3)
    s = g.get_state(); e = g.get_embedded()
    a, b = np.argsort(s["tag"]), np.argsort(o.tag)
    tol = 1e-11 if dtype == np.float64 else 3e-5
    assert np.max(np.abs(s["vel"][a][:, :3].astype(np.float64) - o.vel[b][:, :3].astype(np.float64))) <= tol
    assert np.max(np.abs(e["vel"] - o.emb["vel"])) <= tol
    assert np.max(np.abs(e["pos"] - o.emb["pos"])) <= tol
    assert np.array_equal(e["cell"], o.emb["cell"])


def test_step_by_step_equals_one_call_with_beads(oracle):
    """mpcd_step(1) x 4 (no fused kernel) and mpcd_step(4) (fused kernels, a sort on the way) give the same beads and solvent."""
    ga, _, _ = _pair(oracle, (8, 8, 8), 5, 44, np.float64, 8, 16, sort_period=2)
    gb, _, _ = _pair(oracle, (8, 8, 8), 5, 44, np.float64, 8, 16, sort_period=2)
    ga.step(4)
    for _ in range(4):
        gb.step(1)
    ea, eb = ga.get_embedded(), gb.get_embedded()
    np.testing.assert_allclose(ea["pos"], eb["pos"], rtol=0, atol=1e-11)
    np.testing.assert_allclose(ea["vel"], eb["vel"], rtol=0, atol=1e-11)
    sa, sb = ga.get_state(), gb.get_state()
    a, b = np.argsort(sa["tag"]), np.argsort(sb["tag"])
    np.testing.assert_allclose(sa["vel"][a], sb["vel"][b], rtol=0, atol=1e-11)
    np.testing.assert_allclose(sa["pos"][a], sb["pos"][b], rtol=0, atol=1e-11)


def test_config5_like_run_conserves_momentum_and_equilibrates():
    """BASELINE config 5 at reduced size: 32^3 cells, density 5, 100 chains of 50 beads (mass 5, k = 1000, r0 = 0.5),
    10 MD substeps per collision, mixed precision; the beads start twice too hot."""
    from paper_1801_10187_b200 import MPCD
    n, M = (32, 32, 32), 5
    pos, vel, tag = synth.solvent(n, M, seed=50, dtype=np.float32)
    bp, bv, bm = synth.chains(n, 100, 50, seed=51, kT=2.0, mass=MB, r0=R0)
    N = pos.shape[0]
    g = MPCD([float(x) for x in n], N, seed=50, init_state=False)
    g.set_state(pos, vel, tag); g.set_embedded(bp, bv, bm, 50, K, R0, NSUB)
    P0 = vel[:, :3].astype(np.float64).sum(axis=0) + (bm[:, None] * bv).sum(axis=0)
    g.step(200)
    kTb = []
    for _ in range(20):
        g.step(10)
        kTb.append((bm[:, None] * g.get_embedded()["vel"] ** 2).sum() / (3 * bm.size))
    s = g.get_state(); e = g.get_embedded()
    P1 = s["vel"][:, :3].astype(np.float64).sum(axis=0) + (bm[:, None] * e["vel"]).sum(axis=0)
    assert np.max(np.abs(P1 - P0)) / (N + MB * bm.size) <= 1e-6                     # total momentum incl. the beads
    assert abs(np.mean(kTb) - 1.0) < 0.05, np.mean(kTb)                            # equipartition with the solvent at kT = 1
    d = e["pos"].reshape(100, 50, 3); bond = d[:, 1:] - d[:, :-1]; bond -= 32.0 * np.round(bond / 32.0)
    r = np.linalg.norm(bond, axis=2)
    assert abs(r.mean() - R0) < 0.02 and abs(r.std() - math.sqrt(1.0 / K)) < 0.01   # thermal bond fluctuations sqrt(kT/k)
    assert g.stats()["sorts"] == 16 and np.array_equal(np.sort(s["tag"]), tag)
    g.close()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_cell_thermostat_with_beads_matches_the_oracle(oracle, dtype):
    """Reading A28: the beads count in the cell's kinetic energy and particle number, xi scales their
    relative velocities too.  Unfused calls: xi to 1e-9 (one-pass E_k against the oracle's two passes), velocities within
    tolerance; then fused steps through mpcd_step, including the sort on the fused kernel's way out."""
    n = (9, 8, 7)
    pos, vel, tag = synth.solvent(n, 5, seed=70, kT=1.5, dtype=dtype)
    bp, bv, bm = synth.chains(n, 14, 12, seed=71, kT=3.0, mass=MB, r0=R0)
    box = [float(x) for x in n]
    from paper_1801_10187_b200 import MPCD
    kw = dict(sort_period=2)
    g = MPCD(box, pos.shape[0], seed=70, precision="fp64" if dtype == np.float64 else "mixed", init_state=False, thermostat=True, **kw)
    g.set_state(pos, vel, tag); g.set_embedded(bp, bv, bm, 12, K, R0, NSUB)
    o = oracle.OracleMPCD(box, pos.shape[0], seed=70, dtype=dtype, init=False, thermostat=True, **kw)
    o.set_state(pos, vel, tag); o.set_embedded(bp, bv, bm, 12, K, R0, NSUB)
    g.stream(); o.stream(); g.shift_and_bin(); o.shift_and_bin()
    xi = g.get_xi()
    assert np.all(xi[o.ntot < 2] == 1.0) and np.any((o.count < 2) & (o.ntot >= 2))     # a lone solvent particle with a bead IS thermostatted
    np.testing.assert_allclose(xi, o.xi, rtol=1e-9)
    g.collide_srd(math.radians(130.0)); o.collide_srd(math.radians(130.0))
    tol = 1e-11 if dtype == np.float64 else 1e-5
    np.testing.assert_allclose(g.get_embedded()["vel"], o.emb["vel"], rtol=0, atol=max(tol, 1e-11) if dtype == np.float64 else tol)
    assert np.max(np.abs(g.get_state()["vel"][:, :3].astype(np.float64) - o.vel[:, :3].astype(np.float64))) <= tol
    # fused steps from a common state
    st = g.get_state(); e = g.get_embedded()
    for x in (g, o):
        x.set_state(st["pos"], st["vel"], st["tag"], step=1)
    g.set_embedded(e["pos"], e["vel"], bm, 12, K, R0, NSUB); o.emb["pos"][:] = e["pos"]; o.emb["vel"][:] = e["vel"]
    g.step(3); o.step(3)
    s = g.get_state(); e = g.get_embedded()
    a, b = np.argsort(s["tag"]), np.argsort(o.tag)
    tol3 = 1e-10 if dtype == np.float64 else 1e-4
    assert np.max(np.abs(s["vel"][a][:, :3].astype(np.float64) - o.vel[b][:, :3].astype(np.float64))) <= tol3
    assert np.max(np.abs(e["vel"] - o.emb["vel"])) <= tol3 and np.max(np.abs(e["pos"] - o.emb["pos"])) <= tol3
    assert np.array_equal(e["cell"], o.emb["cell"]) and np.array_equal(s["cell"][a], o.cell[b])
    g.close()


def test_thermostat_cools_hot_beads_and_solvent_to_kT():
    """Equipartition under the thermostat: solvent at 1.8 kT and beads at 4 kT both end at the thermostat's kT."""
    from paper_1801_10187_b200 import MPCD
    n, M = (24, 24, 24), 5
    pos, vel, tag = synth.solvent(n, M, seed=80, kT=1.8, dtype=np.float32)
    bp, bv, bm = synth.chains(n, 200, 20, seed=81, kT=4.0, mass=MB, r0=R0)
    g = MPCD([float(x) for x in n], pos.shape[0], kT=1.0, seed=80, init_state=False, thermostat=True)
    g.set_state(pos, vel, tag); g.set_embedded(bp, bv, bm, 20, K, R0, NSUB)
    P0 = vel[:, :3].astype(np.float64).sum(axis=0) + (bm[:, None] * bv).sum(axis=0)
    g.step(100)
    kb, ks = [], []
    for _ in range(20):
        g.step(5)
        kb.append((bm[:, None] * g.get_embedded()["vel"] ** 2).sum() / (3 * bm.size))
        ks.append((g.get_state(pos=False, tag=False, cell=False)["vel"][:, :3].astype(np.float64) ** 2).sum() / (3 * pos.shape[0]))
    assert abs(np.mean(ks) - 1.0) < 0.01 and abs(np.mean(kb) - 1.0) < 0.04, (np.mean(ks), np.mean(kb))
    P1 = g.get_state(pos=False, tag=False, cell=False)["vel"][:, :3].astype(np.float64).sum(axis=0) + (bm[:, None] * g.get_embedded()["vel"]).sum(axis=0)
    assert np.max(np.abs(P1 - P0)) / (pos.shape[0] + MB * bm.size) <= 1e-6
    g.close()


def test_embedded_argument_checks():
    from paper_1801_10187_b200 import MPCD, MPCDError
    bp, bv, bm = synth.chains((4, 4, 4), 2, 5, seed=1)
    for kw in (dict(rule="at"), dict(deterministic=True)):
        g = MPCD([4.0] * 3, 320, seed=1, **kw)
        with pytest.raises(MPCDError) as err:
            g.set_embedded(bp, bv, bm, 5, K, R0, NSUB)
        assert err.value.code == -1
        g.close()
    g = MPCD([4.0] * 3, 320, seed=1)
    for bad in (dict(chain_len=3), dict(md_substeps=0), dict(chain_len=1024)):
        args = dict(chain_len=5, k=K, r0=R0, md_substeps=NSUB); args.update(bad)
        with pytest.raises(MPCDError):
            g.set_embedded(bp, bv, bm, **args)
    with pytest.raises(MPCDError):
        g.get_embedded()
    g.close()

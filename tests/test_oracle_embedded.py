"""Pins for the oracle's embedded solute (BASELINE config 5).

From outside the oracle: the velocity-Verlet map of a harmonic dimer has a closed form (x_n = x_0 cos(n theta),
cos(theta) = 1 - omega^2 dt^2 / 2), forces must be minus the numerical gradient of the bond energy, MD conserves
momentum exactly, the collision with mass-weighted cell means conserves every cell's momentum and relative kinetic
energy, and hot beads in a cold solvent must relax to the solvent's temperature (equipartition)."""
import math

import numpy as np
import pytest

import workloads as synth


def test_velocity_verlet_dimer_closed_form_and_minimum_image(oracle):
    k, r0, m, dt, A = 1000.0, 0.5, 5.0, 0.01, 0.03
    L = [7.0, 5.0, 6.0]
    theta = math.acos(1.0 - (2.0 * k / m) * dt * dt / 2.0)           # omega^2 = k / mu, mu = m / 2
    for x0 in (2.0, 6.9):                                            # the second dimer straddles the periodic boundary
        pos = np.array([[x0, 1.0, 1.0], [(x0 + r0 + A) % L[0], 1.0, 1.0]])
        vel = np.zeros((2, 3)); mass = np.full(2, m)
        for nstep in range(1, 60):
            oracle.md_verlet(pos, vel, mass, 2, k, r0, L, dt, 1)
            d = pos[1, 0] - pos[0, 0]; d -= L[0] * round(d / L[0])
            assert abs(d - (r0 + A * math.cos(nstep * theta))) < 1e-12
            com = (pos[0, 0] + (pos[0, 0] + d)) / 2
            assert abs((com - (x0 + (r0 + A) / 2) + L[0] / 2) % L[0] - L[0] / 2) < 1e-12      # centre of mass at rest
            assert np.all(pos[:, 1:] == 1.0) and abs(vel[:, 0].sum()) < 1e-13


def test_forces_are_minus_the_gradient_and_chains_are_not_linked(oracle):
    rng = np.random.default_rng(3)
    L = [6.0, 6.0, 6.0]; k, r0, clen = 37.0, 0.5, 5
    pos, _, _ = synth.chains((6, 6, 6), 3, clen, seed=4)
    pos += 0.05 * rng.standard_normal(pos.shape); pos %= 6.0

    def energy(x):
        e = 0.0
        for i in range(len(x) - 1):
            if (i + 1) % clen == 0:
                continue
            d = x[i + 1] - x[i]; d -= 6.0 * np.round(d / 6.0)
            e += 0.5 * k * (np.linalg.norm(d) - r0) ** 2
        return e
    f = oracle.md_forces(pos, clen, k, r0, L)
    h = 1e-6
    for i in (0, 4, 5, 7, 14):
        for a in range(3):
            xp, xm = pos.copy(), pos.copy()
            xp[i, a] += h; xm[i, a] -= h
            assert abs(f[i, a] + (energy(xp) - energy(xm)) / (2 * h)) < 1e-6
    assert np.abs(f.sum(axis=0)).max() < 1e-12                       # Newton's third law
    # moving a whole chain rigidly changes no force: no bond between the last bead of a chain and the first of the next
    pos2 = pos.copy(); pos2[clen:2 * clen] = (pos2[clen:2 * clen] + [1.3, -0.7, 2.1]) % 6.0
    np.testing.assert_allclose(oracle.md_forces(pos2, clen, k, r0, L), f, atol=1e-10)


def test_md_conserves_momentum_and_keeps_energy_bounded(oracle):
    n = (8, 8, 8); L = [8.0] * 3; k, r0, clen = 1000.0, 0.5, 10
    pos, vel, mass = synth.chains(n, 6, clen, seed=9)

    def total(x, v):
        e = 0.5 * (mass[:, None] * v * v).sum()
        d = x.reshape(6, clen, 3); b = d[:, 1:] - d[:, :-1]; b -= 8.0 * np.round(b / 8.0)
        return e + 0.5 * k * ((np.linalg.norm(b, axis=2) - r0) ** 2).sum()
    P0, E0 = (mass[:, None] * vel).sum(axis=0), total(pos, vel)
    Es = []
    for _ in range(50):
        oracle.md_verlet(pos, vel, mass, clen, k, r0, L, 0.01, 10)
        Es.append(total(pos, vel))
    assert np.abs((mass[:, None] * vel).sum(axis=0) - P0).max() < 1e-11
    assert max(abs(e - E0) for e in Es) / E0 < 0.02                  # symplectic: bounded O((omega dt)^2) oscillation, no drift
    assert abs(Es[-1] - Es[len(Es) // 2]) / E0 < 0.02
    assert np.all((pos >= 0) & (pos < 8.0))


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_collision_with_beads_conserves_cell_momentum_and_relative_energy(oracle, dtype):
    n = (6, 6, 5); M = 5
    pos, vel, tag = synth.solvent(n, M, seed=12, dtype=dtype)
    bp, bv, bm = synth.chains(n, 12, 10, seed=13)
    o = oracle.OracleMPCD([float(x) for x in n], pos.shape[0], seed=12, dtype=dtype, init=False)
    o.set_state(pos, vel, tag); o.set_embedded(bp, bv, bm, 10, 1000.0, 0.5, 10)
    o.shift_and_bin()
    cs, cb = o.cell.copy(), o.emb["cell"].copy()

    def moments(vs, vb):
        P = np.zeros((o.Nc, 3)); Mc = np.zeros(o.Nc)
        np.add.at(P, cs, vs); np.add.at(Mc, cs, 1.0)
        np.add.at(P, cb, bm[:, None] * vb); np.add.at(Mc, cb, bm)
        u = P / np.maximum(Mc, 1e-300)[:, None]
        E = np.zeros(o.Nc)
        np.add.at(E, cs, 0.5 * ((vs - u[cs]) ** 2).sum(axis=1))
        np.add.at(E, cb, 0.5 * bm * ((vb - u[cb]) ** 2).sum(axis=1))
        return P, Mc, u, E
    P0, Mc, u0, E0 = moments(o.vel[:, :3].astype(np.float64), o.emb["vel"])
    np.testing.assert_allclose(o.u, u0, atol=1e-13)                  # the mass-weighted mean (A10)
    np.testing.assert_allclose(o.Mc, Mc, atol=1e-12)
    vb_before = o.emb["vel"].copy()
    o.collide_srd()
    P1, _, _, E1 = moments(o.vel[:, :3].astype(np.float64), o.emb["vel"])
    tol = 1e-12 if dtype == np.float64 else 2e-6
    np.testing.assert_allclose(P1, P0, atol=20 * tol)
    np.testing.assert_allclose(E1, E0, rtol=20 * tol, atol=20 * tol)
    alone = np.array([np.count_nonzero(cs == c) == 0 and np.count_nonzero(cb == c) == 1 for c in cb])
    if alone.any():                                                  # a bead alone in its cell keeps its velocity
        np.testing.assert_allclose(o.emb["vel"][alone], vb_before[alone], atol=1e-14)


@pytest.mark.slow
def test_hot_beads_relax_to_the_solvent_temperature(oracle):
    n = (10, 10, 10); M = 5; kT = 1.0
    pos, vel, tag = synth.solvent(n, M, seed=21, dtype=np.float64)
    bp, bv, bm = synth.chains(n, 30, 10, seed=22, kT=4.0)            # beads four times too hot
    o = oracle.OracleMPCD([float(x) for x in n], pos.shape[0], seed=21, dtype=np.float64, init=False, sort_period=0)
    o.set_state(pos, vel, tag); o.set_embedded(bp, bv, bm, 10, 1000.0, 0.5, 10)
    o.step(150)
    samples = []
    for _ in range(40):
        o.step(5)
        samples.append((bm[:, None] * o.emb["vel"] ** 2).sum() / (3 * bm.size))
    # energy flows into 5000 solvent particles: the common temperature ends slightly above 1
    kT_solvent = (o.vel[:, :3] ** 2).sum() / (3 * pos.shape[0])
    assert abs(np.mean(samples) - kT_solvent) < 0.06, (np.mean(samples), kT_solvent)
    assert 1.0 < kT_solvent < 1.2


# ---- thermostat with embedded beads (reading A28; PAPER.md:47 eq. 3, :157, :159) ----

def _thermo_pair(oracle, dtype, seed=31, kT_beads=3.0):
    n = (7, 6, 5); M = 6
    pos, vel, tag = synth.solvent(n, M, seed=seed, kT=1.6, dtype=dtype)
    bp, bv, bm = synth.chains(n, 9, 8, seed=seed + 1, kT=kT_beads)
    o = oracle.OracleMPCD([float(x) for x in n], pos.shape[0], kT=1.0, seed=seed, dtype=dtype, init=False, sort_period=0, thermostat=True)
    o.set_state(pos, vel, tag); o.set_embedded(bp, bv, bm, 8, 1000.0, 0.5, 10)
    return o, bm


def test_bead_rotation_with_xi_reduces_to_the_plain_one_and_scales_the_relative_velocity(oracle):
    rng = np.random.default_rng(5)
    nb, Nc = 40, 12
    cell = rng.integers(0, Nc, nb).astype(np.int32)
    u = rng.standard_normal((Nc, 3)); axis = oracle.draw_axis(9, 4, Nc)
    v0 = rng.standard_normal((nb, 3))
    a = v0.copy(); b = v0.copy(); c = v0.copy()
    oracle.collide_srd_beads(a, cell, u, axis, 2.2)
    oracle.collide_srd_beads_xi(b, cell, u, axis, np.ones(Nc), 2.2)
    np.testing.assert_allclose(a, b, rtol=0, atol=1e-14)               # xi = 1: the pinned plain rotation (sense, angle) up to the order of the additions
    oracle.collide_srd_beads_xi(c, cell, u, axis, np.full(Nc, 2.0), 2.2)
    np.testing.assert_allclose(c - u[cell], 2.0 * (a - u[cell]), rtol=0, atol=1e-14)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_cell_energy_with_beads_is_the_sum_over_all_particles_of_the_cell(oracle, dtype):
    o, bm = _thermo_pair(oracle, dtype)
    o.stream(); o.shift_and_bin()
    Nc = o.Nc
    vs = o.vel[:, :3].astype(np.float64); vb = o.emb["vel"]; cs = o.cell; cb = o.emb["cell"]
    P = np.stack([np.bincount(cs, o.m * vs[:, d], Nc) + np.bincount(cb, bm * vb[:, d], Nc) for d in range(3)], axis=1)
    Mc = np.bincount(cs, None, Nc) * o.m + np.bincount(cb, bm, Nc)
    u = np.where(Mc[:, None] > 0, P / np.maximum(Mc, 1e-300)[:, None], 0.0)
    E = np.bincount(cs, 0.5 * o.m * ((vs - u[cs]) ** 2).sum(axis=1), Nc) + np.bincount(cb, 0.5 * bm * ((vb - u[cb]) ** 2).sum(axis=1), Nc)
    np.testing.assert_allclose(o.erel_tot, E, rtol=1e-12, atol=1e-13)
    assert np.array_equal(o.ntot, np.bincount(cs, None, Nc) + np.bincount(cb, None, Nc))
    # no beads: the same routine about u = S / N_c is the pinned two-pass E_rel of oracle_finalize, bit for bit
    erel, ntot = oracle.erel_with_beads(o.vel, o.cell, o.m, o.count, oracle.finalize_cells(o.vel, o.cell, Nc, o.m, o.count, o.sumv)[0],
                                        np.zeros(0, np.int32), np.zeros((0, 3)), np.zeros(0))
    assert np.array_equal(erel, oracle.finalize_cells(o.vel, o.cell, Nc, o.m, o.count, o.sumv)[1]) and np.array_equal(ntot, o.count)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_thermostatted_collision_with_beads_sets_every_cell_to_its_drawn_energy(oracle, dtype):
    """xi^2 E_k = E^ over solvent and beads together, the cell's momentum (incl. the beads) kept; cells with fewer than two
    particles untouched; the drawn energies follow the cell's particle count incl. beads."""
    o, bm = _thermo_pair(oracle, dtype)
    o.stream(); o.shift_and_bin()
    Nc = o.Nc
    cs, cb = o.cell.copy(), o.emb["cell"].copy()
    def moments():
        vs = o.vel[:, :3].astype(np.float64); vb = o.emb["vel"]
        P = np.stack([np.bincount(cs, o.m * vs[:, d], Nc) + np.bincount(cb, bm * vb[:, d], Nc) for d in range(3)], axis=1)
        E = np.bincount(cs, 0.5 * o.m * ((vs - o.u[cs]) ** 2).sum(axis=1), Nc) + np.bincount(cb, 0.5 * bm * ((vb - o.u[cb]) ** 2).sum(axis=1), Nc)
        return P, E
    P0, E0 = moments()
    ehat, xi, ntot = o.ehat.copy(), o.xi.copy(), o.ntot.copy()
    v_before, b_before = o.vel.copy(), o.emb["vel"].copy()
    o.collide_srd()
    P1, E1 = moments()
    tol = 1e-12 if dtype == np.float64 else 3e-6
    np.testing.assert_allclose(P1, P0, atol=30 * tol)
    live = (ntot >= 2) & (E0 > 0)
    np.testing.assert_allclose(E1[live], ehat[live], rtol=30 * tol)
    assert np.all(xi[~live] == 1.0)
    lone = ntot < 2
    assert np.array_equal(o.vel[np.isin(cs, np.flatnonzero(lone))], v_before[np.isin(cs, np.flatnonzero(lone))])
    np.testing.assert_allclose(o.emb["vel"][np.isin(cb, np.flatnonzero(lone))], b_before[np.isin(cb, np.flatnonzero(lone))], atol=1e-14)
    # E^ ~ Gamma(3 (n - 1) / 2, kT): its mean over cells of n particles is 1.5 (n - 1) kT
    sel = ntot >= 2
    assert abs(ehat[sel].sum() / (1.5 * (ntot[sel] - 1)).sum() - 1.0) < 5.0 / math.sqrt(1.5 * (ntot[sel] - 1).sum())


@pytest.mark.slow
def test_thermostat_brings_solvent_and_hot_beads_to_kT(oracle):
    n = (9, 9, 9); M = 5
    pos, vel, tag = synth.solvent(n, M, seed=61, kT=1.8, dtype=np.float64)
    bp, bv, bm = synth.chains(n, 25, 10, seed=62, kT=4.0)
    o = oracle.OracleMPCD([float(x) for x in n], pos.shape[0], kT=1.0, seed=61, dtype=np.float64, init=False, sort_period=0, thermostat=True)
    o.set_state(pos, vel, tag); o.set_embedded(bp, bv, bm, 10, 1000.0, 0.5, 10)
    o.step(60)
    kb, ks = [], []
    for _ in range(40):
        o.step(3)
        kb.append((bm[:, None] * o.emb["vel"] ** 2).sum() / (3 * bm.size))
        ks.append((o.vel[:, :3] ** 2).sum() / (3 * pos.shape[0]))
    assert abs(np.mean(ks) - 1.0) < 0.03, np.mean(ks)                 # canonical: <m v^2> = kT (the cell means carry their share)
    assert abs(np.mean(kb) - 1.0) < 0.08, np.mean(kb)                 # equipartition of the beads at the thermostat's kT

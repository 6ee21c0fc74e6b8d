"""Pins for the oracle's Maxwell-Boltzmann cell thermostat (SURVEY.md 8f NEXT-2; PAPER.md:45-50 eq. 3, :157).

What fixes it from outside the oracle: the drawn energy must follow Gamma(3 (N_c - 1) / 2, kT) (checked
against scipy's distribution, not against the oracle's sampler), the scaled collision must leave every cell
with exactly the drawn relative kinetic energy and its momentum, cells with fewer than two particles must be
left alone, and one thermostatted collision must bring a fluid at the wrong temperature to kT within the
statistical error of the pooled estimator."""
import math

import numpy as np
import pytest
from scipy import stats

import workloads as synth


@pytest.mark.parametrize("n", [2, 3, 10, 31])
def test_drawn_energy_is_gamma_distributed(oracle, n):
    k, kT, M = 1.5 * (n - 1), 0.7, 400_000
    ehat, xi = oracle.thermostat_xi(5, 17, kT, np.full(M, n, np.int32), np.full(M, 2.0))
    dist = stats.gamma(k, scale=kT)
    assert abs(ehat.mean() - k * kT) <= 5 * math.sqrt(k * kT * kT / M)
    assert abs(ehat.var() - k * kT * kT) <= 6 * k * kT * kT * math.sqrt((2 + 6 / k) / M)     # var of the sample variance of a Gamma
    assert stats.kstest(ehat, dist.cdf).pvalue > 1e-3
    np.testing.assert_allclose(xi, np.sqrt(ehat / 2.0), rtol=1e-15)


def test_small_and_cold_cells_are_left_alone_and_stream_is_keyed_by_seed_step_cell(oracle):
    count = np.array([0, 1, 2, 5, 5, 7], np.int32)
    erel = np.array([0.0, 0.0, 1.0, 0.0, 3.0, 2.0])
    ehat, xi = oracle.thermostat_xi(9, 4, 1.0, count, erel)
    assert xi[0] == 1.0 and xi[1] == 1.0 and ehat[0] == 0.0 and ehat[1] == 0.0      # N_c < 2
    assert xi[3] == 1.0 and ehat[3] > 0.0                                            # E_k = 0: nothing to scale (A26)
    assert np.all(xi[[2, 4, 5]] == np.sqrt(ehat[[2, 4, 5]] / erel[[2, 4, 5]]))
    # same (seed, step, cell, N_c) -> same draw whatever else is in the call
    e2, _ = oracle.thermostat_xi(9, 4, 1.0, np.array([9, 9, 9, 9, 5, 9], np.int32), np.ones(6))
    assert e2[4] == ehat[4] and e2[5] != ehat[5]
    e3, _ = oracle.thermostat_xi(9, 5, 1.0, count, erel)
    e4, _ = oracle.thermostat_xi(10, 4, 1.0, count, erel)
    assert e3[4] != ehat[4] and e4[4] != ehat[4]
    # kT is a pure scale
    e5, _ = oracle.thermostat_xi(9, 4, 2.5, count, erel)
    np.testing.assert_allclose(e5, 2.5 * ehat, rtol=1e-15)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_scaled_collision_sets_the_relative_energy_and_keeps_momentum(oracle, dtype):
    n, M = (6, 5, 4), 8
    pos, vel, tag = synth.solvent(n, M, seed=31, dtype=dtype)
    o = oracle.OracleMPCD([float(x) for x in n], pos.shape[0], seed=31, dtype=dtype, init=False, thermostat=True, kT=1.3)
    o.set_state(pos, vel, tag)
    o.shift_and_bin()
    cell, count, ehat, xi = o.cell.copy(), o.count.copy(), o.ehat.copy(), o.xi.copy()
    P0 = np.zeros((o.Nc, 3)); np.add.at(P0, cell, o.vel[:, :3].astype(np.float64))
    o.collide_srd()
    v = o.vel[:, :3].astype(np.float64)
    P1 = np.zeros((o.Nc, 3)); np.add.at(P1, cell, v)
    u = P1 / np.maximum(count, 1)[:, None]
    erel = np.zeros(o.Nc); np.add.at(erel, cell, 0.5 * ((v - u[cell]) ** 2).sum(axis=1))
    tol = 1e-12 if dtype == np.float64 else 2e-6
    np.testing.assert_allclose(P1, P0, rtol=0, atol=tol * 10)
    big = count >= 2
    np.testing.assert_allclose(erel[big], ehat[big], rtol=tol * 10)                 # E_k' = E^ exactly (eq. 3, xi^2 E_k)
    assert np.all(xi[~big] == 1.0)


def test_one_collision_brings_a_hot_fluid_to_kT(oracle):
    n, M, kT = (24, 24, 24), 10, 1.0
    pos, vel, tag = synth.solvent(n, M, seed=77, kT=2.0, dtype=np.float64)        # twice too hot
    o = oracle.OracleMPCD([float(x) for x in n], pos.shape[0], seed=77, dtype=np.float64, init=False, thermostat=True, kT=kT)
    o.set_state(pos, vel, tag)
    o.step(1)
    dof = 1.5 * np.maximum(o.count - 1, 0)[o.count >= 2].sum()
    got = o.thermo()[2]                                                              # pooled kT under the same binning (A11)
    assert abs(got - kT) <= 5 * kT * math.sqrt(1.0 / dof), got                       # Gamma(dof, kT) / dof: sigma = kT / sqrt(dof)
    # canonical fluctuations of the cell energies: var(E_k) = k kT^2 for each shape k
    erel = np.zeros(o.Nc)
    v = o.vel[:, :3]; S = np.zeros((o.Nc, 3)); np.add.at(S, o.cell, v)
    u = S / np.maximum(o.count, 1)[:, None]
    np.add.at(erel, o.cell, 0.5 * ((v - u[o.cell]) ** 2).sum(axis=1))
    sel = o.count == 10
    k = 13.5
    assert sel.sum() > 1000
    assert abs(erel[sel].mean() - k * kT) <= 5 * math.sqrt(k / sel.sum())
    assert abs(erel[sel].var() / (k * kT * kT) - 1.0) <= 6 * math.sqrt((2 + 6 / k) / sel.sum())

"""Physics of the CUDA path at sizes the oracle cannot reach in a test: the transport coefficients of the SRD fluid
against the kinetic-theory closed forms (tests/golden/closed_forms.json; eta = 8.70 is the value the paper prints,
PAPER.md:177) and the Maxwell-Boltzmann velocity distribution.  These do not involve the oracle: they
pin the GPU trajectory to what the method must produce."""
import json
import math
import os

import numpy as np
import pytest
from scipy import stats

import workloads as synth

pytestmark = pytest.mark.gpu

FORMS = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.json")))["cases"]


def _form(M, dt):
    return next(c for c in FORMS if c["M"] == M and c["dt"] == dt and c["alpha_deg"] == 130)


@pytest.mark.parametrize("precision", ["mixed", "fp64"])
def test_srd_viscosity_from_shear_wave_decay(precision):
    """Transverse mode v_x ~ sin(k z) in a 128 x 128 x 32 box (5.2 M particles): amplitude ~ exp(-nu k^2 t)."""
    from paper_1801_10187_b200 import MPCD
    form = _form(10, 0.1)
    n, A = (128, 128, 32), 0.2
    k = 2 * math.pi / n[2]
    dtype = np.float32 if precision == "mixed" else np.float64
    nus = []
    for seed in (11, 22, 33):
        pos, vel, tag = synth.solvent(n, 10, seed=seed, dtype=dtype)
        vel[:, 0] += (A * np.sin(k * pos[:, 2].astype(np.float64))).astype(dtype)
        g = MPCD([float(x) for x in n], pos.shape[0], seed=seed, precision=precision, init_state=False)
        g.set_state(pos, vel, tag)
        t, amp = [], []
        for i in range(16):
            s = g.get_state(tag=False, cell=False)
            t.append(s["step"] * 0.1)
            amp.append(2 * np.mean(s["vel"][:, 0].astype(np.float64) * np.sin(k * s["pos"][:, 2].astype(np.float64))))
            g.step(20)
        g.close()
        nus.append(-np.polyfit(t, np.log(amp), 1)[0] / k ** 2)
    nu = float(np.mean(nus))
    assert abs(nu / form["nu"] - 1) < 0.03, (nus, form["nu"])
    assert 8.65 * 0.97 < 10 * nu < 8.75 * 1.03                       # eta = rho nu: the paper's 8.7


def test_srd_self_diffusion_at_large_mean_free_path():
    """D = 0.5145 at dt = 1 (lambda = a), where molecular chaos holds; from the mean-square displacement."""
    from paper_1801_10187_b200 import MPCD
    form = _form(10, 1.0)
    n = (32, 32, 32)
    pos, vel, tag = synth.solvent(n, 10, seed=9, dtype=np.float64)
    g = MPCD([32.0] * 3, pos.shape[0], seed=9, precision="fp64", dt=1.0, sort_period=0, init_state=False)
    g.set_state(pos, vel, tag)
    g.step(20)
    disp = np.zeros((pos.shape[0], 3)); msd = []
    for _ in range(60):
        disp += g.get_state(pos=False, tag=False, cell=False)["vel"][:, :3] * 1.0     # sort_period = 0: the order never changes
        g.step(1)
        msd.append((disp ** 2).sum(axis=1).mean())
    g.close()
    t = np.arange(1, 61) * 1.0
    D = np.polyfit(t[20:], np.array(msd)[20:], 1)[0] / 6
    assert abs(D / form["D"] - 1) < 0.03, (D, form["D"])


@pytest.mark.parametrize("rule", ["srd", "at"])
def test_velocity_distribution_stays_maxwell_boltzmann(rule):
    from paper_1801_10187_b200 import MPCD
    n, kT = (64, 64, 64), 1.0
    M = 10 if rule == "srd" else 5
    pos, vel, tag = synth.solvent(n, M, seed=4, dtype=np.float32)
    g = MPCD([64.0] * 3, pos.shape[0], seed=4, rule=rule, init_state=False)
    var0 = float(vel[:, :3].astype(np.float64).var())
    g.set_state(pos, vel, tag)
    g.step(300)
    v = g.get_state(pos=False, tag=False, cell=False)["vel"][:, :3].astype(np.float64)
    g.close()
    N = v.shape[0]
    assert np.max(np.abs(v.mean(axis=0))) < 1e-5
    if rule == "srd":
        assert abs(v.var() - var0) < 2e-5 * var0                    # SRD conserves energy: only fp32 store rounding
    else:
        assert abs(v.var() / kT - 1) < 5 * math.sqrt(2.0 / (3 * N)) + 1e-3   # AT thermostats to kT
    for d in range(3):
        x = v[::37, d] / math.sqrt(kT)
        assert abs(stats.kurtosis(x)) < 5 * math.sqrt(24.0 / x.size)
        assert stats.kstest(x, "norm").pvalue > 1e-3
    assert stats.kstest(np.linalg.norm(v[::37], axis=1) / math.sqrt(kT), "maxwell").pvalue > 1e-3

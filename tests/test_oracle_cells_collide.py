"""Pins for the oracle's cell properties, SRD collision (eq. 2, Alg. 1),
Andersen-thermostat collision (eq. 4) and sort.  CPU only."""
import json
import math
import os

import numpy as np
import pytest
from scipy import stats
from scipy.spatial.transform import Rotation

import workloads as synth

HERE = os.path.dirname(os.path.abspath(__file__))
FORMS = json.load(open(os.path.join(HERE, "golden", "closed_forms.json")))["cases"]


def _form(M, dt):
    return next(c for c in FORMS if c["M"] == M and c["dt"] == dt)


def _setup(oracle, n, M, seed, dtype=np.float32, m=1.0, a=1.0, step=0):
    pos, vel, tag = synth.solvent(n, M, seed=seed, dtype=dtype, a=a)
    Nc = n[0] * n[1] * n[2]
    shift = oracle.draw_shift(seed, step, a)
    cell = oracle.bin_cells(pos, shift, a, n)
    count, sumv, ke = oracle.reduce_cells(vel, cell, Nc, m)
    u, erel, kTc = oracle.finalize_cells(vel, cell, Nc, m, count, sumv)
    return dict(pos=pos, vel=vel, tag=tag, Nc=Nc, cell=cell, count=count, sumv=sumv, ke=ke, u=u, erel=erel, kTc=kTc)


# ------------------------------------------------------------------ cell sums
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_cell_sums_against_library_and_exact_sums(oracle, dtype):
    n, m = (6, 5, 4), 2.5
    s = _setup(oracle, n, 7, 13, dtype=dtype, m=m)
    v = s["vel"][:, :3].astype(np.float64)
    cell, Nc = s["cell"], s["Nc"]
    assert np.array_equal(s["count"], np.bincount(cell, minlength=Nc))          # bit-exact counts
    for d in range(3):
        lib = np.bincount(cell, weights=v[:, d], minlength=Nc)                  # library routine
        np.testing.assert_allclose(s["sumv"][:, d], lib, rtol=0, atol=1e-13)
    np.testing.assert_allclose(s["ke"], 0.5 * m * np.bincount(cell, weights=(v**2).sum(axis=1), minlength=Nc), rtol=1e-13)
    # totals against exactly rounded sums (fsum): Sum_c S_c = Sum_i v_i, Sum_c K_c = KE_total
    for d in range(3):
        assert abs(math.fsum(s["sumv"][:, d]) - math.fsum(v[:, d])) <= 1e-13 * np.abs(v[:, d]).sum()
    assert abs(math.fsum(s["ke"]) - 0.5 * m * math.fsum((v**2).sum(axis=1))) <= 1e-13 * math.fsum(s["ke"])
    # per-cell exact check on a few cells
    for c in (0, 17, Nc - 1):
        mem = np.nonzero(cell == c)[0]
        for d in range(3):
            assert abs(s["sumv"][c, d] - math.fsum(v[mem, d])) <= 1e-14 * max(1.0, np.abs(v[mem, d]).sum())


def test_finalize_mean_erel_temperature(oracle):
    n, m = (5, 5, 5), 1.7
    s = _setup(oracle, n, 6, 99, m=m)
    v = s["vel"][:, :3].astype(np.float64)
    for c in range(s["Nc"]):
        mem = np.nonzero(s["cell"] == c)[0]
        k = len(mem)
        if k == 0:
            assert np.all(s["u"][c] == 0) and s["erel"][c] == 0 and s["kTc"][c] == 0   # A16
            continue
        np.testing.assert_allclose(s["u"][c], v[mem].mean(axis=0), rtol=0, atol=1e-14)
        erel = 0.5 * m * ((v[mem] - v[mem].mean(axis=0)) ** 2).sum()                  # eq. (3)
        np.testing.assert_allclose(s["erel"][c], erel, rtol=1e-12, atol=1e-14)
        # single-pass identity KE - M_c u^2 / 2 (A12)
        np.testing.assert_allclose(s["erel"][c], s["ke"][c] - 0.5 * m * k * (s["u"][c] ** 2).sum(), rtol=0, atol=1e-12)
        want_kT = 2 * erel / (3 * (k - 1)) if k >= 2 else 0.0                           # A11
        np.testing.assert_allclose(s["kTc"][c], want_kT, rtol=1e-12, atol=1e-14)
    assert np.count_nonzero(s["count"] < 2) > 0          # the edge case is present in this draw


def test_thermo_totals(oracle):
    n, m = (8, 8, 8), 1.0
    s = _setup(oracle, n, 10, 5, m=m)
    P, KE, kT = oracle.thermo(m, s["count"], s["sumv"], s["ke"], s["erel"])
    v = s["vel"][:, :3].astype(np.float64)
    np.testing.assert_allclose(P, m * v.sum(axis=0), atol=1e-10)
    np.testing.assert_allclose(KE, 0.5 * m * (v**2).sum(), rtol=1e-13)
    dof = 1.5 * (s["count"][s["count"] >= 2] - 1).sum()
    assert abs(kT - 1.0) < 4 * math.sqrt(1.0 / dof)       # chi-square: sd(kT)/kT = sqrt(2/(2 dof)) = sqrt(1/dof)


# ------------------------------------------------------------------ rotation
def _rotation_matrix(oracle, axis, alpha):
    """R's columns = images of the basis vectors under the oracle's collide with u = 0."""
    vel = np.zeros((3, 4), dtype=np.float64)
    vel[:, :3] = np.eye(3)
    oracle.collide_srd(vel, np.zeros(3, dtype=np.int32), np.zeros((1, 3)), np.asarray(axis, dtype=np.float64).reshape(1, 3), alpha)
    return vel[:, :3].T.copy()


def test_rotation_matrix_properties_and_handedness(oracle):
    axes = oracle.draw_axis(3, 0, 50)
    alpha = math.radians(130.0)
    for n in axes:
        R = _rotation_matrix(oracle, n, alpha)
        np.testing.assert_allclose(R @ R.T, np.eye(3), atol=1e-15)
        assert abs(np.linalg.det(R) - 1) < 1e-15
        np.testing.assert_allclose(R @ n, n, atol=1e-15)
        assert abs(np.trace(R) - (1 + 2 * math.cos(alpha))) < 1e-15
        # library rotation: right-handed +alpha about n (A14)
        np.testing.assert_allclose(R, Rotation.from_rotvec(alpha * n).as_matrix(), atol=1e-15)
    n = axes[7]
    np.testing.assert_allclose(_rotation_matrix(oracle, n, 0.0), np.eye(3), atol=0)
    np.testing.assert_allclose(_rotation_matrix(oracle, n, 2 * math.pi), np.eye(3), atol=1e-15)
    np.testing.assert_allclose(_rotation_matrix(oracle, n, math.pi), 2 * np.outer(n, n) - np.eye(3), atol=1e-15)
    np.testing.assert_allclose(_rotation_matrix(oracle, n, alpha) @ _rotation_matrix(oracle, n, -alpha), np.eye(3), atol=1e-15)
    # z axis, +90 degrees: x -> y
    np.testing.assert_allclose(_rotation_matrix(oracle, [0, 0, 1], math.pi / 2) @ [1, 0, 0], [0, 1, 0], atol=1e-16)


# ------------------------------------------------------------------ SRD
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_srd_conserves_cell_momentum_and_relative_energy(oracle, dtype):
    n = (6, 6, 6)
    s = _setup(oracle, n, 5, 31, dtype=dtype)
    axis = oracle.draw_axis(31, 0, s["Nc"])
    v0 = s["vel"].copy()
    oracle.collide_srd(s["vel"], s["cell"], s["u"], axis, math.radians(130.0))
    c2, sumv2, ke2 = oracle.reduce_cells(s["vel"], s["cell"], s["Nc"], 1.0)
    u2, erel2, _ = oracle.finalize_cells(s["vel"], s["cell"], s["Nc"], 1.0, c2, sumv2)
    cnt = s["count"]
    if dtype == np.float64:
        np.testing.assert_allclose(sumv2, s["sumv"], rtol=0, atol=1e-13)
        np.testing.assert_allclose(erel2, s["erel"], rtol=1e-13, atol=1e-13)
    else:   # bounded by the fp32 store rounding: N_c * 2^-24 * max|v|
        bound = (cnt * 2.0**-24 * np.abs(v0).max())[:, None] + 1e-12
        assert np.all(np.abs(sumv2 - s["sumv"]) <= bound)
        np.testing.assert_allclose(erel2, s["erel"], rtol=2e-6, atol=1e-6)
    single = np.nonzero(cnt[s["cell"]] == 1)[0]
    assert len(single) > 0
    assert np.array_equal(s["vel"][single], v0[single])                                  # N_c = 1: v' = v exactly
    changed = np.nonzero(cnt[s["cell"]] >= 2)[0]
    assert np.count_nonzero(np.any(s["vel"][changed, :3] != v0[changed, :3], axis=1)) > 0.99 * len(changed)
    # N_c = 2: relative speed preserved
    for c in np.nonzero(cnt == 2)[0][:20]:
        i, j = np.nonzero(s["cell"] == c)[0]
        d0 = np.linalg.norm(v0[i, :3].astype(np.float64) - v0[j, :3])
        d1 = np.linalg.norm(s["vel"][i, :3].astype(np.float64) - s["vel"][j, :3])
        assert abs(d0 - d1) <= (1e-12 if dtype == np.float64 else 1e-5)


def test_srd_rotates_relative_velocity_by_alpha(oracle):
    """eq. (2): the component of (v - u) perpendicular to the axis turns by exactly alpha,
    the parallel component is unchanged."""
    n = (4, 4, 4)
    s = _setup(oracle, n, 10, 77, dtype=np.float64)
    axis = oracle.draw_axis(77, 0, s["Nc"])
    alpha = math.radians(130.0)
    v0 = s["vel"][:, :3].copy()
    oracle.collide_srd(s["vel"], s["cell"], s["u"], axis, alpha)
    nh = axis[s["cell"]]
    w0 = v0 - s["u"][s["cell"]]
    w1 = s["vel"][:, :3] - s["u"][s["cell"]]
    par0, par1 = (w0 * nh).sum(1), (w1 * nh).sum(1)
    np.testing.assert_allclose(par1, par0, atol=1e-13)
    p0 = w0 - par0[:, None] * nh
    p1 = w1 - par1[:, None] * nh
    cosang = (p0 * p1).sum(1) / (np.linalg.norm(p0, axis=1) * np.linalg.norm(p1, axis=1))
    np.testing.assert_allclose(cosang, math.cos(alpha), atol=1e-10)
    sinang = (np.cross(p0, p1) * nh).sum(1) / (np.linalg.norm(p0, axis=1) * np.linalg.norm(p1, axis=1))
    np.testing.assert_allclose(sinang, math.sin(alpha), atol=1e-10)                      # right-handed


@pytest.mark.parametrize("M", [10, 5])
def test_srd_one_step_decorrelation_closed_form(oracle, M):
    """<v.v'>/<v.v> = 1 - (2/3)(1 - cos a)(M - 1 + e^-M)/M for i.i.d. velocities."""
    n = (32, 32, 32)
    vals = []
    for seed in (1, 2, 3):
        s = _setup(oracle, n, M, seed, dtype=np.float64)
        axis = oracle.draw_axis(seed, 0, s["Nc"])
        v0 = s["vel"][:, :3].copy()
        oracle.collide_srd(s["vel"], s["cell"], s["u"], axis, math.radians(130.0))
        vals.append((v0 * s["vel"][:, :3]).sum() / (v0 * v0).sum())
    N = n[0] * n[1] * n[2] * M
    want = _form(M, 0.1)["srd_decorrelation"]
    assert abs(np.mean(vals) - want) < 4 / math.sqrt(3 * N * len(vals))


# ------------------------------------------------------------------ AT
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_at_conserves_cell_momentum_and_thermalises(oracle, dtype):
    n, kT, m = (12, 12, 12), 1.5, 2.0
    sigma = math.sqrt(kT / m)
    s = _setup(oracle, n, 5, 41, dtype=dtype, m=m)
    s["vel"][:, :3] *= dtype(3.0)                                   # start far from the target temperature
    count, sumv, ke = oracle.reduce_cells(s["vel"], s["cell"], s["Nc"], m)
    u, erel, _ = oracle.finalize_cells(s["vel"], s["cell"], s["Nc"], m, count, sumv)
    v0 = s["vel"].copy()
    dv = oracle.at_draw(41, 0, s["tag"], sigma)
    oracle.collide_at(s["vel"], s["cell"], s["Nc"], count, u, dv)
    c2, sumv2, ke2 = oracle.reduce_cells(s["vel"], s["cell"], s["Nc"], m)
    u2, erel2, _ = oracle.finalize_cells(s["vel"], s["cell"], s["Nc"], m, c2, sumv2)
    tol = 1e-12 if dtype == np.float64 else 40 * 2.0**-24 * 10
    np.testing.assert_allclose(sumv2, sumv, rtol=0, atol=tol)       # eq. (4) last term: momentum restored
    single = np.nonzero(count[s["cell"]] == 1)[0]
    assert len(single) > 0
    np.testing.assert_allclose(s["vel"][single, :3], v0[single, :3], rtol=0, atol=1e-15 if dtype == np.float64 else 0)
    # pooled kT = kT +- kT sqrt(1/dof) after ONE collision from any initial velocities
    _, _, kT_pooled = oracle.thermo(m, c2, sumv2, ke2, erel2)
    dof = 1.5 * (count[count >= 2] - 1).sum()
    assert abs(kT_pooled - kT) < 4 * kT * math.sqrt(1 / dof)
    # direct restatement of eq. (4) with numpy
    D = np.zeros((s["Nc"], 3))
    np.add.at(D, s["cell"], dv)
    want = u[s["cell"]] + dv - D[s["cell"]] / count[s["cell"]][:, None]
    np.testing.assert_allclose(s["vel"][:, :3], want.astype(dtype), rtol=0, atol=1e-12 if dtype == np.float64 else 1e-6)


def test_at_is_keyed_by_tag_not_by_position_in_array(oracle):
    """RNG seeds are (timestep, particle tag, seed): permuting the arrays with the
    tags attached leaves every tagged particle's result unchanged."""
    n = (6, 6, 6)
    s = _setup(oracle, n, 5, 17, dtype=np.float64)
    perm = np.random.default_rng(3).permutation(s["vel"].shape[0])

    def run(vel, cell, tag):
        vel = vel.copy()
        count, sumv, _ = oracle.reduce_cells(vel, cell, s["Nc"], 1.0)
        u, _, _ = oracle.finalize_cells(vel, cell, s["Nc"], 1.0, count, sumv)
        oracle.collide_at(vel, cell, s["Nc"], count, u, oracle.at_draw(17, 4, tag, 1.0))
        return vel

    a = run(s["vel"], s["cell"], s["tag"])
    b = run(np.ascontiguousarray(s["vel"][perm]), np.ascontiguousarray(s["cell"][perm]), np.ascontiguousarray(s["tag"][perm]))
    np.testing.assert_allclose(b, a[perm], rtol=0, atol=1e-13)      # only fp64 summation order differs


def test_at_one_step_decorrelation_closed_form(oracle):
    n, M = (32, 32, 32), 5
    vals = []
    for seed in (1, 2, 3):
        s = _setup(oracle, n, M, seed, dtype=np.float64)
        v0 = s["vel"][:, :3].copy()
        oracle.collide_at(s["vel"], s["cell"], s["Nc"], s["count"], s["u"], oracle.at_draw(seed, 0, s["tag"], 1.0))
        vals.append((v0 * s["vel"][:, :3]).sum() / (v0 * v0).sum())
    N = n[0] * n[1] * n[2] * M
    assert abs(np.mean(vals) - _form(M, 0.1)["at_decorrelation"]) < 4 / math.sqrt(3 * N * len(vals))


# ------------------------------------------------------------------ sort
def test_sort_is_a_stable_permutation_into_cell_order(oracle):
    n = (5, 4, 3)
    s = _setup(oracle, n, 9, 23)
    perm = oracle.sort_perm(s["cell"], s["Nc"])
    assert np.array_equal(np.sort(perm), np.arange(len(perm)))
    assert np.array_equal(perm, np.argsort(s["cell"], kind="stable"))                    # library routine
    pos, vel, tag, cell = oracle.permute(perm, s["pos"], s["vel"], s["tag"], s["cell"])
    assert np.all(np.diff(cell) >= 0)
    # multiset of (tag, pos, vel) unchanged bit for bit
    back = np.argsort(tag)
    assert np.array_equal(tag[back], s["tag"])
    assert np.array_equal(pos[back], s["pos"]) and np.array_equal(vel[back], s["vel"])
    assert np.array_equal(cell[back], s["cell"])

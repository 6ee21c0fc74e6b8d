"""Pins for the three oracle pieces round 1 left unpinned: the initial condition `oracle_init_*`
(reading A23), the rotation inside `oracle_collide_srd_beads` (eq. 2; A14) and inside
`oracle_collide_srd_xi` (Alg. 1 lines 8-10 PAPER.md:150-152).  Each is checked against something other than itself:
the Philox block function and the uniform maps (pinned in test_oracle_rng.py) restated for single indices, library
distributions (scipy KS), a library rotation (scipy Rotation), and the already pinned `oracle_collide_srd`.  CPU only."""
import math

import numpy as np
import pytest
from scipy import stats
from scipy.spatial.transform import Rotation

DOM_INITPOS, DOM_INITVEL = 4, 5          # reading A24


def _block(oracle, seed, step, index, domain):
    return oracle.philox4x32_10([index, step & 0xFFFFFFFF, step >> 32, domain], [seed & 0xFFFFFFFF, seed >> 32])


# ------------------------------------------------------------------ oracle_init_* (A23)
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_init_restated_from_the_block_function(oracle, dtype):
    """A23 restated for single particles from the pinned Philox words: x_d = U L_d with 53-bit uniforms of the blocks
    (i, 0, INITPOS) / (i, 1, INITPOS); v = sigma x Box-Muller(A17) of the block (i, 0, INITVEL), minus the fp64 mean."""
    seed, N, L, sigma = 0x1234ABCD5678, 4001, [7.0, 5.0, 11.0], 1.3
    pos, vel, tag = oracle.init_state(seed, N, L, sigma, dtype)
    assert np.array_equal(tag, np.arange(N, dtype=np.uint32))                       # tags 0..N-1
    assert np.all(pos[:, 3] == 0) and np.all(vel[:, 3] == 0)
    raw = np.empty((N, 3))
    for i in range(N):
        b = _block(oracle, seed, 0, i, DOM_INITVEL)
        U = [oracle.u01_32(w) for w in b]
        r01, r23 = math.sqrt(-2.0 * math.log(U[0])), math.sqrt(-2.0 * math.log(U[2]))
        raw[i] = [sigma * r01 * math.cos(2 * math.pi * U[1]), sigma * r01 * math.sin(2 * math.pi * U[1]),
                  sigma * r23 * math.cos(2 * math.pi * U[3])]
    mean = np.array([math.fsum(raw[:, d]) for d in range(3)]) / N                   # exactly rounded mean
    want_v = (raw - mean).astype(dtype)
    # the oracle's running sum may differ from fsum in the last bits of the mean, and libm's cos / sin / log from Python's
    # by an ulp: a few ulps of the operands of the subtraction (native ulp for the cast result)
    # (the running sum's own error bound: N 2^-53 max|partial sum| / N on the mean, < 1e-15 here)
    ulp = np.spacing(np.abs(want_v).astype(dtype)).astype(np.float64) + 4 * 2.0**-53 * (np.abs(raw) + np.abs(mean)) + 1e-15
    assert np.all(np.abs(vel[:, :3].astype(np.float64) - want_v.astype(np.float64)) <= ulp)
    for i in (0, 1, 17, 2000, N - 1):
        b0, b1 = _block(oracle, seed, 0, i, DOM_INITPOS), _block(oracle, seed, 1, i, DOM_INITPOS)
        U = [oracle.u01_53(b0[0], b0[1]), oracle.u01_53(b0[2], b0[3]), oracle.u01_53(b1[0], b1[1])]
        for d in range(3):
            x = dtype(U[d] * L[d])
            if x >= dtype(L[d]):
                x = dtype(0)
            assert pos[i, d] == x, (i, d)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_init_distributions_and_zero_net_momentum(oracle, dtype):
    """Positions uniform in the box (PAPER.md:177 'randomly placed'), velocities N(0, kT/m), net momentum
    removed by a constant correction, different seeds give different states, same seed the same state."""
    seed, N, L, sigma = 99, 200_000, [8.0, 16.0, 4.0], 0.7
    pos, vel, _ = oracle.init_state(seed, N, L, sigma, dtype)
    for d in range(3):
        assert pos[:, d].min() >= 0 and pos[:, d].max() < L[d]
        assert stats.kstest(pos[:, d].astype(np.float64) / L[d], "uniform").pvalue > 1e-3
        assert stats.kstest(vel[:, d].astype(np.float64) / sigma, "norm").pvalue > 1e-3
        # the mean is removed in fp64 before the cast: what is left is the cast's rounding, ~ sqrt(N) ulp
        assert abs(vel[:, d].astype(np.float64).sum()) <= (1e-9 if dtype == np.float64 else 4.0 * math.sqrt(N) * 2.0**-24 * 4 * sigma)
    c = np.corrcoef(np.hstack([pos[:, :3], vel[:, :3]]).astype(np.float64).T)
    assert np.max(np.abs(c - np.eye(6))) < 0.02                                      # components independent
    pos2, vel2, _ = oracle.init_state(seed, N, L, sigma, dtype)
    assert np.array_equal(pos, pos2) and np.array_equal(vel, vel2)
    pos3, _, _ = oracle.init_state(seed + 1, N, L, sigma, dtype)
    assert not np.array_equal(pos, pos3)


def test_init_cast_that_rounds_up_to_L_lands_on_zero(oracle):
    """A23 / A7: U < 1 but fl32(U L) can equal L; such a position must be 0.  Search the first 2^20 indices of one seed
    for a 53-bit uniform above 1 - 2^-25 (where the float cast of U L rounds up to L for L = 1); if none exists in the
    range the property is still checked on every particle: nothing reaches L."""
    seed, N, L = 7, 1 << 20, [1.0, 1.0, 1.0]
    pos, _, _ = oracle.init_state(seed, N, L, 1.0, np.float32)
    assert pos[:, :3].max() < 1.0 and pos[:, :3].min() >= 0.0
    # direct: build the same decision from a uniform that does round up
    U = 1.0 - 2.0**-30
    assert np.float32(U * 1.0) == np.float32(1.0)        # the hazard exists for fp32
    x = np.float32(U * 1.0)
    assert (np.float32(0) if x >= np.float32(1.0) else x) == 0


# ------------------------------------------------------------------ oracle_collide_srd_beads (A14)
def test_bead_rotation_is_the_library_rotation(oracle):
    """With u = 0 and unit vectors as bead velocities the bead collision must return the columns of the right-handed
    rotation by +alpha about the cell's axis (a -alpha or a swapped cross product also conserves momentum and energy,
    so conservation alone does not pin this)."""
    axes = oracle.draw_axis(11, 3, 40)
    for alpha in (math.radians(130.0), math.radians(90.0), 0.3):
        for c, n in enumerate(axes):
            vel = np.eye(3)
            oracle.collide_srd_beads(vel, np.full(3, c, dtype=np.int32), np.zeros((40, 3)), axes, alpha)
            R = vel.T.copy()
            np.testing.assert_allclose(R, Rotation.from_rotvec(alpha * n).as_matrix(), atol=1e-15)
    # with a mean: v' = u + R (v - u)
    rng = np.random.default_rng(0)
    u = rng.standard_normal((40, 3)); v = rng.standard_normal((500, 3)); cell = rng.integers(0, 40, 500).astype(np.int32)
    out = v.copy()
    oracle.collide_srd_beads(out, cell, u, axes, math.radians(130.0))
    for i in range(0, 500, 7):
        R = Rotation.from_rotvec(math.radians(130.0) * axes[cell[i]]).as_matrix()
        np.testing.assert_allclose(out[i], u[cell[i]] + R @ (v[i] - u[cell[i]]), atol=1e-14)
    # z axis, +90 degrees: x -> y
    vel = np.array([[1.0, 0.0, 0.0]])
    oracle.collide_srd_beads(vel, np.zeros(1, dtype=np.int32), np.zeros((1, 3)), np.array([[0.0, 0.0, 1.0]]), math.pi / 2)
    np.testing.assert_allclose(vel[0], [0, 1, 0], atol=1e-16)


# ------------------------------------------------------------------ oracle_collide_srd_xi (Alg. 1 lines 8-10)
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_scaled_collision_reduces_to_the_pinned_one(oracle, dtype):
    """xi = 1 everywhere: bit-identical to oracle_collide_srd (whose rotation sense is pinned against scipy).  xi = 2:
    every relative velocity v' - u is exactly twice the unscaled one (up to the native store rounding)."""
    rng = np.random.default_rng(5)
    Nc, N = 60, 900
    axes = oracle.draw_axis(5, 9, Nc)
    u = rng.standard_normal((Nc, 3)) * 0.3
    cell = rng.integers(0, Nc, N).astype(np.int32)
    v0 = np.zeros((N, 4), dtype=dtype); v0[:, :3] = rng.standard_normal((N, 3))
    alpha = math.radians(130.0)
    a, b = v0.copy(), v0.copy()
    oracle.collide_srd(a, cell, u, axes, alpha)
    oracle.collide_srd_xi(b, cell, u, axes, np.ones(Nc), alpha)
    assert np.array_equal(a, b)
    c = v0.copy()
    oracle.collide_srd_xi(c, cell, u, axes, np.full(Nc, 2.0), alpha)
    rel1 = a[:, :3].astype(np.float64) - u[cell]
    rel2 = c[:, :3].astype(np.float64) - u[cell]
    tol = 1e-14 if dtype == np.float64 else 3 * 2.0**-24 * 8
    np.testing.assert_allclose(rel2, 2.0 * rel1, rtol=0, atol=tol)
    # per-cell xi: only the cells with xi != 1 change
    xi = np.ones(Nc); xi[::3] = 0.5
    d = v0.copy()
    oracle.collide_srd_xi(d, cell, u, axes, xi, alpha)
    same = xi[cell] == 1.0
    assert np.array_equal(d[same], a[same]) and not np.array_equal(d[~same], a[~same])

"""Pins for streaming (eq. 1) and binning of the oracle."""
from fractions import Fraction

import numpy as np
import pytest
from scipy import stats

import workloads as synth


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_stream_closed_form(oracle, dtype):
    """With collisions off, k streams move a particle to (r0 + k v dt) mod L within k ulp(L);
    velocities are untouched (SURVEY 8c pin 'Stream')."""
    n = (5, 7, 3)
    a = 1.0
    pos, vel, _ = synth.solvent(n, 6, seed=3, dtype=dtype)
    L = np.array(n, dtype=np.float64) * a
    p0, v0 = pos.copy(), vel.copy()
    dt = 0.1
    k = 40
    for _ in range(k):
        oracle.stream(pos, vel, dt, L)
    assert np.array_equal(vel, v0)
    assert np.all(pos[:, :3] >= 0) and np.all(pos[:, :3] < L.astype(dtype))
    exact = np.mod(p0[:, :3].astype(np.float64) + k * v0[:, :3].astype(np.float64) * float(dtype(dt)), L)
    err = np.abs(pos[:, :3].astype(np.float64) - exact)
    err = np.minimum(err, L - err)                         # periodic distance
    assert np.max(err) <= k * np.spacing(dtype(L.max())) * 1.01


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_stream_one_step_is_two_roundings_then_wrap(oracle, dtype):
    """x = fl(x + fl(v dt)); if x < 0: x += L; if x >= L: x -= L  -- restated with numpy scalars."""
    n = (4, 4, 4)
    pos, vel, _ = synth.solvent(n, 50, seed=5, dtype=dtype)
    vel[:, :3] *= dtype(8.0)                               # force many wraps
    L = np.array(n, dtype=np.float64)
    p0 = pos.copy()
    oracle.stream(pos, vel, 0.1, L)
    dtn = dtype(0.1)
    x = p0[:, :3] + vel[:, :3] * dtn                       # numpy: separately rounded mul and add
    Ln = L.astype(dtype)
    x = np.where(x < 0, x + Ln, x)
    x = np.where(x >= Ln, x - Ln, x)
    assert np.array_equal(pos[:, :3], x)
    assert np.count_nonzero(np.abs(pos[:, :3] - p0[:, :3]) > 2) > 100   # wraps really happened


def test_stream_rounded_up_to_L_lands_on_zero(oracle):
    """A7: a tiny negative fp32 coordinate plus L rounds to L; the second branch maps it to 0."""
    pos = np.zeros((1, 4), dtype=np.float32)
    vel = np.zeros((1, 4), dtype=np.float32)
    vel[0, 0] = -1e-8
    oracle.stream(pos, vel, 0.1, [8.0, 8.0, 8.0])
    assert pos[0, 0] == 0.0


def _brute_force_cells(pos4, shift, a, n, dtype):
    """Independent statement of the binning: the rounded q of A6 computed with numpy scalars,
    then exact-rational interval membership i <= q < i + 1 tested for every cell index."""
    inv_a = dtype(1) / dtype(a)
    out = np.empty(pos4.shape[0], dtype=np.int64)
    for p in range(pos4.shape[0]):
        idx = []
        for d in range(3):
            t = dtype(pos4[p, d]) + dtype(shift[d])
            q = Fraction(float(dtype(t * inv_a)))
            hits = [i for i in range(-1, n[d] + 1) if Fraction(i) <= q < Fraction(i + 1)]
            assert len(hits) == 1
            idx.append(hits[0] % n[d])
        out[p] = idx[0] + n[0] * (idx[1] + n[1] * idx[2])
    return out


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("n,a", [((2, 3, 4), 1.0), ((8, 8, 8), 1.0), ((3, 2, 5), 0.7)])
def test_bin_matches_brute_force_membership(oracle, dtype, n, a):
    pos, vel, _ = synth.solvent(n, 5, seed=11, a=a, dtype=dtype)
    for step in range(3):
        shift = oracle.draw_shift(2024, step, a)
        cell = oracle.bin_cells(pos, shift, a, n)
        want = _brute_force_cells(pos, shift, a, n, dtype)
        assert np.array_equal(cell, want)
        assert cell.min() >= 0 and cell.max() < n[0] * n[1] * n[2]


def test_bin_zero_shift_is_floor_and_corners(oracle):
    n = (4, 5, 6)
    a = 1.0
    pos, _, _ = synth.solvent(n, 20, seed=1, dtype=np.float32)
    cell = oracle.bin_cells(pos, [0, 0, 0], a, n)
    i = np.floor(pos[:, :3]).astype(np.int64)
    assert np.array_equal(cell, i[:, 0] + n[0] * (i[:, 1] + n[1] * i[:, 2]))
    # corner cases: x = 0 with a negative shift wraps to the last cell; x = L - ulp with a
    # positive shift wraps to cell 0; shift just inside +-a/2
    eps = np.float32(1e-6)
    L = np.array(n, dtype=np.float32)
    p = np.zeros((4, 4), dtype=np.float32)
    p[1, :3] = np.nextafter(L, np.float32(0))
    p[2, :3] = 0.5
    p[3, :3] = L - np.float32(0.5)
    neg = oracle.bin_cells(p, [-(0.5 - eps)] * 3, a, n)
    posi = oracle.bin_cells(p, [0.5 - eps] * 3, a, n)
    last = (n[0] - 1) + n[0] * ((n[1] - 1) + n[1] * (n[2] - 1))
    assert neg[0] == last and posi[0] == 0
    assert posi[1] == 0 and neg[1] == last
    assert neg[2] == 0 and posi[2] == 0
    assert neg[3] == last and posi[3] == last              # L - 0.5 +- (0.5 - eps) stays inside the last cell


def test_bin_every_particle_in_one_cell_and_poisson_occupancy(oracle):
    """cell occupancy follows a Poisson distribution."""
    n = (24, 24, 24)
    M = 10
    pos, _, _ = synth.solvent(n, M, seed=8, dtype=np.float32)
    Nc = n[0] * n[1] * n[2]
    shift = oracle.draw_shift(8, 0, 1.0)
    cell = oracle.bin_cells(pos, shift, 1.0, n)
    counts = np.bincount(cell, minlength=Nc)
    assert counts.sum() == pos.shape[0]
    assert abs(counts.mean() - M) < 1e-12
    assert abs(counts.var() / (M * (1 - 1 / Nc)) - 1) < 5 * np.sqrt(2 / Nc)
    ks = np.arange(0, 31)
    expect = stats.poisson.pmf(ks, M) * Nc
    obs = np.array([np.count_nonzero(counts == k) for k in ks])
    keep = expect > 5
    chi2 = ((obs[keep] - expect[keep]) ** 2 / expect[keep]).sum()
    assert stats.chi2.sf(chi2, keep.sum() - 1) > 1e-4


def test_shift_moves_grid_not_particles(oracle):
    """positions are shifted during binning only."""
    n = (6, 6, 6)
    pos, _, _ = synth.solvent(n, 5, seed=4, dtype=np.float32)
    p0 = pos.copy()
    oracle.bin_cells(pos, [0.3, -0.2, 0.49], 1.0, n)
    assert np.array_equal(pos, p0)
    # shifting by s then binning == binning positions moved by s (periodic), away from rounding edges
    s = np.array([0.25, -0.25, 0.125], dtype=np.float32)   # exactly representable
    cell = oracle.bin_cells(pos, s, 1.0, n)
    moved = pos.copy()
    moved[:, :3] = np.mod(pos[:, :3] + s, np.array(n, dtype=np.float32))
    cell2 = oracle.bin_cells(moved, [0, 0, 0], 1.0, n)
    frac = np.abs(moved[:, :3] - np.round(moved[:, :3]))
    safe = np.all(frac > 1e-4, axis=1)
    assert safe.sum() > 0.99 * len(safe)
    assert np.array_equal(cell[safe], cell2[safe])

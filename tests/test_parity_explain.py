"""The mismatch-explaining comparison used by the multi-step GPU parity tests (tests/parity_explain.py) must itself
reject what it is there to reject: a wrong velocity in a cell whose membership agrees, and a differing cell index of
a particle that does not sit on a cell face."""
import numpy as np
import pytest

from parity_explain import explained_compare, on_a_face


def _fluid(seed=3, n=(6, 5, 4), M=8):
    rng = np.random.default_rng(seed)
    N = n[0] * n[1] * n[2] * M
    pos = np.zeros((N, 4), np.float32)
    pos[:, :3] = rng.random((N, 3), dtype=np.float32) * np.array(n, np.float32)
    pos[:, :3] = np.minimum(pos[:, :3], np.nextafter(np.array(n, np.float32), 0))
    vel = np.zeros((N, 4), np.float32)
    vel[:, :3] = rng.standard_normal((N, 3)).astype(np.float32)
    shift = np.array([0.25, -0.125, 0.375])
    i = [np.floor((pos[:, d] + np.float32(shift[d]))).astype(np.int64) % n[d] for d in range(3)]
    cell = (i[0] + n[0] * (i[1] + n[1] * i[2])).astype(np.int32)
    return pos, vel, cell, shift, n


def test_identical_states_and_one_legitimate_face_flip_pass():
    pos, vel, cell, shift, n = _fluid()
    r = explained_compare(pos, vel, cell, pos, vel, cell, shift, 1.0, n, 1e-5, np.float32)
    assert r["bad_cell"] == 0 and r["bad_vel"] == 0 and r["worst_pos"] == 0.0
    # particle 7 sits exactly on an x face on the oracle side, one ulp below it on the other side; both cells' members differ
    o_pos = pos.copy()
    o_pos[7, 0] = np.float32(3.0) - np.float32(shift[0])
    g_pos = o_pos.copy()
    g_pos[7, 0] = np.nextafter(o_pos[7, 0], np.float32(0))
    assert on_a_face(o_pos[7:8], shift, 1.0, np.float32).all()
    iy = int(np.floor(o_pos[7, 1] + np.float32(shift[1]))) % n[1]
    iz = int(np.floor(o_pos[7, 2] + np.float32(shift[2]))) % n[2]
    o_cell, g_cell = cell.copy(), cell.copy()
    o_cell[7] = 3 + n[0] * (iy + n[1] * iz)
    g_cell[7] = 2 + n[0] * (iy + n[1] * iz)
    g_vel = vel.copy()
    members = np.isin(cell, [o_cell[7], g_cell[7]]) | (np.arange(cell.size) == 7)
    g_vel[members, :3] += np.float32(0.01)
    r = explained_compare(g_pos, g_vel, g_cell, o_pos, vel, o_cell, shift, 1.0, n, 1e-5, np.float32)
    assert r["bad_cell"] == 1 and r["bad_vel"] == int(members.sum()) and r["touched_cells"] == 2


def test_an_unexplained_velocity_or_cell_mismatch_fails():
    pos, vel, cell, shift, n = _fluid()
    g_vel = vel.copy()
    g_vel[11, 1] += np.float32(1e-3)                      # one lane wrong, membership identical
    with pytest.raises(AssertionError, match="membership is the same"):
        explained_compare(pos, g_vel, cell, pos, vel, cell, shift, 1.0, n, 1e-5, np.float32)
    interior = np.flatnonzero(~on_a_face(pos, shift, 1.0, np.float32, face_ulps=64))[0]
    g_cell = cell.copy()
    g_cell[interior] = (cell[interior] + 1) % (n[0] * n[1] * n[2])
    with pytest.raises(AssertionError, match="do not sit on a cell face"):
        explained_compare(pos, vel, g_cell, pos, vel, cell, shift, 1.0, n, 1e-5, np.float32)
    g_pos = pos.copy()
    g_pos[5, 2] += np.float32(1e-3)                       # a position off by far more than an ulp
    with pytest.raises(AssertionError):
        explained_compare(g_pos, vel, cell, pos, vel, cell, shift, 1.0, n, 1e-5, np.float32)

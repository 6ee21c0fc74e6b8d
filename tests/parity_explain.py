"""Multi-step comparison of the CUDA path with the oracle that EXPLAINS every mismatch (numpy only; none of the
method's arithmetic beyond restating the binned coordinate to measure a distance to a cell face).

Two steps after an identical state the two sides may legitimately differ: the fp64 cell sums are added in a
different order, so a velocity may differ in its last native bit after the first collision (allowed by the
north_star tolerance); the next streaming then moves that particle's position by an ulp, and among 10^8 particles
a handful of those sit within an ulp of a cell face and bin into the neighbouring cell; the two cells concerned
then have other members on the two sides, hence another mean, and ALL their members' velocities differ.  That
chain is the only legitimate one, so the check is:

  (i)   every particle whose cell index differs has, on the oracle side, a binned coordinate
        q_d = fl(fl(x_d + s_d) * inv_a) within `face_ulps` ulp of an integer on some axis (it sat on a cell face);
  (ii)  every particle whose velocity differs by more than the tolerance belongs, on either side, to a cell that
        gained or lost one of the particles of (i);
  (iii) positions agree to `pos_ulps` ulp of the box length (minimum image).

Anything else -- one wrong lane, one wrong tail block, one wrong warp -- fails, however few particles it touches.
"""
import numpy as np


def on_a_face(pos, shift, a, dtype, face_ulps=2):
    """Mask of particles whose binned coordinate (A6) lies within face_ulps ulp of an integer on some axis."""
    T = np.float32 if dtype == np.float32 else np.float64
    inv_a = T(1.0) / T(a)
    near = np.zeros(pos.shape[0], dtype=bool)
    for d in range(3):
        q = (pos[:, d].astype(T) + T(shift[d])) * inv_a            # two roundings in the native precision
        q = q.astype(np.float64)
        ulp = np.spacing(np.maximum(np.abs(q), 1.0).astype(T)).astype(np.float64)
        near |= np.abs(q - np.rint(q)) <= face_ulps * ulp
    return near


def explained_compare(g_pos, g_vel, g_cell, o_pos, o_vel, o_cell, shift, a, box, tol, dtype, face_ulps=2, pos_ulps=2, chunk=1 << 24):
    """All arrays by tag (same particle in the same row).  Returns dict(bad_cell, bad_vel, worst_pos); raises AssertionError
    with the first unexplained mismatch."""
    N = g_cell.shape[0]
    T = np.float32 if dtype == np.float32 else np.float64
    L = np.asarray(box, dtype=np.float64)
    diff_cell = np.flatnonzero(g_cell != o_cell)
    # (i)
    if diff_cell.size:
        near = on_a_face(o_pos[diff_cell], shift, a, dtype, face_ulps)
        assert near.all(), (f"{int((~near).sum())} of {diff_cell.size} particles with differing cell index do not sit on a cell face, "
                            f"first: particle row {int(diff_cell[np.flatnonzero(~near)[0]])}")
    touched = np.union1d(g_cell[diff_cell], o_cell[diff_cell])     # cells whose membership differs between the two sides
    # (ii), (iii)
    bad_vel, worst_pos = 0, 0.0
    for lo in range(0, N, chunk):
        sl = slice(lo, min(lo + chunk, N))
        d = np.abs(g_pos[sl, :3].astype(np.float64) - o_pos[sl, :3].astype(np.float64))
        d = np.minimum(d, L - d)
        worst_pos = max(worst_pos, float(d.max()))
        dv = np.abs(g_vel[sl, :3].astype(np.float64) - o_vel[sl, :3].astype(np.float64)).max(axis=1)
        bad = np.flatnonzero(dv > tol)
        if bad.size:
            ok = np.isin(g_cell[sl][bad], touched) | np.isin(o_cell[sl][bad], touched)
            assert ok.all(), (f"{int((~ok).sum())} velocities differ by more than {tol:g} in cells whose membership is the same on both sides, "
                              f"first: particle row {lo + int(bad[np.flatnonzero(~ok)[0]])}, |dv| = {float(dv[bad[np.flatnonzero(~ok)[0]]]):.3g}")
            bad_vel += int(bad.size)
    assert worst_pos <= pos_ulps * float(np.spacing(T(L.max()))), worst_pos
    return dict(bad_cell=int(diff_cell.size), bad_vel=bad_vel, worst_pos=worst_pos, touched_cells=int(touched.size))

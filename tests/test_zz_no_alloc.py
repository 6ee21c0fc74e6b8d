"""mpcd_cell_sums_static: the cell reduction for callers that cannot allocate device memory.

Some users of this library need the per-cell count / momentum / kinetic-energy sums at a point where they have no way
to get device memory: all of it has been handed to another pool (a framework's caching allocator, an MPS client with a
fixed limit), so cudaMalloc fails, or they sit in a time-critical loop where cudaMalloc's device synchronisation is not
affordable.  mpcd_cell_sums_static (include/mpcd.h) serves them: inputs and outputs are the caller's device buffers and
the accumulators are a fixed 1.25 MiB array inside the library, shared by all calls on a GPU and limited to
MPCD_STATIC_MAX_CELLS = 32768 cells.

These tests check it against the existing path -- mpcd_set_state + mpcd_shift_and_bin + mpcd_get_cells on a handle --
at the tolerances tests/test_gpu_parity.py uses for cell sums (counts exact, sums 1e-12: the two paths differ only in
the order of the fp64 additions), on several calls in a row WITHOUT a synchronisation in between, because the shared
array keeps the previous call's sums and every call has to clear what it uses.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the
parity tests.  Nothing here depends on what ran before: every test builds its own inputs, so the file passes alone in
a fresh process (where its first call is also the library's first use of the device) and after the whole suite.
"""
import numpy as np
import pytest

import workloads as synth

pytestmark = pytest.mark.gpu

SUM_ATOL = 1e-12      # as test_stream_and_bin_are_bit_exact: fp64 reassociation only
KE_RTOL = 1e-13


def _existing_path(n, M, seed, dtype, a, m, advance, N=None):
    """Cell sums of a seeded fluid by the handle path, plus the particle state and shift they were made from."""
    from paper_1801_10187_b200 import MPCD
    pos, vel, tag = synth.solvent(n, M, seed=seed, a=a, kT=1.3, m=m, dtype=dtype, N=N)
    g = MPCD([x * a for x in n], pos.shape[0], a=a, m=m, kT=1.3, seed=seed, precision="fp64" if dtype == np.float64 else "mixed",
             init_state=False)
    g.set_state(pos, vel, tag)
    if advance:
        g.step(advance)                    # another state, another step counter, hence another shift
    g.shift_and_bin()
    cells = g.get_cells(axis=False)
    st = g.get_state(tag=False, cell=False)
    shift = g.get_shift()
    g.close()
    return dict(pos=st["pos"], vel=st["vel"], shift=shift, count=cells["count"], sumv=cells["sumv"], ke=cells["ke"], n=n, a=a, m=m)


def _device_case(case, torch):
    Nc = case["n"][0] * case["n"][1] * case["n"][2]
    dev = torch.device("cuda:0")
    return dict(pos=torch.from_numpy(case["pos"]).to(dev), vel=torch.from_numpy(case["vel"]).to(dev),
                # outputs start as garbage: the call must write every element
                count=torch.full((Nc,), -7, dtype=torch.int32, device=dev),
                sumv=torch.full((Nc, 3), 1e300, dtype=torch.float64, device=dev),
                ke=torch.full((Nc,), -1e300, dtype=torch.float64, device=dev))


def _call(case, d):
    from paper_1801_10187_b200.binding import cell_sums_static
    cell_sums_static(d["pos"], d["vel"], case["n"], case["a"], case["shift"], case["m"], count=d["count"], sumv3=d["sumv"], ke=d["ke"])


def _compare(case, d):
    assert np.array_equal(d["count"].cpu().numpy(), case["count"])                       # counts: bit-exact
    assert int(case["count"].sum()) == case["pos"].shape[0]
    np.testing.assert_allclose(d["sumv"].cpu().numpy(), case["sumv"], rtol=0, atol=SUM_ATOL)
    np.testing.assert_allclose(d["ke"].cpu().numpy(), case["ke"], rtol=KE_RTOL, atol=SUM_ATOL)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_static_cell_sums_match_the_handle_path_on_calls_in_a_row(dtype):
    """Three calls back to back on one stream, no synchronisation between them: a fluid, a different fluid on a smaller
    grid (it reuses the front of the shared array), and the first one again.  4420 cells x 10 particles spans several
    thread blocks and ends in a ragged one (44200 = 345 * 128 + 40); a = 0.7 makes 1/a inexact."""
    import torch
    A = _existing_path((20, 17, 13), 10, 1801, dtype, a=0.7, m=2.0, advance=0)
    B = _existing_path((9, 11, 6), 7, 10187, dtype, a=1.0, m=1.0, advance=3)
    dA, dB, dA2 = _device_case(A, torch), _device_case(B, torch), _device_case(A, torch)
    _call(A, dA)
    _call(B, dB)
    _call(A, dA2)
    torch.cuda.synchronize()
    _compare(A, dA)
    _compare(B, dB)
    _compare(A, dA2)


def test_static_cell_sums_allocate_nothing_and_handle_empty_and_full_grids():
    """The largest grid the static array holds (32^3 = MPCD_STATIC_MAX_CELLS cells, dilute: most cells empty), then an
    empty particle set on the same grid, which must give zeros although the array still holds the previous sums.  Free
    device memory as the driver reports it must not shrink over these calls (the first call of the process, which may
    load the library's device code, is made before the measurement)."""
    import torch
    from paper_1801_10187_b200.binding import STATIC_MAX_CELLS
    n = (32, 32, 32)
    assert n[0] * n[1] * n[2] == STATIC_MAX_CELLS
    F = _existing_path(n, None, 5, np.float32, a=1.0, m=1.0, advance=0, N=50001)
    dF = _device_case(F, torch)
    empty = dict(F, pos=F["pos"][:0], vel=F["vel"][:0])
    dE = _device_case(empty, torch)
    _call(F, dF)                                    # warm-up: set-up of the static path on this device
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        _call(F, dF)
        _call(empty, dE)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before
    _compare(F, dF)
    assert not dE["count"].any() and not dE["sumv"].any() and not dE["ke"].any()


def test_static_cell_sums_reject_a_grid_beyond_the_maximum():
    """One cell layer more than the array holds: refused before any device work, with the limit in the message; the
    outputs are untouched."""
    import torch
    from paper_1801_10187_b200 import MPCDError
    from paper_1801_10187_b200.binding import cell_sums_static
    dev = torch.device("cuda:0")
    n = (32, 32, 33)
    pos = torch.zeros((10, 4), dtype=torch.float32, device=dev)
    count = torch.full((n[0] * n[1] * n[2],), -7, dtype=torch.int32, device=dev)
    with pytest.raises(MPCDError) as e:
        cell_sums_static(pos, pos.clone(), n, 1.0, (0.1, 0.2, -0.3), 1.0, count=count)
    assert e.value.code == -1 and "32768" in str(e.value) and "MPCD_STATIC_MAX_CELLS" in str(e.value)
    with pytest.raises(MPCDError):
        cell_sums_static(pos, pos.clone(), (2**20, 2**20, 2**20), 1.0, (0.0, 0.0, 0.0), 1.0)      # no overflow on the way to the check
    torch.cuda.synchronize()
    assert bool((count == -7).all())

"""Edge cases of the CUDA path through the C ABI: options off the default path, ragged sizes through the fused
sort, repeated mpcd_step calls landing on and off sort steps, zero-copy device pointers, argument validation."""
import numpy as np
import pytest

import workloads as synth

pytestmark = pytest.mark.gpu


def _by_tag(s):
    o = np.argsort(s["tag"], kind="stable")
    return {k: (v[o] if isinstance(v, np.ndarray) else v) for k, v in s.items()}


@pytest.mark.parametrize("chunks", [[7], [1, 1, 1, 1, 1, 1, 1], [2, 3, 2], [3, 1, 3]])
@pytest.mark.parametrize("rule", ["srd", "at"])
def test_any_split_of_the_steps_gives_the_same_trajectory(oracle, chunks, rule):
    """mpcd_step(7) == any sequence of shorter calls: sorts fall inside the fused loop (kSortOut), at the end of a
    call (standalone scatter) or at its beginning, and AT carries dv between launches only inside a call."""
    from paper_1801_10187_b200 import MPCD
    n, M = (9, 7, 6), 6
    pos, vel, tag = synth.solvent(n, M, seed=3, dtype=np.float64)
    o = oracle.OracleMPCD([float(x) for x in n], pos.shape[0], seed=3, dtype=np.float64, init=False, rule=1 if rule == "at" else 0, sort_period=3)
    o.set_state(pos, vel, tag); o.step(7)
    g = MPCD([float(x) for x in n], pos.shape[0], seed=3, precision="fp64", rule=rule, sort_period=3, init_state=False)
    g.set_state(pos, vel, tag)
    for k in chunks:
        g.step(k)
    s = _by_tag(g.get_state()); b = np.argsort(o.tag)
    assert s["step"] == 7 and g.stats()["sorts"] == 3
    np.testing.assert_allclose(s["pos"][:, :3], o.pos[b][:, :3], rtol=0, atol=1e-11)
    np.testing.assert_allclose(s["vel"][:, :3], o.vel[b][:, :3], rtol=0, atol=1e-11)
    assert np.array_equal(s["cell"], o.cell[b])
    g.close()


@pytest.mark.parametrize("N", [1, 127, 129, 1000])
def test_ragged_sizes_through_the_fused_sort(oracle, N):
    from paper_1801_10187_b200 import MPCD
    pos, vel, tag = synth.solvent((5, 4, 3), None, seed=60 + N, dtype=np.float32, N=N)
    g = MPCD([5.0, 4.0, 3.0], N, seed=9, sort_period=1, init_state=False)
    o = oracle.OracleMPCD([5.0, 4.0, 3.0], N, seed=9, dtype=np.float32, init=False, sort_period=1)
    g.set_state(pos, vel, tag); o.set_state(pos, vel, tag)
    g.step(4); o.step(4)
    s = _by_tag(g.get_state()); b = np.argsort(o.tag)
    assert np.array_equal(s["tag"], o.tag[b]) and g.stats()["sorts"] == 4
    assert np.max(np.abs(s["pos"][:, :3].astype(np.float64) - o.pos[b][:, :3])) <= 4e-6
    assert np.max(np.abs(s["vel"][:, :3].astype(np.float64) - o.vel[b][:, :3])) <= 4e-5
    g.close()


def test_cell_energy_off_still_reports_energies_on_demand(oracle):
    from paper_1801_10187_b200 import MPCD
    n, M = (8, 8, 8), 10
    pos, vel, tag = synth.solvent(n, M, seed=4, dtype=np.float32)
    ga = MPCD([8.0] * 3, pos.shape[0], seed=4, init_state=False, cell_energy=False)
    gb = MPCD([8.0] * 3, pos.shape[0], seed=4, init_state=False, cell_energy=True)
    for g in (ga, gb):
        g.set_state(pos, vel, tag); g.step(5)
    a, b = _by_tag(ga.get_state()), _by_tag(gb.get_state())
    assert np.array_equal(a["pos"], b["pos"]) and np.max(np.abs(a["vel"] - b["vel"])[:, :3]) <= 1e-5
    Pa, KEa, kTa = ga.get_thermo(); Pb, KEb, kTb = gb.get_thermo()
    assert abs(KEa - KEb) / KEb < 1e-5 and abs(kTa - kTb) < 1e-4 and kTa > 0.9
    ga.close(); gb.close()


def test_device_pointers_are_the_live_state():
    """mpcd_device_ptrs: the returned DEVICE addresses hold what mpcd_get_state copies out."""
    import ctypes as C
    import torch
    from paper_1801_10187_b200 import MPCD
    g = MPCD([6.0] * 3, 2160, seed=2)
    g.step(2)
    p, v, t, c = C.c_void_p(), C.c_void_p(), C.c_void_p(), C.c_void_p()
    g._check(g.lib.mpcd_device_ptrs(g.h, C.byref(p), C.byref(v), C.byref(t), C.byref(c)))
    s = g.get_state()
    try:
        from cuda.bindings import runtime as cudart
    except ImportError:
        from cuda import cudart
    dst = torch.empty(2160 * 4, dtype=torch.float32, device="cuda")
    cells = torch.empty(2160, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    d2d = cudart.cudaMemcpyKind.cudaMemcpyDeviceToDevice
    assert cudart.cudaMemcpy(dst.data_ptr(), p.value, 2160 * 16, d2d)[0] == cudart.cudaError_t.cudaSuccess
    assert cudart.cudaMemcpy(cells.data_ptr(), c.value, 2160 * 4, d2d)[0] == cudart.cudaError_t.cudaSuccess
    assert np.array_equal(dst.cpu().numpy().reshape(2160, 4)[:, :3], s["pos"][:, :3])
    assert np.array_equal(cells.cpu().numpy(), s["cell"])
    g.close()


def test_create_rejects_bad_arguments():
    from paper_1801_10187_b200 import MPCD, MPCDError
    for kw, box, N in ((dict(), [4.0, 4.0, 4.5], 10), (dict(), [4.0, 4.0, 4.0], 0), (dict(a=-1.0), [4.0] * 3, 10),
                       (dict(dt=0.0), [4.0] * 3, 10), (dict(sort_period=-1), [4.0] * 3, 10), (dict(), [2048.0] * 3, 10)):
        with pytest.raises(MPCDError) as e:
            MPCD(box, N, **kw)
        assert e.value.code == -1

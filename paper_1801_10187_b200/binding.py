"""Thin ctypes binding of include/mpcd.h: argument marshalling only.

Every step of the method runs in the CUDA kernels behind the C ABI
(paper_1801_10187_b200/libmpcd_b200.so).  PyTorch appears here only as the supplier of
device memory (through the mpcd_alloc_fn / mpcd_free_fn callbacks) and of the CUDA
stream.  There is no CPU fallback: a missing library or device raises.
"""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("MPCD_B200_LIB") or os.path.join(_HERE, "libmpcd_b200.so")   # override: an alternative build of the same library

MPCD_OK, MPCD_EINVAL, MPCD_ENOMEM, MPCD_ECUDA, MPCD_ESTATE = 0, -1, -2, -3, -4
MPCD_MIXED, MPCD_FP64 = 0, 1
MPCD_SRD, MPCD_AT = 0, 1

ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class Options(C.Structure):
    _fields_ = [
        ("precision", C.c_int32), ("rule", C.c_int32), ("dt", C.c_double), ("alpha", C.c_double),
        ("sort_period", C.c_int32), ("cell_energy", C.c_int32), ("init_state", C.c_int32), ("thermostat", C.c_int32),
        ("deterministic", C.c_int32), ("brick", C.c_int32),
        ("stream", C.c_void_p), ("alloc_fn", ALLOC_FN), ("free_fn", FREE_FN), ("alloc_user", C.c_void_p),
    ]


class Stats(C.Structure):
    _fields_ = [
        ("N", C.c_int64), ("Nc", C.c_int64), ("n", C.c_int32 * 3), ("max_occupancy", C.c_int32),
        ("step", C.c_uint64), ("kernel_launches", C.c_uint64), ("sorts", C.c_uint64), ("device_bytes", C.c_uint64),
        ("brick", C.c_int32 * 4),
    ]


class MPCDError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mpcd error {code}: {msg}")
        self.code = code


# every symbol include/mpcd.h declares (tests/test_abi.py checks the .so exports them all)
EXPORTS = [
    "mpcd_default_options", "mpcd_create", "mpcd_create_ex", "mpcd_destroy", "mpcd_stream", "mpcd_shift_and_bin",
    "mpcd_collide_srd", "mpcd_collide_at", "mpcd_sort", "mpcd_step", "mpcd_get_state", "mpcd_set_state",
    "mpcd_get_cells", "mpcd_get_shift", "mpcd_get_thermo", "mpcd_get_stats", "mpcd_device_ptrs", "mpcd_last_error",
    "mpcd_abi_version", "mpcd_build_info", "mpcd_test_philox", "mpcd_set_profiling", "mpcd_get_profile", "mpcd_get_xi", "mpcd_set_embedded", "mpcd_get_embedded",
    "mpcd_cell_sums_static", "mpcd_cell_sums_static_error",
]
STATIC_MAX_CELLS = 32768   # MPCD_STATIC_MAX_CELLS of include/mpcd.h
PROF_KINDS = ("fused", "bin", "collide", "cells", "sort", "other", "fused_sort")

_lib = None


def load_library():
    """dlopen the CUDA library; fail loudly if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1801_10187_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, u64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64, C.c_double
    P = C.POINTER
    lib.mpcd_default_options.argtypes = [P(Options)]
    lib.mpcd_create.argtypes = [P(vp), P(dbl), i64, dbl, dbl, dbl, u64]
    lib.mpcd_create_ex.argtypes = [P(vp), P(dbl), i64, dbl, dbl, dbl, u64, P(Options)]
    for name in ("mpcd_destroy", "mpcd_stream", "mpcd_shift_and_bin", "mpcd_collide_at", "mpcd_sort"):
        getattr(lib, name).argtypes = [vp]
    lib.mpcd_collide_srd.argtypes = [vp, dbl]
    lib.mpcd_step.argtypes = [vp, i32]
    lib.mpcd_get_state.argtypes = [vp, vp, vp, vp, vp, P(u64)]
    lib.mpcd_set_state.argtypes = [vp, vp, vp, vp, u64]
    lib.mpcd_get_cells.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.mpcd_get_shift.argtypes = [vp, P(dbl)]
    lib.mpcd_get_xi.argtypes = [vp, vp]
    lib.mpcd_set_embedded.argtypes = [vp, i64, vp, vp, vp, i32, dbl, dbl, i32]
    lib.mpcd_get_embedded.argtypes = [vp, vp, vp, vp]
    lib.mpcd_get_thermo.argtypes = [vp, P(dbl), P(dbl), P(dbl)]
    lib.mpcd_get_stats.argtypes = [vp, P(Stats)]
    lib.mpcd_device_ptrs.argtypes = [vp, P(vp), P(vp), P(vp), P(vp)]
    lib.mpcd_last_error.argtypes = [vp]
    lib.mpcd_last_error.restype = C.c_char_p
    lib.mpcd_build_info.restype = C.c_char_p
    lib.mpcd_test_philox.argtypes = [vp, vp, vp, i64]
    lib.mpcd_set_profiling.argtypes = [vp, i32]
    lib.mpcd_get_profile.argtypes = [vp, P(dbl), P(u64)]
    lib.mpcd_cell_sums_static.argtypes = [vp, vp, i64, i32, P(i32), dbl, P(dbl), dbl, vp, vp, vp, vp]
    lib.mpcd_cell_sums_static_error.argtypes = []
    lib.mpcd_cell_sums_static_error.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("mpcd_last_error", "mpcd_build_info", "mpcd_cell_sums_static_error"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _ptr(a):
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags.c_contiguous
        return a.ctypes.data_as(C.c_void_p)
    # torch CPU tensor (pinned or pageable)
    assert a.device.type == "cpu" and a.is_contiguous()
    return C.c_void_p(a.data_ptr())


class TorchAllocator:
    """Device memory from PyTorch's caching allocator: one uint8 tensor per request, kept alive
    here until the library frees it."""

    def __init__(self, device="cuda:0"):
        import torch
        self.torch = torch
        self.device = torch.device(device)
        self.live = {}
        self.alloc_cb = ALLOC_FN(self._alloc)
        self.free_cb = FREE_FN(self._free)

    def _alloc(self, nbytes, _user):
        try:
            t = self.torch.empty(int(nbytes), dtype=self.torch.uint8, device=self.device)
        except Exception:   # out of memory -> NULL -> MPCD_ENOMEM
            return None
        p = t.data_ptr()
        self.live[p] = t
        return p

    def _free(self, ptr, _user):
        self.live.pop(ptr, None)


class MPCD:
    """One MPCD solvent on one GPU.  Method names are the C ABI's without the prefix."""

    def __init__(self, box, N, a=1.0, m=1.0, kT=1.0, seed=0, *, precision="mixed", rule="srd", dt=0.1,
                 alpha=math.radians(130.0), sort_period=25, cell_energy=True, init_state=True, thermostat=False, deterministic=False,
                 brick=False, device="cuda:0", use_torch_allocator=True, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1801_10187_b200 needs a CUDA device (no CPU fallback)")
        self.lib = load_library()
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.N = int(N)
        self.dtype = np.float64 if precision in ("fp64", MPCD_FP64) else np.float32
        opt = Options()
        self.lib.mpcd_default_options(C.byref(opt))
        opt.precision = MPCD_FP64 if self.dtype == np.float64 else MPCD_MIXED
        opt.rule = MPCD_AT if rule in ("at", MPCD_AT) else MPCD_SRD
        opt.dt, opt.alpha = float(dt), float(alpha)
        opt.sort_period, opt.cell_energy, opt.init_state = int(sort_period), int(bool(cell_energy)), int(bool(init_state))
        opt.thermostat = int(bool(thermostat))
        opt.deterministic = int(bool(deterministic))
        opt.brick = int(bool(brick))
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        opt.stream = C.c_void_p(self._stream.cuda_stream)
        self._alloc = TorchAllocator(device) if use_torch_allocator else None
        if self._alloc is not None:
            opt.alloc_fn, opt.free_fn = self._alloc.alloc_cb, self._alloc.free_cb
        self._opt = opt
        h = C.c_void_p()
        b = (C.c_double * 3)(*[float(x) for x in box])
        rc = self.lib.mpcd_create_ex(C.byref(h), b, self.N, float(a), float(m), float(kT), int(seed), C.byref(opt))
        if rc != MPCD_OK:
            raise MPCDError(rc, self.lib.mpcd_last_error(None).decode())
        self.h = h
        st = self.stats()
        self.Nc, self.n = st["Nc"], st["n"]

    def _check(self, rc):
        if rc != MPCD_OK:
            raise MPCDError(rc, self.lib.mpcd_last_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None):
            self.lib.mpcd_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the calls of include/mpcd.h --
    def stream(self):
        self._check(self.lib.mpcd_stream(self.h))

    def shift_and_bin(self):
        self._check(self.lib.mpcd_shift_and_bin(self.h))

    def collide_srd(self, alpha=math.radians(130.0)):
        self._check(self.lib.mpcd_collide_srd(self.h, float(alpha)))

    def collide_at(self):
        self._check(self.lib.mpcd_collide_at(self.h))

    def sort(self):
        self._check(self.lib.mpcd_sort(self.h))

    def step(self, nsteps=1):
        self._check(self.lib.mpcd_step(self.h, int(nsteps)))

    def get_state(self, pos=True, vel=True, tag=True, cell=True, out=None):
        """Returns dict(pos, vel, tag, cell, step) of host numpy arrays (or fills `out`, a dict of
        preallocated host arrays / pinned tensors)."""
        o = out if out is not None else {}
        if out is None:
            if pos: o["pos"] = np.empty((self.N, 4), dtype=self.dtype)
            if vel: o["vel"] = np.empty((self.N, 4), dtype=self.dtype)
            if tag: o["tag"] = np.empty(self.N, dtype=np.uint32)
            if cell: o["cell"] = np.empty(self.N, dtype=np.int32)
        step = C.c_uint64()
        self._check(self.lib.mpcd_get_state(self.h, _ptr(o.get("pos")), _ptr(o.get("vel")), _ptr(o.get("tag")), _ptr(o.get("cell")), C.byref(step)))
        o["step"] = int(step.value)
        return o

    def set_state(self, pos4, vel4, tag=None, step=0):
        if isinstance(pos4, np.ndarray):
            pos4 = np.ascontiguousarray(pos4, dtype=self.dtype)
            vel4 = np.ascontiguousarray(vel4, dtype=self.dtype)
            assert pos4.shape == (self.N, 4) and vel4.shape == (self.N, 4)
            if tag is not None:
                tag = np.ascontiguousarray(tag, dtype=np.uint32)
        self._check(self.lib.mpcd_set_state(self.h, _ptr(pos4), _ptr(vel4), _ptr(tag), int(step)))

    def get_cells(self, axis=True):
        Nc = self.Nc
        o = dict(count=np.empty(Nc, np.int32), sumv=np.empty((Nc, 3)), ke=np.empty(Nc), u=np.empty((Nc, 3)), kTc=np.empty(Nc))
        if axis:
            o["axis"] = np.empty((Nc, 3))
        self._check(self.lib.mpcd_get_cells(self.h, _ptr(o["count"]), _ptr(o["sumv"]), _ptr(o["ke"]), _ptr(o["u"]), _ptr(o.get("axis")), _ptr(o["kTc"])))
        return o

    def set_embedded(self, pos3, vel3, mass, chain_len, k, r0, md_substeps):
        pos3 = np.ascontiguousarray(pos3, dtype=np.float64); vel3 = np.ascontiguousarray(vel3, dtype=np.float64)
        mass = np.ascontiguousarray(mass, dtype=np.float64)
        assert pos3.shape == vel3.shape and pos3.shape[1] == 3 and mass.shape == (pos3.shape[0],)
        self.nb = pos3.shape[0]
        self._check(self.lib.mpcd_set_embedded(self.h, self.nb, _ptr(pos3), _ptr(vel3), _ptr(mass), int(chain_len), float(k), float(r0), int(md_substeps)))

    def get_embedded(self):
        o = dict(pos=np.empty((self.nb, 3)), vel=np.empty((self.nb, 3)), cell=np.empty(self.nb, np.int32))
        self._check(self.lib.mpcd_get_embedded(self.h, _ptr(o["pos"]), _ptr(o["vel"]), _ptr(o["cell"])))
        return o

    def get_xi(self):
        xi = np.empty(self.Nc)
        self._check(self.lib.mpcd_get_xi(self.h, _ptr(xi)))
        return xi

    def get_shift(self):
        s = (C.c_double * 3)()
        self._check(self.lib.mpcd_get_shift(self.h, s))
        return np.array(s[:])

    def get_thermo(self):
        P = (C.c_double * 3)()
        KE, kT = C.c_double(), C.c_double()
        self._check(self.lib.mpcd_get_thermo(self.h, P, C.byref(KE), C.byref(kT)))
        return np.array(P[:]), KE.value, kT.value

    def stats(self):
        s = Stats()
        self._check(self.lib.mpcd_get_stats(self.h, C.byref(s)))
        return dict(N=s.N, Nc=s.Nc, n=tuple(s.n), max_occupancy=s.max_occupancy, step=s.step,
                    kernel_launches=s.kernel_launches, sorts=s.sorts, device_bytes=s.device_bytes, brick=tuple(s.brick))

    def set_profiling(self, on=True):
        self._check(self.lib.mpcd_set_profiling(self.h, int(bool(on))))

    def get_profile(self):
        """{kind: (summed ms, launch groups)} since profiling was switched on."""
        ms = (C.c_double * len(PROF_KINDS))()
        n = (C.c_uint64 * len(PROF_KINDS))()
        self._check(self.lib.mpcd_get_profile(self.h, ms, n))
        return {k: (ms[i], int(n[i])) for i, k in enumerate(PROF_KINDS)}

    def synchronize(self):
        self._stream.synchronize()


def cell_sums_static(pos4, vel4, n, a, shift, m, count=None, sumv3=None, ke=None, stream=None):
    """mpcd_cell_sums_static of include/mpcd.h: per-cell count, sum of velocities and kinetic energy of the particles in
    the CUDA tensors pos4 / vel4 (N x 4, float32 = mixed model or float64), written into the caller's CUDA tensors
    count (int32, Nc), sumv3 (float64, Nc x 3), ke (float64, Nc); any of the three may be None.

    For callers that cannot allocate device memory where they need the sums (all of it belongs to another pool, or a
    cudaMalloc's device synchronisation is not affordable): the library allocates nothing in this call, its accumulators
    are a fixed 1.25 MiB array per GPU that holds at most STATIC_MAX_CELLS cells and that all calls on that GPU share.
    Keep the calls of one GPU on one stream; the work is enqueued on `stream` (default: torch's current stream) and not
    synchronised.  This wrapper allocates nothing on the device either: every tensor is the caller's."""
    import torch
    lib = load_library()
    assert pos4.is_cuda and vel4.is_cuda and pos4.is_contiguous() and vel4.is_contiguous()
    assert pos4.dtype == vel4.dtype and pos4.dtype in (torch.float32, torch.float64)
    assert pos4.dim() == 2 and pos4.shape[1] == 4 and vel4.shape == pos4.shape
    nn = (C.c_int32 * 3)(*[int(x) for x in n])
    Nc = int(n[0]) * int(n[1]) * int(n[2])
    for t, dt, numel in ((count, torch.int32, Nc), (sumv3, torch.float64, 3 * Nc), (ke, torch.float64, Nc)):
        assert t is None or (t.is_cuda and t.is_contiguous() and t.dtype == dt and t.numel() == numel and t.device == pos4.device)
    sh = (C.c_double * 3)(*[float(x) for x in shift])
    st = stream if stream is not None else torch.cuda.current_stream(pos4.device)
    dp = lambda t: None if t is None else C.c_void_p(t.data_ptr())
    with torch.cuda.device(pos4.device):
        rc = lib.mpcd_cell_sums_static(dp(pos4) if pos4.shape[0] else None, dp(vel4) if pos4.shape[0] else None, pos4.shape[0],
                                       MPCD_FP64 if pos4.dtype == torch.float64 else MPCD_MIXED, nn, float(a), sh, float(m),
                                       dp(count), dp(sumv3), dp(ke), C.c_void_p(st.cuda_stream))
    if rc != MPCD_OK:
        raise MPCDError(rc, lib.mpcd_cell_sums_static_error().decode())


def test_philox(ctr4, key2):
    """The CUDA library's Philox4x32-10 evaluated on the device (test hook)."""
    lib = load_library()
    ctr4 = np.ascontiguousarray(ctr4, dtype=np.uint32).reshape(-1, 4)
    key2 = np.ascontiguousarray(key2, dtype=np.uint32).reshape(-1, 2)
    out = np.empty_like(ctr4)
    rc = lib.mpcd_test_philox(_ptr(ctr4), _ptr(key2), _ptr(out), ctr4.shape[0])
    if rc != MPCD_OK:
        raise MPCDError(rc, "mpcd_test_philox failed")
    return out

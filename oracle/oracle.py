"""ctypes front end of the CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

The arithmetic lives in oracle/mpcd_oracle.c (+ mpcd_oracle_steps.inc), written from
PAPER.md.  This file only marshals numpy arrays and strings the steps together in
the paper's order (PAPER.md:70 and Fig. 1; SURVEY.md 8c reading A3):

    stream -> shift + bin -> [sort, every sort_period steps] -> cell properties
           -> axis draw -> collide (SRD eq. 2 / AT eq. 4) -> step += 1

It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

from . import build as _build

_LIB = None


def lib():
    global _LIB
    if _LIB is None:
        _LIB = C.CDLL(_build.build())
        _LIB.oracle_u01_32.restype = C.c_double
        _LIB.oracle_u01_32.argtypes = [C.c_uint32]
        _LIB.oracle_u01_53.restype = C.c_double
        _LIB.oracle_u01_53.argtypes = [C.c_uint32, C.c_uint32]
    return _LIB


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _d3(x):
    return (C.c_double * 3)(*[float(v) for v in x])


def _i3(x):
    return (C.c_int32 * 3)(*[int(v) for v in x])


def philox4x32_10(ctr, key):
    """Philox4x32-10 block: ctr = 4 words, key = 2 words -> 4 words."""
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def u01_32(b):
    return lib().oracle_u01_32(C.c_uint32(int(b)))


def u01_53(lo, hi):
    return lib().oracle_u01_53(C.c_uint32(int(lo)), C.c_uint32(int(hi)))


def draw_shift(seed, step, a):
    """a2: the step's grid shift, in double."""
    s = (C.c_double * 3)()
    lib().oracle_shift(C.c_uint64(seed), C.c_uint64(step), C.c_double(a), s)
    return np.array([s[0], s[1], s[2]], dtype=np.float64)


def draw_axis(seed, step, Nc):
    """a5: per-cell random unit axis."""
    ax = np.empty((Nc, 3), dtype=np.float64)
    lib().oracle_axis(C.c_uint64(seed), C.c_uint64(step), C.c_int64(Nc), _p(ax))
    return ax


def at_draw(seed, step, tag, sigma):
    """a7: per-particle Gaussian velocities keyed by tag."""
    tag = np.ascontiguousarray(tag, dtype=np.uint32)
    dv = np.empty((tag.shape[0], 3), dtype=np.float64)
    lib().oracle_at_draw(C.c_uint64(seed), C.c_uint64(step), C.c_int64(tag.shape[0]), _p(tag), C.c_double(sigma), _p(dv))
    return dv


def _suf(dtype):
    dtype = np.dtype(dtype)
    if dtype == np.float32:
        return "_f32"
    if dtype == np.float64:
        return "_f64"
    raise TypeError("native precision must be float32 (mixed model) or float64")


def stream(pos4, vel4, dt, L):
    """a1: eq. (1) + periodic wrap, in place on pos4 (N x 4, native precision)."""
    assert pos4.dtype == vel4.dtype and pos4.flags.c_contiguous and vel4.flags.c_contiguous
    getattr(lib(), "oracle_stream" + _suf(pos4.dtype))(C.c_int64(pos4.shape[0]), _p(pos4), _p(vel4), C.c_double(dt), _d3(L))


def bin_cells(pos4, shift, a, n):
    """a3: cell index of every particle for the given shift."""
    cell = np.empty(pos4.shape[0], dtype=np.int32)
    getattr(lib(), "oracle_bin" + _suf(pos4.dtype))(C.c_int64(pos4.shape[0]), _p(pos4), _d3(shift), C.c_double(a), _i3(n), _p(cell))
    return cell


def reduce_cells(vel4, cell, Nc, m):
    """a4: per-cell count, sum of velocities, kinetic energy."""
    count = np.empty(Nc, dtype=np.int32)
    sumv = np.empty((Nc, 3), dtype=np.float64)
    ke = np.empty(Nc, dtype=np.float64)
    getattr(lib(), "oracle_reduce" + _suf(vel4.dtype))(C.c_int64(vel4.shape[0]), _p(vel4), _p(cell), C.c_int64(Nc), C.c_double(m), _p(count), _p(sumv), _p(ke))
    return count, sumv, ke


def finalize_cells(vel4, cell, Nc, m, count, sumv):
    """a5: u, E_rel (eq. 3), kT_c."""
    u = np.empty((Nc, 3), dtype=np.float64)
    erel = np.empty(Nc, dtype=np.float64)
    kTc = np.empty(Nc, dtype=np.float64)
    getattr(lib(), "oracle_finalize" + _suf(vel4.dtype))(C.c_int64(vel4.shape[0]), _p(vel4), _p(cell), C.c_int64(Nc), C.c_double(m), _p(count), _p(sumv), _p(u), _p(erel), _p(kTc))
    return u, erel, kTc


def collide_srd(vel4, cell, u, axis, alpha):
    """a6: Algorithm 1, in place on vel4.  cos/sin of alpha by libm in double (reading A15)."""
    getattr(lib(), "oracle_collide_srd" + _suf(vel4.dtype))(C.c_int64(vel4.shape[0]), _p(vel4), _p(cell), _p(u), _p(axis), C.c_double(math.cos(alpha)), C.c_double(math.sin(alpha)))


def thermostat_xi(seed, step, kT, count, erel):
    """NEXT-2: Maxwell-Boltzmann cell thermostat: (E^ per cell, xi per cell)."""
    Nc = count.shape[0]
    ehat, xi = np.empty(Nc), np.empty(Nc)
    lib().oracle_thermostat_xi(C.c_uint64(seed), C.c_uint64(step), C.c_int64(Nc), C.c_double(kT),
                               _p(np.ascontiguousarray(count, dtype=np.int32)), _p(np.ascontiguousarray(erel, dtype=np.float64)),
                               _p(ehat), _p(xi))
    return ehat, xi


def collide_srd_xi(vel4, cell, u, axis, xi, alpha):
    """a6 + Alg. 1 lines 8-10: SRD rotation with the relative velocities scaled by the cell's xi."""
    getattr(lib(), "oracle_collide_srd_xi" + _suf(vel4.dtype))(
        C.c_int64(vel4.shape[0]), _p(vel4), _p(cell), _p(u), _p(axis), _p(np.ascontiguousarray(xi, dtype=np.float64)),
        C.c_double(math.cos(alpha)), C.c_double(math.sin(alpha)))


def md_forces(pos3, chain_len, k, r0, L):
    """NEXT-1: harmonic bond forces on the beads of linear chains (minimum image)."""
    f = np.empty_like(pos3)
    lib().oracle_md_forces(C.c_int64(pos3.shape[0]), C.c_int32(chain_len), _p(pos3), C.c_double(k), C.c_double(r0), _d3(L), _p(f))
    return f


def md_verlet(pos3, vel3, mass, chain_len, k, r0, L, dt, nsub):
    """NEXT-1: nsub velocity-Verlet steps of the beads, in place."""
    assert pos3.dtype == np.float64 and vel3.dtype == np.float64 and mass.dtype == np.float64
    lib().oracle_md_verlet(C.c_int64(pos3.shape[0]), C.c_int32(chain_len), _p(pos3), _p(vel3), _p(mass), C.c_double(k), C.c_double(r0),
                           _d3(L), C.c_double(dt), C.c_int32(nsub))


def embedded_means(m, count, sumv, cell_b, vel3_b, mass_b):
    """NEXT-1: mass-weighted cell mean velocity and cell mass with embedded beads."""
    Nc = count.shape[0]
    u, Mc = np.empty((Nc, 3)), np.empty(Nc)
    lib().oracle_embedded_means(C.c_int64(Nc), C.c_double(m), _p(count), _p(sumv), C.c_int64(cell_b.shape[0]), _p(cell_b), _p(vel3_b),
                                _p(mass_b), _p(u), _p(Mc))
    return u, Mc


def collide_srd_beads(vel3, cell_b, u, axis, alpha):
    lib().oracle_collide_srd_beads(C.c_int64(vel3.shape[0]), _p(vel3), _p(cell_b), _p(u), _p(axis), C.c_double(math.cos(alpha)),
                                   C.c_double(math.sin(alpha)))


def collide_srd_beads_xi(vel3, cell_b, u, axis, xi, alpha):
    lib().oracle_collide_srd_beads_xi(C.c_int64(vel3.shape[0]), _p(vel3), _p(cell_b), _p(u), _p(axis), _p(np.ascontiguousarray(xi, dtype=np.float64)),
                                      C.c_double(math.cos(alpha)), C.c_double(math.sin(alpha)))


def erel_with_beads(vel4, cell, m, count, u, cell_b, vel3_b, mass_b):
    """NEXT-1 + NEXT-2 (reading A28): relative kinetic energy of every cell over solvent AND beads about the mass-weighted
    mean u, and the number of particles of the cell (solvent + beads)."""
    Nc = count.shape[0]
    erel, ntot = np.empty(Nc), np.empty(Nc, dtype=np.int32)
    getattr(lib(), "oracle_erel_about" + _suf(vel4.dtype))(C.c_int64(vel4.shape[0]), _p(vel4), _p(cell), C.c_int64(Nc), C.c_double(m), _p(u), _p(erel))
    lib().oracle_embedded_energy(C.c_int64(Nc), _p(count), C.c_int64(cell_b.shape[0]), _p(cell_b), _p(vel3_b), _p(mass_b), _p(u), _p(erel), _p(ntot))
    return erel, ntot


def collide_at(vel4, cell, Nc, count, u, dv):
    """a7: eq. (4), in place on vel4."""
    getattr(lib(), "oracle_collide_at" + _suf(vel4.dtype))(C.c_int64(vel4.shape[0]), _p(vel4), _p(cell), C.c_int64(Nc), _p(count), _p(u), _p(dv))


def sort_perm(cell, Nc):
    """a8: stable permutation into cell order; perm[k] = old index."""
    perm = np.empty(cell.shape[0], dtype=np.int64)
    lib().oracle_sort_perm(C.c_int64(cell.shape[0]), _p(cell), C.c_int64(Nc), _p(perm))
    return perm


def permute(perm, pos4, vel4, tag, cell):
    out = (np.empty_like(pos4), np.empty_like(vel4), np.empty_like(tag), np.empty_like(cell))
    getattr(lib(), "oracle_permute" + _suf(pos4.dtype))(C.c_int64(pos4.shape[0]), _p(perm), _p(pos4), _p(vel4), _p(tag), _p(cell), _p(out[0]), _p(out[1]), _p(out[2]), _p(out[3]))
    return out


def thermo(m, count, sumv, ke, erel):
    """a9: {P (3), KE, pooled kT} from the cell arrays."""
    out = (C.c_double * 5)()
    lib().oracle_thermo(C.c_int64(count.shape[0]), C.c_double(m), _p(count), _p(sumv), _p(ke), _p(erel), out)
    return np.array(out[0:3]), out[3], out[4]


def init_state(seed, N, L, sigma, dtype):
    """Initial condition (reading A23)."""
    pos4 = np.empty((N, 4), dtype=dtype)
    vel4 = np.empty((N, 4), dtype=dtype)
    tag = np.empty(N, dtype=np.uint32)
    getattr(lib(), "oracle_init" + _suf(dtype))(C.c_uint64(seed), C.c_int64(N), _d3(L), C.c_double(sigma), _p(pos4), _p(vel4), _p(tag))
    return pos4, vel4, tag


class OracleMPCD:
    """State + one-step driver in the paper's order.  Mirrors the C-ABI's semantics
    (include/mpcd.h) without sharing any code with it."""

    SRD, AT = 0, 1

    def __init__(self, box, N, a=1.0, m=1.0, kT=1.0, seed=0, *, dtype=np.float32, dt=0.1,
                 alpha=math.radians(130.0), rule=0, sort_period=25, init=True, thermostat=False):
        self.a, self.m, self.kT, self.seed = float(a), float(m), float(kT), int(seed)
        self.n = [int(round(b / a)) for b in box]
        for b, n in zip(box, self.n):
            assert n >= 1 and abs(b / a - n) <= 1e-9, "box must be an integer multiple of a"
        self.L = [float(b) for b in box]
        self.Nc = self.n[0] * self.n[1] * self.n[2]
        self.N = int(N)
        self.dtype = np.dtype(dtype)
        self.dt, self.alpha, self.rule, self.sort_period = float(dt), float(alpha), int(rule), int(sort_period)
        self.thermostat = bool(thermostat)
        self.ehat = self.xi = None
        self.emb = None          # embedded beads (NEXT-1): dict(pos, vel, mass, chain_len, k, r0, nsub, cell)
        self.sigma = math.sqrt(self.kT / self.m)
        self.step_count = 0
        if init:
            self.pos, self.vel, self.tag = init_state(self.seed, self.N, self.L, self.sigma, self.dtype)
        else:
            self.pos = np.zeros((self.N, 4), dtype=self.dtype)
            self.vel = np.zeros((self.N, 4), dtype=self.dtype)
            self.tag = np.arange(self.N, dtype=np.uint32)
        self.cell = np.zeros(self.N, dtype=np.int32)
        self.shift = np.zeros(3)
        self.count = self.sumv = self.ke = self.u = self.erel = self.kTc = self.axis = None

    def set_state(self, pos4, vel4, tag=None, step=0):
        self.pos = np.ascontiguousarray(pos4, dtype=self.dtype).copy()
        self.vel = np.ascontiguousarray(vel4, dtype=self.dtype).copy()
        self.tag = np.arange(self.N, dtype=np.uint32) if tag is None else np.ascontiguousarray(tag, dtype=np.uint32).copy()
        self.step_count = int(step)

    def set_embedded(self, pos3, vel3, mass, chain_len, k, r0, md_substeps):
        """NEXT-1 (BASELINE config 5): beads of linear harmonic chains that join the SRD collision and
        move by md_substeps velocity-Verlet steps per collision step.  Beads are kept in double (A27)."""
        assert self.rule == self.SRD
        self.emb = dict(pos=np.ascontiguousarray(pos3, dtype=np.float64).copy(), vel=np.ascontiguousarray(vel3, dtype=np.float64).copy(),
                        mass=np.ascontiguousarray(mass, dtype=np.float64).copy(), chain_len=int(chain_len), k=float(k), r0=float(r0),
                        nsub=int(md_substeps), cell=None)

    def _bin_embedded(self):
        e = self.emb
        p4 = np.zeros((e["pos"].shape[0], 4)); p4[:, :3] = e["pos"]
        shift_used = self.shift.astype(self.dtype).astype(np.float64)        # the shift as the solvent's binning applies it (A5)
        e["cell"] = bin_cells(p4, shift_used, self.a, self.n)

    # -- the blocks of Fig. 1 --
    def stream(self):
        assert float(np.abs(self.vel[:, :3]).max(initial=0.0)) * self.dt < min(self.L), "single-image wrap (A7)"
        stream(self.pos, self.vel, self.dt, self.L)
        if self.emb is not None:     # the solute moves by MD over the same interval
            e = self.emb
            md_verlet(e["pos"], e["vel"], e["mass"], e["chain_len"], e["k"], e["r0"], self.L, self.dt / e["nsub"], e["nsub"])

    def shift_and_bin(self):
        t = self.step_count
        self.shift = draw_shift(self.seed, t, self.a)
        self.cell = bin_cells(self.pos, self.shift, self.a, self.n)
        self._cell_properties()

    def _cell_properties(self):
        self.count, self.sumv, self.ke = reduce_cells(self.vel, self.cell, self.Nc, self.m)
        self.u, self.erel, self.kTc = finalize_cells(self.vel, self.cell, self.Nc, self.m, self.count, self.sumv)
        self.axis = draw_axis(self.seed, self.step_count, self.Nc)
        if self.emb is not None:
            self._bin_embedded()
            self.u, self.Mc = embedded_means(self.m, self.count, self.sumv, self.emb["cell"], self.emb["vel"], self.emb["mass"])
        if self.thermostat:      # "we compute xi for each cell at the same time that we draw the rotation vectors"
            if self.emb is not None:         # the cell's particles are solvent AND beads (reading A28)
                self.erel_tot, self.ntot = erel_with_beads(self.vel, self.cell, self.m, self.count, self.u, self.emb["cell"], self.emb["vel"], self.emb["mass"])
                self.ehat, self.xi = thermostat_xi(self.seed, self.step_count, self.kT, self.ntot, self.erel_tot)
            else:
                self.ehat, self.xi = thermostat_xi(self.seed, self.step_count, self.kT, self.count, self.erel)

    def sort(self):
        perm = sort_perm(self.cell, self.Nc)
        self.pos, self.vel, self.tag, self.cell = permute(perm, self.pos, self.vel, self.tag, self.cell)
        return perm

    def collide_srd(self, alpha=None):
        alpha = self.alpha if alpha is None else alpha
        if self.emb is not None:
            if self.thermostat:
                collide_srd_beads_xi(self.emb["vel"], self.emb["cell"], self.u, self.axis, self.xi, alpha)
            else:
                collide_srd_beads(self.emb["vel"], self.emb["cell"], self.u, self.axis, alpha)
        if self.thermostat:
            collide_srd_xi(self.vel, self.cell, self.u, self.axis, self.xi, alpha)
        else:
            collide_srd(self.vel, self.cell, self.u, self.axis, alpha)

    def collide_at(self):
        dv = at_draw(self.seed, self.step_count, self.tag, self.sigma)
        collide_at(self.vel, self.cell, self.Nc, self.count, self.u, dv)

    def step(self, nsteps=1):
        for _ in range(nsteps):
            t = self.step_count
            self.stream()
            self.shift = draw_shift(self.seed, t, self.a)
            self.cell = bin_cells(self.pos, self.shift, self.a, self.n)
            if self.sort_period > 0 and t % self.sort_period == 0:
                self.sort()
            self._cell_properties()
            if self.rule == self.SRD:
                self.collide_srd()
            else:
                self.collide_at()
            self.step_count = t + 1

    def thermo(self):
        """Thermo of the *current* velocities under the last binning."""
        count, sumv, ke = reduce_cells(self.vel, self.cell, self.Nc, self.m)
        u, erel, _ = finalize_cells(self.vel, self.cell, self.Nc, self.m, count, sumv)
        return thermo(self.m, count, sumv, ke, erel)

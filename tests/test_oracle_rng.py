"""Pins for the oracle's random numbers: Philox4x32-10 block function,
uniform conversions, grid shift, per-cell axis, AT Gaussians.  CPU only."""
import ctypes as C
import json
import math
import os
import subprocess
import sysconfig

import numpy as np
import pytest
from scipy import stats

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def libs(tmp_path_factory):
    """Two independent library Philox implementations compiled from vendor headers."""
    import torch
    out = str(tmp_path_factory.mktemp("philox") / "philox_libs.so")
    tinc = os.path.join(os.path.dirname(torch.__file__), "include")
    cmd = ["g++", "-O1", "-std=c++17", "-fPIC", "-shared", "-I" + tinc, "-I/usr/local/cuda/include",
           "-DWITH_CURAND_HOST", "-o", out, os.path.join(HERE, "helpers", "philox_libs.cpp")]
    subprocess.run(cmd, check=True)
    return C.CDLL(out)


def _call(fn, ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    fn(c, k, o)
    return [int(v) for v in o]


def test_philox_known_answer_vectors(oracle):
    kat = json.load(open(os.path.join(HERE, "golden", "philox_kat.json")))
    for v in kat["vectors"]:
        ctr = [int(x, 16) for x in v["ctr"]]
        key = [int(x, 16) for x in v["key"]]
        assert oracle.philox4x32_10(ctr, key) == [int(x, 16) for x in v["out"]]


def test_philox_matches_aten_and_curand(oracle, libs):
    rng = np.random.default_rng(7)
    cases = [([0, 0, 0, 0], [0, 0]), ([0xFFFFFFFF] * 4, [0xFFFFFFFF] * 2), ([1, 0, 0, 0], [0, 0]), ([0, 0, 0, 1], [0, 1])]
    for _ in range(2000):
        w = rng.integers(0, 2**32, size=6, dtype=np.uint64)
        cases.append(([int(x) for x in w[:4]], [int(x) for x in w[4:]]))
    for ctr, key in cases:
        mine = oracle.philox4x32_10(ctr, key)
        assert mine == _call(libs.aten_philox4x32_10, ctr, key)
        assert mine == _call(libs.curand_host_philox4x32_10, ctr, key)


def test_kat_vectors_hold_for_library_implementations(libs):
    kat = json.load(open(os.path.join(HERE, "golden", "philox_kat.json")))
    for v in kat["vectors"]:
        ctr = [int(x, 16) for x in v["ctr"]]
        key = [int(x, 16) for x in v["key"]]
        want = [int(x, 16) for x in v["out"]]
        assert _call(libs.aten_philox4x32_10, ctr, key) == want
        assert _call(libs.curand_host_philox4x32_10, ctr, key) == want


def test_uniform_conversions_are_exact(oracle):
    from fractions import Fraction
    # (b + 1/2) 2^-32: exactly representable, strictly inside (0, 1)
    for b in (0, 1, 2**31, 2**32 - 2, 2**32 - 1, 123456789):
        u = oracle.u01_32(b)
        assert Fraction(u) == (Fraction(b) + Fraction(1, 2)) / 2**32
    assert oracle.u01_32(0) == 2.0**-33 and oracle.u01_32(2**32 - 1) == 1 - 2.0**-33
    # 53-bit form: ((lo | hi << 32) >> 11) 2^-53 in [0, 1)
    for lo, hi in ((0, 0), (0xFFFFFFFF, 0xFFFFFFFF), (0x7FF, 0), (0x800, 0), (0xDEADBEEF, 0x12345678)):
        u = oracle.u01_53(lo, hi)
        assert Fraction(u) == Fraction(((hi << 32) | lo) >> 11, 2**53)
    assert oracle.u01_53(0xFFFFFFFF, 0xFFFFFFFF) == 1 - 2.0**-53 and oracle.u01_53(0x7FF, 0) == 0.0


def test_shift_is_uniform_in_open_half_cell(oracle):
    a = 1.7
    s = np.array([oracle.draw_shift(99, t, a) for t in range(6000)])
    assert np.all(np.abs(s) < a / 2)                       # open interval (A4)
    for d in range(3):
        assert stats.kstest(s[:, d] / a + 0.5, "uniform").pvalue > 1e-3
    assert abs(np.corrcoef(s[:, 0], s[:, 1])[0, 1]) < 0.05
    # keyed by (seed, step) only: repeatable, and different for another seed / step
    assert np.array_equal(oracle.draw_shift(99, 17, a), s[17])
    assert not np.array_equal(oracle.draw_shift(98, 17, a), s[17])
    # the draw is Philox(seed, (0, t, 0, SHIFT=1)) words 0..2 through u01_32 (A24)
    b = oracle.philox4x32_10([0, 17, 0, 1], [99, 0])
    assert np.array_equal(s[17], [(oracle.u01_32(b[d]) - 0.5) * a for d in range(3)])


def test_axis_is_unit_and_uniform_on_sphere(oracle):
    Nc = 400_000
    ax = oracle.draw_axis(5, 3, Nc)
    assert np.max(np.abs((ax**2).sum(axis=1) - 1)) <= 1e-15    # a handful of 1.1e-16 roundings
    assert np.all(np.abs(ax.mean(axis=0)) < 3 / math.sqrt(Nc))
    second = ax.T @ ax / Nc
    assert np.max(np.abs(second - np.eye(3) / 3)) < 3 / math.sqrt(Nc)
    # Archimedes' hat-box: z uniform on [-1, 1) and azimuth uniform <=> uniform on the sphere
    assert stats.kstest((ax[:, 2] + 1) / 2, "uniform").pvalue > 1e-3
    phi = np.mod(np.arctan2(ax[:, 1], ax[:, 0]), 2 * np.pi) / (2 * np.pi)
    assert stats.kstest(phi, "uniform").pvalue > 1e-3
    # A13: words (0,1) -> z, words (2,3) -> phi
    b = oracle.philox4x32_10([1234, 3, 0, 2], [5, 0])
    z = 2 * oracle.u01_53(b[0], b[1]) - 1
    ph = 2 * math.pi * oracle.u01_53(b[2], b[3])
    assert ax[1234, 2] == z
    np.testing.assert_allclose(ax[1234, :2], [math.sqrt(1 - z * z) * math.cos(ph), math.sqrt(1 - z * z) * math.sin(ph)], rtol=0, atol=4e-16)


def test_axis_depends_only_on_seed_step_cell(oracle):
    """any cell's vector can be reproduced at any step regardless of history."""
    big = oracle.draw_axis(11, 40, 5000)
    small = oracle.draw_axis(11, 40, 100)
    assert np.array_equal(big[:100], small)
    assert not np.array_equal(oracle.draw_axis(11, 41, 100), small)
    assert not np.array_equal(oracle.draw_axis(12, 40, 100), small)
    # 64-bit step counter: high word participates
    assert not np.array_equal(oracle.draw_axis(11, 40 + 2**32, 100), small)


def test_at_gaussians(oracle):
    N = 300_000
    tag = np.arange(N, dtype=np.uint32)
    sigma = 1.3
    dv = oracle.at_draw(21, 9, tag, sigma)
    for d in range(3):
        assert stats.kstest(dv[:, d] / sigma, "norm").pvalue > 1e-3
    np.testing.assert_allclose(dv.var(axis=0), sigma**2, rtol=4 * math.sqrt(2 / N))
    c = np.corrcoef(dv.T)
    assert np.max(np.abs(c - np.eye(3))) < 5 / math.sqrt(N)
    # keyed by tag (A18): a permuted tag array gives permuted draws
    perm = np.random.default_rng(0).permutation(N)
    assert np.array_equal(oracle.at_draw(21, 9, tag[perm], sigma), dv[perm])
    # Box-Muller (A17) on the four words of Philox(seed, (tag, t, 0, AT=3))
    b = oracle.philox4x32_10([777, 9, 0, 3], [21, 0])
    U = [oracle.u01_32(x) for x in b]
    want = [sigma * math.sqrt(-2 * math.log(U[0])) * math.cos(2 * math.pi * U[1]),
            sigma * math.sqrt(-2 * math.log(U[0])) * math.sin(2 * math.pi * U[1]),
            sigma * math.sqrt(-2 * math.log(U[2])) * math.cos(2 * math.pi * U[3])]
    np.testing.assert_allclose(dv[777], want, rtol=1e-14)

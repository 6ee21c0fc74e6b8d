"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol
include/mpcd.h declares; argument validation happens before any device work; without a device
the library refuses to compute (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1801_10187_b200 import build
    build.build()
    from paper_1801_10187_b200 import binding
    return binding.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "mpcd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mpcd_[a-z_0-9]+)\s*\(", text)) - {"mpcd_alloc_fn", "mpcd_free_fn"})


def test_library_exports_every_declared_symbol(lib):
    from paper_1801_10187_b200 import binding
    declared = _declared_symbols()
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/mpcd.h but not exported"
    assert sorted(binding.EXPORTS) == declared


def test_north_star_entry_points_present(lib):
    for name in ("mpcd_create", "mpcd_stream", "mpcd_shift_and_bin", "mpcd_collide_srd", "mpcd_collide_at",
                 "mpcd_sort", "mpcd_step", "mpcd_get_state"):
        assert hasattr(lib, name)


def test_abi_version_and_defaults(lib):
    from paper_1801_10187_b200.binding import Options
    assert lib.mpcd_abi_version() == 3
    assert b"sm_100a" in lib.mpcd_build_info()
    o = Options()
    assert lib.mpcd_default_options(C.byref(o)) == 0
    assert o.precision == 0 and o.rule == 0 and o.sort_period == 25 and o.cell_energy == 1 and o.brick == 0
    assert abs(o.dt - 0.1) < 1e-15 and abs(o.alpha - 130 * 3.141592653589793 / 180) < 1e-15
    assert lib.mpcd_default_options(None) == -1


def test_argument_validation_and_no_cpu_fallback(lib):
    import torch
    h = C.c_void_p()
    box = (C.c_double * 3)(8, 8, 8)
    bad_box = (C.c_double * 3)(8, 8.5, 8)
    assert lib.mpcd_create(None, box, 10, 1.0, 1.0, 1.0, 1) == -1
    assert lib.mpcd_create(C.byref(h), box, 0, 1.0, 1.0, 1.0, 1) == -1
    assert lib.mpcd_create(C.byref(h), box, 2**31, 1.0, 1.0, 1.0, 1) == -1
    assert lib.mpcd_create(C.byref(h), box, 10, -1.0, 1.0, 1.0, 1) == -1
    assert lib.mpcd_create(C.byref(h), bad_box, 10, 1.0, 1.0, 1.0, 1) == -1
    assert b"multiple" in lib.mpcd_last_error(None)
    assert h.value is None
    for fn in (lib.mpcd_stream, lib.mpcd_shift_and_bin, lib.mpcd_collide_at, lib.mpcd_sort, lib.mpcd_destroy):
        assert fn(None) == -1
    assert lib.mpcd_step(None, 1) == -1 and lib.mpcd_collide_srd(None, 1.0) == -1
    if not torch.cuda.is_available():
        assert lib.mpcd_create(C.byref(h), box, 10, 1.0, 1.0, 1.0, 1) == -3        # MPCD_ECUDA
        assert b"no CPU fallback" in lib.mpcd_last_error(None)
        from paper_1801_10187_b200 import MPCD
        with pytest.raises(RuntimeError):
            MPCD([8, 8, 8], 2560)


def test_product_does_not_import_the_oracle():
    """The CUDA package never imports, links or reads anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1801_10187_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "oracle/" not in src.replace("shares nothing with oracle/", ""), f


def test_static_cell_sums_validate_before_any_device_work(lib):
    """mpcd_cell_sums_static (the no-allocation entry point): size and argument errors are reported on a box without a
    GPU too, the limit is named in the message, and without a device a valid call fails loudly instead of computing."""
    import torch
    n_ok = (C.c_int32 * 3)(8, 8, 8)
    n_big = (C.c_int32 * 3)(32, 32, 33)
    n_huge = (C.c_int32 * 3)(2**31 - 1, 2**31 - 1, 2**31 - 1)
    s = (C.c_double * 3)(0.1, -0.2, 0.3)
    s_bad = (C.c_double * 3)(0.1, 1.0, 0.3)
    f = lib.mpcd_cell_sums_static
    err = lib.mpcd_cell_sums_static_error
    assert f(None, None, 0, 0, n_big, 1.0, s, 1.0, None, None, None, None) == -1
    assert b"32768" in err() and b"MPCD_STATIC_MAX_CELLS" in err()
    assert f(None, None, 0, 0, n_huge, 1.0, s, 1.0, None, None, None, None) == -1
    assert f(None, None, 5, 0, n_ok, 1.0, s, 1.0, None, None, None, None) == -1          # N > 0 without particle arrays
    assert f(None, None, -1, 0, n_ok, 1.0, s, 1.0, None, None, None, None) == -1
    assert f(None, None, 0, 2, n_ok, 1.0, s, 1.0, None, None, None, None) == -1          # precision
    assert f(None, None, 0, 0, n_ok, 0.0, s, 1.0, None, None, None, None) == -1
    assert f(None, None, 0, 0, n_ok, 1.0, s_bad, 1.0, None, None, None, None) == -1
    assert f(None, None, 0, 0, None, 1.0, s, 1.0, None, None, None, None) == -1
    if not torch.cuda.is_available():
        assert f(None, None, 0, 0, n_ok, 1.0, s, 1.0, None, None, None, None) == -3      # MPCD_ECUDA
        assert b"no CPU fallback" in err()

"""CPU checks of the boundary: the C-ABI library builds, loads without a GPU and exports every
function include/fe.h declares; the binding's struct layouts match the header."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2605_28800_b200 import build
    return ctypes.CDLL(build.build_lib())


def _declared():
    src = open(os.path.join(ROOT, "include", "fe.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fe_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = _declared()
    for need in ("fe_create_grid", "fe_set_material", "fe_precompute_tensor", "fe_rhs", "fe_step", "fe_energy"):
        assert need in names


def test_library_exports_every_declared_symbol(lib):
    names = _declared()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), n


def test_binding_lists_the_same_symbols():
    from paper_2605_28800_b200 import binding
    assert sorted(binding.SYMBOLS) == _declared()


def test_struct_sizes_match_the_header_layout():
    from paper_2605_28800_b200 import binding
    # fe_grid_desc: 3 int32 (+4 pad) + 3 double + 3+3+4 int32 = 16 + 24 + 40 = 80
    assert ctypes.sizeof(binding.fe_grid_desc) == 80
    assert ctypes.sizeof(binding.fe_landau) == 12 * 8 + 8
    assert ctypes.sizeof(binding.fe_global) == 7 * 8


def test_version_and_error_strings_without_gpu(lib):
    lib.fe_version.restype = ctypes.c_char_p
    lib.fe_last_error.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.fe_version()
    assert isinstance(lib.fe_last_error(), bytes)
    # argument validation happens before any CUDA call
    from paper_2605_28800_b200 import binding
    d = binding.fe_grid_desc()
    d.nx, d.ny, d.nz = 12, 16, 8          # 12 is not a power of two: refused on a periodic axis
    d.periodic[0] = 1
    d.dx = d.dy = d.dz = 1.0
    d.batch, d.n_materials = 1, 1
    h = ctypes.c_void_p()
    lib.fe_create_grid.argtypes = [ctypes.POINTER(binding.fe_grid_desc), ctypes.POINTER(ctypes.c_void_p)]
    assert lib.fe_create_grid(ctypes.byref(d), ctypes.byref(h)) == binding.FE_EINVAL
    assert b"power of two" in lib.fe_last_error()
    d.nx = 16
    d.dx = -1.0
    assert lib.fe_create_grid(ctypes.byref(d), ctypes.byref(h)) == binding.FE_EINVAL

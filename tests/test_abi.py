"""Host-side checks of the C-ABI library that need no GPU (-m "not gpu")."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_0908_4362_b200 import build
    build.build()
    from paper_0908_4362_b200 import binding as b
    return b


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "mhd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mhd_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(binding):
    names = _declared_symbols()
    assert len(names) >= 18
    lib = ctypes.CDLL(binding.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"libmhd.so does not export {n}"
    assert set(names) == set(binding.SIGNATURES), "binding and header disagree"


def test_binding_has_same_names(binding):
    for n in _declared_symbols():
        assert callable(getattr(binding, n))
    assert b"sm_100a" in binding.mhd_version()


def test_argument_validation_without_a_device(binding):
    b = binding
    h = ctypes.c_void_p()
    assert b.mhd_create(0, 4, 4, 1.4, b.MHD_F32, 0, ctypes.byref(h)) == b.MHD_EINVAL
    assert b"extents" in b.mhd_last_error(None)
    assert b.mhd_create(4, 4, 4, 1.0, b.MHD_F32, 0, ctypes.byref(h)) == b.MHD_EINVAL
    assert b.mhd_create(4, 4, 4, 1.4, 7, 0, ctypes.byref(h)) == b.MHD_EINVAL
    assert b.mhd_create(4, 4, 4, 1.4, b.MHD_F64, 9, ctypes.byref(h)) == b.MHD_EINVAL
    assert b.mhd_create(4, 4, 4, 1.4, b.MHD_F64, 0, None) == b.MHD_EINVAL
    assert b.mhd_create(16, 8, 4, 5 / 3, b.MHD_F64, b.MHD_BC_OUTFLOW, ctypes.byref(h)) == b.MHD_OK
    # stepping before a state exists must fail without touching the device
    assert b.mhd_step(h, 1, 0.8, None) == b.MHD_ENOSTATE
    assert b.mhd_step_fixed(h, 1, 0.1) == b.MHD_ENOSTATE
    assert b.mhd_apply(h, b.MHD_OP_FLUID, 0, 0, 0.1) == b.MHD_ENOSTATE
    dt = ctypes.c_double()
    assert b.mhd_cfl_dt(h, 0.8, ctypes.byref(dt), None) == b.MHD_ENOSTATE
    assert b.mhd_cfl_dt(h, -1.0, ctypes.byref(dt), None) == b.MHD_EINVAL
    assert b.mhd_step(h, -1, 0.8, None) == b.MHD_EINVAL
    assert b.mhd_set_option(h, b"nonsense", 1) == b.MHD_EINVAL
    assert b.mhd_set_option(h, b"segment", 64) == b.MHD_OK
    s = ctypes.c_longlong()
    assert b.mhd_set_step_index(h, 5) == b.MHD_OK and b.mhd_get_step_index(h, ctypes.byref(s)) == b.MHD_OK and s.value == 5
    assert b.mhd_launch_count(h) == 0
    assert b.mhd_destroy(h) == b.MHD_OK
    assert b.mhd_destroy(None) == b.MHD_OK


def test_workspace_bytes(binding):
    b = binding
    assert b.mhd_workspace_bytes(0, 1, 1, 0) == 0
    assert b.mhd_workspace_bytes(4, 4, 4, 5) == 0
    n = 512 ** 3
    assert b.mhd_workspace_bytes(512, 512, 512, b.MHD_F32) == 16 * n * 4 + 1024
    assert b.mhd_workspace_bytes(512, 512, 512, b.MHD_F64) == 16 * n * 8 + 1024
    # fields are padded to 256 bytes
    assert b.mhd_workspace_bytes(3, 1, 1, b.MHD_F32) == 16 * 256 + 1024


def test_product_does_not_import_the_oracle():
    """the CUDA path and its binding must never route through oracle/ (no CPU fallback)"""
    pkg = os.path.join(ROOT, "paper_0908_4362_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), fn
                assert "mhd_oracle" not in text and "mhdo_" not in text, fn
    otext = open(os.path.join(ROOT, "oracle", "mhd_oracle.cpp")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "csrc" not in otext.replace("paper_0908_4362_b200/csrc (the CUDA path)", "") and "libmhd.so" not in otext

"""CPU-only checks of the boundary: libgrav.so loads and exports every symbol include/grav.h declares; the Python
binding names them all; host-side argument validation that needs no device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "grav.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(grav_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2602_03857_b200 import _build
    return ctypes.CDLL(_build.build())


def test_header_declares_the_north_star_calls():
    names = _declared()
    for must in ["grav_mesh_create", "grav_forward", "grav_adjoint", "grav_depth_weights", "grav_dataspace_cg"]:
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    for name in _declared():
        assert hasattr(lib, name), f"libgrav.so does not export {name}"


def test_binding_lists_every_declared_symbol():
    from paper_2602_03857_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()


def test_no_oracle_in_product_path():
    """The product path must not import, link or execute anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2602_03857_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) == "build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "liboracle" not in txt and "oracle.cpp" not in txt, f


def test_last_error_without_device(lib):
    lib.grav_last_error.restype = ctypes.c_char_p
    lib.grav_workspace_bytes.restype = ctypes.c_size_t
    lib.grav_workspace_bytes.argtypes = [ctypes.c_void_p, ctypes.c_int]
    assert lib.grav_workspace_bytes(None, 0) == 0
    lib.grav_mesh_create.restype = ctypes.c_int
    out = ctypes.c_void_p()
    # NULL arrays / bad sizes are rejected before any CUDA call
    st = lib.grav_mesh_create(ctypes.byref(out), 0, 1, 1, None, None, None, ctypes.c_longlong(1), None, None, None,
                              ctypes.c_double(1.0), 0)
    assert st == -1 and b"positive" in lib.grav_last_error()
    st = lib.grav_mesh_create(ctypes.byref(out), 1, 1, 1, None, None, None, ctypes.c_longlong(1), None, None, None,
                              ctypes.c_double(1.0), 0)
    assert st == -1 and b"NULL" in lib.grav_last_error()

"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/u1mps.h declares; argument validation that needs no GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2303_11409_b200 import build, binding
    build.build()
    return binding.load_library()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "u1mps.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(u1mps_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_exported(lib):
    names = declared_symbols()
    assert len(names) >= 28
    for n in names:
        assert hasattr(lib, n), n


def test_binding_lists_every_symbol():
    from paper_2303_11409_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()


def test_strerror_and_version(lib):
    assert lib.u1mps_strerror(0) == b"ok"
    assert b"charge" in lib.u1mps_strerror(-2)
    assert b"sm_100a" in lib.u1mps_version()


def test_workspace_bytes(lib):
    assert lib.u1mps_workspace_bytes(1, 2, 1, 8) == 0          # M < 2
    assert lib.u1mps_workspace_bytes(16, 2, 8, 5000) == 0      # chi > U1MPS_CHI_MAX
    assert lib.u1mps_workspace_bytes(16, 9, 8, 32) == 0        # d > U1MPS_D_MAX
    assert lib.u1mps_workspace_bytes(16, 2, 17, 32) == 0       # N > M (d-1)
    small = lib.u1mps_workspace_bytes(16, 2, 8, 32)
    big = lib.u1mps_workspace_bytes(128, 2, 64, 1024)
    assert 0 < small < big
    # state alone: M chi^2 complex128
    assert big >= 128 * 1024 * 1024 * 16
    huge = lib.u1mps_workspace_bytes(100, 4, 50, 4096)
    assert 100 * 4096 * 4096 * 16 <= huge < 40 * 2 ** 30       # config 5 fits a 180 GB GPU many times over


def test_create_rejects_bad_arguments_without_gpu(lib):
    h = ctypes.c_void_p()
    assert lib.u1mps_create(ctypes.byref(h), 16, 2, 8, 32, None, 1 << 20, None) == -1
    assert lib.u1mps_create(None, 16, 2, 8, 32, ctypes.c_void_p(256), 1 << 20, None) == -1
    # too small an arena
    assert lib.u1mps_create(ctypes.byref(h), 16, 2, 8, 32, ctypes.c_void_p(256), 1024, None) == -4


def test_product_path_has_no_oracle_import():
    pkg = os.path.join(ROOT, "paper_2303_11409_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "u1mps_oracle" not in txt and "import oracle" not in txt, f

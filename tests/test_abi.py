"""CPU-side checks of the boundary: the library builds, loads, and exports every symbol that
include/tdse.h declares.  No compute calls (there is no GPU here)."""
import ctypes
import os
import re

import pytest

import paper_2401_07416_b200 as pkg
from paper_2401_07416_b200.build import build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build()
    return pkg.load()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "tdse.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tdse_[a-z_]+)\s*\(", text)))


def test_header_and_binding_agree_on_the_symbol_list():
    assert declared_symbols() == sorted(pkg.SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert getattr(lib, name) is not None


def test_workspace_bytes_is_pure_host_arithmetic(lib):
    n3 = lib.tdse_workspace_bytes(64, 64, 64, 1, pkg.TDSE_F64, 0)
    n5 = lib.tdse_workspace_bytes(64, 64, 64, 1, pkg.TDSE_F64, 1)
    # device storage frames every xy plane with 4 columns / 4 rows on each side (include/tdse.h, tdse_workspace_bytes)
    assert n3 == 3 * 72 * 72 * 64 * 8 and n5 == 5 * 72 * 72 * 64 * 8
    assert lib.tdse_workspace_bytes(5, 3, 7, 2, pkg.TDSE_F32, 0) == 3 * 8192   # 13*11*7*2*4 = 8008 B rounded up to 256-B multiples
    assert lib.tdse_workspace_bytes(0, 3, 7, 2, pkg.TDSE_F32, 0) == 0
    assert lib.tdse_workspace_bytes(4, 4, 4, 1, 7, 0) == 0


def test_create_fails_loudly_without_a_device_or_with_bad_arguments(lib):
    import torch
    h = ctypes.c_void_p()
    assert lib.tdse_create(ctypes.byref(h), 0, 4, 4, 1, 0.1, 0.1, 1.0, 1.0, pkg.TDSE_F64) == pkg.TDSE_EINVAL
    assert lib.tdse_create(ctypes.byref(h), 4, 4, 4, 1, -0.1, 0.1, 1.0, 1.0, pkg.TDSE_F64) == pkg.TDSE_EINVAL
    assert b"dx" in lib.tdse_last_error(None)
    if not torch.cuda.is_available():
        code = lib.tdse_create(ctypes.byref(h), 4, 4, 4, 1, 0.1, 0.1, 1.0, 1.0, pkg.TDSE_F64)
        assert code == pkg.TDSE_ECUDA                       # no CPU fallback
        assert b"no CPU fallback" in lib.tdse_last_error(None)
        assert not h.value


def test_null_context_is_rejected(lib):
    assert lib.tdse_step(None, 1) == pkg.TDSE_EINVAL
    assert lib.tdse_destroy(None) == pkg.TDSE_OK
    assert lib.tdse_last_error(None) is not None


def test_product_path_does_not_import_the_oracle():
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2401_07416_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(root, f)).read()
                assert "oracle" not in src.lower(), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".inc")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2401_07416_b200" not in src and "libtdse" not in src, f

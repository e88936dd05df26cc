"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol include/submatrix.h
declares, argument validation answers without a GPU, and the binding has no CPU fallback."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2205_14741_b200 import build
    return ctypes.CDLL(build.build())


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "submatrix.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sm_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_five_path_calls():
    syms = declared_symbols()
    for name in ("sm_build_pattern", "sm_gather", "sm_sign_ns", "sm_scatter", "sm_density"):
        assert name in syms


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_binding_lists_the_same_symbols():
    src = open(os.path.join(ROOT, "paper_2205_14741_b200", "binding.py")).read()
    for name in declared_symbols():
        assert name in src, name
    assert "oracle" not in src.replace("oracle/", "")       # the product never routes through the oracle


def test_argument_errors_without_a_gpu(lib):
    lib.sm_sign_ws_bytes.restype = ctypes.c_int64
    assert lib.sm_pattern_sizes(None, 16, None, None, None) == -1           # SM_ERR_ARG
    assert lib.sm_build_pattern(None, 16, None, None, ctypes.c_int64(0), None) == -1
    assert lib.sm_sign_ns(None, None, 0, None, ctypes.c_int64(0), 0, None, None, ctypes.c_int64(0), 1,
                          ctypes.c_double(0.0), None, None, None) == -1
    assert lib.sm_sign_ws_bytes(None, 0, ctypes.c_int64(0), 0) == -1
    assert lib.sm_last_cuda_error() == 0


def test_product_sources_do_not_touch_the_oracle_or_work_dirs():
    pkg = os.path.join(ROOT, "paper_2205_14741_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "_work" not in text, f
                assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), f

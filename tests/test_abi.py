"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every
symbol include/tsm.h declares (no compute calls), and the Python binding fails loudly
without a GPU instead of falling back to anything."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1211_0126_b200.build import build_library
    return build_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "tsm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tsm_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_boundary_calls():
    syms = declared_symbols()
    for need in ["tsm_create", "tsm_set_gauge", "tsm_noise", "tsm_dslash", "tsm_solve",
                 "tsm_loops_add_correction", "tsm_loops_add_lp", "tsm_loops_finalize", "tsm_run_loop_set"]:
        assert need in syms


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/tsm.h but not exported by libtsm.so"


def test_binding_covers_every_declared_symbol(lib_path):
    from paper_1211_0126_b200 import tsm
    assert sorted(tsm.EXPORTS) == declared_symbols()
    lib = tsm.load_library()
    for name in tsm.EXPORTS:
        assert getattr(lib, name).argtypes is not None or name == "tsm_last_error"


def test_argument_validation_needs_no_gpu(lib_path):
    lib = ctypes.CDLL(lib_path)
    h = ctypes.c_void_p()
    bad = (ctypes.c_int * 4)(4, 4, 3, 8)        # odd extent
    assert lib.tsm_create(ctypes.byref(h), bad, -1, 0) == -1
    small = (ctypes.c_int * 4)(2, 4, 4, 8)      # extent < 4
    assert lib.tsm_create(ctypes.byref(h), small, -1, 0) == -1
    ok = (ctypes.c_int * 4)(4, 4, 4, 8)
    assert lib.tsm_create(ctypes.byref(h), ok, 0, 0) == -1      # boundary phase must be +-1
    assert lib.tsm_destroy(None) == -1


def test_no_cpu_fallback(lib_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1211_0126_b200 import tsm
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        tsm.Tsm((4, 4, 4, 8))


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1211_0126_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "tsm_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1211_0126_b200", src, flags=re.M), f
            assert not re.search(r"#include\s+[<\"].*(csrc|tsm\.h)", src), f

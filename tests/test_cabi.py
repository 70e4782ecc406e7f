"""CPU-side checks of the boundary: the built C-ABI library loads and exports every symbol that
include/sfft.h declares; the binding fails loudly without a GPU (no CPU fallback)."""
import ctypes
import os
import re

import pytest

import paper_2603_08593_b200 as pkg
from paper_2603_08593_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _ensure_built():
    if not os.path.exists(pkg.lib_path()):
        from paper_2603_08593_b200 import build
        build.build()


def test_header_symbols_match_binding_list():
    text = open(os.path.join(ROOT, "include", "sfft.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(sfft_[a-z0-9_]+)\s*\(", text))
    assert declared == set(binding.EXPORTED_SYMBOLS)


def test_library_loads_and_exports_every_declared_symbol():
    _ensure_built()
    lib = ctypes.CDLL(pkg.lib_path())
    for name in binding.EXPORTED_SYMBOLS:
        assert hasattr(lib, name), name
    lib.sfft_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.sfft_version()
    lib.sfft_status_string.restype = ctypes.c_char_p
    assert lib.sfft_status_string(0) == b"SFFT_OK"
    assert lib.sfft_status_string(2) == b"SFFT_ERR_UNSUPPORTED"


def test_argument_validation_needs_no_gpu():
    _ensure_built()
    lib = pkg.load_library()
    p = ctypes.c_void_p(0)
    # unsupported sizes are rejected before any CUDA call
    assert lib.sfft_plan_create(ctypes.byref(p), 100, 64, 2, 0, 0) == 2
    assert lib.sfft_plan_create(ctypes.byref(p), 64, 64, 2, 4, 0) == 2
    assert lib.sfft_plan_create(ctypes.byref(p), 32, 32, 9, 0, 0) == 2
    assert lib.sfft_plan_create(ctypes.byref(p), 8, 64, 0, 0, 0) == 2      # below the smallest size (16)
    assert lib.sfft_plan_create(ctypes.byref(p), 16, 16, 4, 0, 0) == 2     # 4w + 1 > min(H, W)
    assert lib.sfft_plan_create(ctypes.byref(p), 128, 128, 16, 0, 0) == 2  # w above the largest half-width (15)
    assert lib.sfft_plan_create(None, 64, 64, 2, 0, 0) == 1
    assert p.value in (None, 0)
    assert lib.sfft_num_coeffs(None) == -1
    assert lib.sfft_workspace_bytes(None) == 0
    assert lib.sfft_build_system(None, None, None, None, None, None, None) == 1
    assert lib.sfft_solve(None, None, None, None, None, None) == 1
    assert lib.sfft_subtract(None, None, None, None, None, None) == 1
    assert lib.sfft_last_launch_count(None, 0) == -1
    # the allocation-free solve validates before any CUDA call: NULL -> INVALID_ARG, N beyond the static
    # workspace -> UNSUPPORTED (the pointers are never dereferenced on the host)
    fake = ctypes.c_void_p(256)
    assert lib.sfft_solve_static(None, None, 5, None, None, None) == 1
    assert lib.sfft_solve_static(fake, fake, 0, fake, None, None) == 1
    assert lib.sfft_solve_static(fake, fake, 769, fake, None, None) == 2


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    _ensure_built()
    with pytest.raises(pkg.SfftError) as ei:
        pkg.SfftPlan(64, 64, 2, 0, 0)
    assert ei.value.code == 4  # SFFT_ERR_CUDA: no device -> loud failure, never an oracle route


def test_product_code_never_imports_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2603_08593_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
    src = open(os.path.join(ROOT, "oracle", "sfft_oracle.py")).read()
    assert "paper_2603_08593_b200" not in src.replace("paper_2603_08593_b200/csrc", "")

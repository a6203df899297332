"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/coarse_mrhs.h declares (no compute calls -- there is no GPU here), and argument validation
that happens before any CUDA call returns the documented status codes."""
import ctypes as C
import os
import re

import pytest

import paper_2409_03904_b200 as cm
from paper_2409_03904_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "coarse_mrhs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = re.findall(r"\b(coarse_[a-z_0-9]+|p?block_cg_[a-z_0-9]+|stacked_cg_[a-z_0-9]+)\s*\(", text)
    return sorted(set(names))


def test_library_exports_every_declared_symbol():
    L = cm.lib()
    declared = _declared_symbols()
    assert len(declared) >= 16
    for name in declared:
        assert hasattr(L, name), f"{name} declared in include/coarse_mrhs.h but not exported"
    assert sorted(binding.EXPORTS) == declared


def test_invalid_arguments_are_rejected_before_any_cuda_call():
    L = cm.lib()
    h = C.c_void_p()
    dims = (C.c_int32 * 4)(4, 4, 4, 0)
    assert L.coarse_op_create(C.byref(h), dims, 8, 4, cm.C64, C.c_void_p(16), 0, None) == binding.INVALID_ARG
    assert b"dims[3]" in L.coarse_last_error()
    dims = (C.c_int32 * 4)(4, 4, 4, 4)
    assert L.coarse_op_create(C.byref(h), dims, 65, 4, cm.C64, C.c_void_p(16), 0, None) == binding.UNSUPPORTED
    assert L.coarse_op_create(C.byref(h), dims, 8, 65, cm.C64, C.c_void_p(16), 0, None) == binding.UNSUPPORTED
    assert L.coarse_op_create(C.byref(h), dims, 8, 4, 7, C.c_void_p(16), 0, None) == binding.INVALID_ARG
    assert L.coarse_op_create(C.byref(h), dims, 8, 4, cm.C64, None, 0, None) == binding.INVALID_ARG
    assert L.coarse_op_apply(None, None, None, 4, None) == binding.INVALID_ARG
    assert L.coarse_op_destroy(None) == binding.OK
    assert L.coarse_launch_count() == 0


def test_result_struct_layout_matches_header():
    # int32 x2, double[64] x2, double[256], double
    assert C.sizeof(binding.BlockCGResult) == 8 + 8 * (64 + 64 + 256 + 1)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2409_03904_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert not re.search(r"#include\s+[\"<][^\">]*oracle", text), f

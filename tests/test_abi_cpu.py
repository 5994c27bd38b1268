"""CPU-side checks of the C-ABI boundary: the library builds, loads and exports every symbol that
include/mwf.h declares, the structs have the paper's sizes, and host-only entry points behave.  No
compute call is made here (there is no GPU in this container)."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1907_02290_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build_mwf()
    return binding.load_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "mwf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mwf_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    syms = declared_symbols()
    assert sorted(binding.SYMBOLS) == syms
    for s in syms:
        assert hasattr(lib, s), s


def test_struct_sizes_match_the_paper(golden):
    # EPJ/SPJ float4 16 B, FORCE float4 16 B, list id 4 B (tests/golden/paper_constants.txt)
    assert np.dtype(np.float32).itemsize * 4 == golden["b_epj_bytes"] == golden["b_force_bytes"]
    assert np.dtype(np.int32).itemsize == golden["b_id_bytes"]
    assert ctypes.sizeof(binding.Params) == 48
    assert (binding.MAKE_LIST, binding.MAKE_LIST_FOR_REUSE, binding.REUSE_LIST) == (
        golden["mode_make_list"], golden["mode_make_list_for_reuse"], golden["mode_reuse_list"])


def test_strerror_and_arena_bytes(lib):
    assert lib.mwf_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4, -5):
        assert lib.mwf_strerror(code) not in (b"ok", b"unknown error code")
    p = binding.Params(1 / 256, 1.0, 1 << 20, 1 << 18, 1 << 14, 1 << 26, 8, 0)
    n = ctypes.c_int64(0)
    assert lib.mwf_arena_bytes(ctypes.byref(p), ctypes.byref(n)) == 0
    # store + results + merged list + staging dominate; velocities, the sort / tree-build buffers of the
    # device-side construction step and its walk stacks (<= 148 x 32 warps x 24 KB) come on top
    lower = (p.max_ptcl + p.max_cell) * 16 + p.max_ptcl * 16 + 2 * p.max_entry * 4
    assert lower < n.value < lower * 1.1 + 80 * p.max_ptcl + 48 * p.max_cell + 148 * 32 * 24576 + (1 << 20)
    bad = binding.Params(0.0, 1.0, 10, 10, 10, 10, 8, 0)          # eps must be > 0 (reading S2)
    assert lib.mwf_arena_bytes(ctypes.byref(bad), ctypes.byref(n)) == binding.EINVAL
    bad = binding.Params(0.1, 1.0, 10, 10, 10, 10, 99, 0)
    assert lib.mwf_arena_bytes(ctypes.byref(bad), ctypes.byref(n)) == binding.EINVAL
    bad = binding.Params(0.1, 1.0, 1 << 31, 10, 10, 10, 8, 0)     # 32-bit list indices
    assert lib.mwf_arena_bytes(ctypes.byref(bad), ctypes.byref(n)) == binding.EINVAL


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        binding.MultiWalkForce(0.1, max_ptcl=10, max_cell=10, max_group=10, max_entry=10)
    # the raw ABI fails loudly too
    lib = binding.load_library()
    p = binding.Params(0.1, 1.0, 10, 10, 10, 10, 1, 0)
    h = ctypes.c_void_p(None)
    assert lib.mwf_create(ctypes.byref(h), ctypes.byref(p), None, 0) == binding.ECUDA
    assert not h.value


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1907_02290_b200")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h", ".cuh")):
                text = open(os.path.join(d, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "mwf_oracle" not in text and "orc_" not in text, f

"""The C-ABI boundary without a GPU: libcpra.so builds, loads and exports every symbol that
include/cpra.h declares; host-only calls validate their arguments; compute calls never fall back
to the CPU.  (No compute call is made here.)"""
import ctypes
import os
import re

import pytest

import paper_2402_05283_b200 as cpra

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "cpra.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(cpra_[a-z0-9_]+)\s*\(", text)))


def test_header_and_binding_agree_and_library_exports_everything():
    names = _declared_symbols()
    assert "cpra_plan" in names and "cpra_iterate" in names and "cpra_assemble_3d" in names
    assert set(names) == set(cpra.SIGNATURES), set(names) ^ set(cpra.SIGNATURES)
    L = ctypes.CDLL(cpra.build())
    for n in names:
        assert hasattr(L, n), n


def test_north_star_entry_points_exist():
    for n in ("cpra_plan", "cpra_set_data", "cpra_set_support", "cpra_iterate", "cpra_get_projections",
              "cpra_assemble_3d"):
        assert n in cpra.SIGNATURES


def test_host_only_argument_validation():
    L = cpra.lib()
    h = ctypes.c_void_p()
    assert L.cpra_plan(None, 64, 4, 0, None) == cpra.ERR_INVALID_ARG
    for N in (0, 8, 15, 22, 34, 1026, 2048):      # too small / odd / a prime factor above 7 / too large
        assert L.cpra_plan(ctypes.byref(h), N, 4, 0, None) == cpra.ERR_UNSUPPORTED_SIZE
    for N in (48, 100, 160, 700):                 # 2^a 3^b 5^c 7^d: the mixed-radix path (the paper's 160 and 700 among them)
        assert L.cpra_plan(ctypes.byref(h), N, 4, 0, None) == cpra.CPRA_OK
        assert L.cpra_destroy(h) == cpra.CPRA_OK
    assert L.cpra_plan(ctypes.byref(h), 64, 0, 0, None) == cpra.ERR_UNSUPPORTED_SIZE
    assert L.cpra_plan(ctypes.byref(h), 64, 5, 8, None) == cpra.ERR_INVALID_ARG       # undefined flag bit
    assert L.cpra_plan(ctypes.byref(h), 64, 5, cpra.FLAG_NO_WALK | cpra.FLAG_NO_CHUNKING, None) == cpra.CPRA_OK
    assert L.cpra_destroy(h) == cpra.CPRA_OK
    assert L.cpra_plan(ctypes.byref(h), 64, 5, 0, None) == cpra.CPRA_OK
    nb = ctypes.c_size_t()
    assert L.cpra_workspace_bytes(h, ctypes.byref(nb)) == cpra.CPRA_OK
    px = 5 * 64 * 64
    assert nb.value >= px * (8 + 8 + 4) and nb.value % 256 == 0
    # nothing bound yet: compute calls must refuse, not fall back
    assert L.cpra_iterate(h, 1, 0.9) == cpra.ERR_WORKSPACE
    assert L.cpra_iterate(h, -1, 0.9) == cpra.ERR_INVALID_ARG
    assert L.cpra_iterate(h, 1, float("nan")) == cpra.ERR_INVALID_ARG
    import numpy as np
    al = np.array([0.5, 0.25], dtype=np.float64)
    assert L.cpra_set_carousel(h, 1, al.ctypes.data, 2) == cpra.CPRA_OK
    assert L.cpra_set_carousel(h, 1, al.ctypes.data, 0) == cpra.ERR_INVALID_ARG
    assert L.cpra_set_carousel(h, 3, al.ctypes.data, 1) == cpra.ERR_INVALID_ARG      # 2K+1 > Np
    assert L.cpra_set_carousel(h, -1, al.ctypes.data, 1) == cpra.ERR_INVALID_ARG
    assert L.cpra_set_carousel(h, 1, None, 1) == cpra.ERR_INVALID_ARG
    t = ctypes.c_long(-1)
    assert L.cpra_get_iteration(h, ctypes.byref(t)) == cpra.CPRA_OK and t.value == 0
    assert L.cpra_set_iteration(h, 7) == cpra.CPRA_OK
    assert L.cpra_get_iteration(h, ctypes.byref(t)) == cpra.CPRA_OK and t.value == 7
    assert L.cpra_set_iteration(h, -1) == cpra.ERR_INVALID_ARG
    assert L.cpra_bind_workspace(h, None, 0) == cpra.ERR_INVALID_ARG
    assert L.cpra_status_string(cpra.ERR_NOT_READY) == b"CPRA_ERR_NOT_READY"
    assert L.cpra_status_string(12345) == b"CPRA_ERR_UNKNOWN"
    assert L.cpra_destroy(h) == cpra.CPRA_OK
    assert L.cpra_destroy(None) == cpra.ERR_INVALID_ARG


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(cpra.CpraError) as e:
        cpra.Plan(64, 4)
    assert e.value.code == cpra.ERR_CUDA
    with pytest.raises(cpra.CpraError) as e:
        cpra.Plan(22, 4)
    assert e.value.code == cpra.ERR_UNSUPPORTED_SIZE


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2402_05283_b200")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert "oracle" not in open(os.path.join(d, f)).read().lower(), os.path.join(d, f)
    for d, _, files in os.walk(os.path.join(ROOT, "oracle")):
        for f in files:
            if f.endswith((".py", ".c", ".h")):
                src = open(os.path.join(d, f)).read()
                assert not re.search(r"^\s*(import|from)\s+paper_2402_05283_b200", src, flags=re.M), f
                assert "libcpra" not in src and "cpra.h" not in src, f

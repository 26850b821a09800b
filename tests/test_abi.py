"""The C-ABI library loads on a CPU-only box and exports every symbol include/joseph_b200.h declares
(no compute calls here).  Also checks host-side argument validation, which needs no GPU."""
import ctypes as C
import os
import re

import pytest

from paper_2212_12519_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "joseph_b200.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(jp_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def test_header_symbols_exported(lib):
    names = declared_functions()
    assert "jp_fwd" in names and "jp_back_tof_lm" in names and "jp_lm_osem" in names
    for name in names:
        assert hasattr(lib, name), f"{name} declared in joseph_b200.h but not exported"
    assert sorted(binding.EXPORTS) == names, "binding.EXPORTS and the header disagree"


def test_struct_layouts_match_header():
    assert C.sizeof(binding.jp_geom) == 36
    assert C.sizeof(binding.jp_tof) == 20
    assert C.sizeof(binding.jp_lors) == 56


def test_version_and_error_string(lib):
    assert lib.jp_version() >= 100
    assert isinstance(lib.jp_last_error(), bytes)


def test_argument_validation_without_gpu(lib):
    """validation happens before anything is enqueued, so it can be exercised on a CPU box"""
    g = binding.make_geom((4, 4, 4), (0, 0, 0), (1, 1, 1))
    l = binding.jp_lors(0, 0, 0, 0, 0, 0, 5)
    assert lib.jp_fwd(C.byref(l), None, C.byref(g), None, None) == -1          # NULL arrays
    l.n = -1
    assert lib.jp_fwd(C.byref(l), None, C.byref(g), None, None) == -2          # n < 0
    assert b"n < 0" in lib.jp_last_error()
    l = binding.jp_lors(8, 8, 8, 8, 8, 8, 1)
    bad = binding.make_geom((4, 0, 4), (0, 0, 0), (1, 1, 1))
    assert lib.jp_fwd(C.byref(l), C.c_void_p(8), C.byref(bad), C.c_void_p(8), None) == -2
    bad = binding.make_geom((4, 4, 4), (0, 0, 0), (1, -1, 1))
    assert lib.jp_back(C.byref(l), C.c_void_p(8), C.byref(bad), C.c_void_p(8), None) == -2
    t = binding.make_tof(17.0, 13.6, 3.0, 0)
    assert lib.jp_fwd_tof_sino(C.byref(l), C.c_void_p(8), C.byref(g), C.byref(t), C.c_void_p(8), None) == -2
    t = binding.make_tof(17.0, 0.0, 3.0, 29)
    assert lib.jp_fwd_tof_lm(C.byref(l), C.c_void_p(8), C.c_void_p(8), C.byref(g), C.byref(t), C.c_void_p(8), None) == -2
    assert lib.jp_fwd(None, None, C.byref(g), None, None) == -1
    assert lib.jp_lm_osem_workspace_bytes(40_000_000, C.byref(binding.make_geom((200, 200, 96), (0,) * 3, (2,) * 3)), 20) \
        >= (200 * 200 * 96 + 2_000_000) * 4


def test_argument_validation_of_the_osem_calls_without_gpu(lib):
    g = binding.make_geom((4, 4, 4), (0, 0, 0), (1, 1, 1))
    t = binding.make_tof(17.0, 13.6, 3.0, 29)
    l = binding.jp_lors(8, 8, 8, 8, 8, 8, 10)
    P = C.c_void_p(8)
    off_ok = (C.c_int64 * 3)(0, 4, 10)
    off_dec = (C.c_int64 * 3)(0, 6, 4)
    off_out = (C.c_int64 * 3)(0, 4, 11)
    call = lambda off, ns, sens=P, ws=P, wb=1 << 20: lib.jp_sino_osem_tof(C.byref(l), off, ns, P, None, None, sens, C.byref(g),
                                                                          C.byref(t), P, 1, ws, wb, None)
    assert call(off_dec, 2) == -2 and b"non-decreasing" in lib.jp_last_error()
    assert call(off_out, 2) == -2
    assert call(off_ok, 0) == -2
    assert call(None, 2) == -1
    assert call(off_ok, 2, sens=None) == -1
    assert call(off_ok, 2, wb=16) == -2 and b"workspace" in lib.jp_last_error()
    assert lib.jp_sino_osem_tof_workspace_bytes(off_ok, 2, 10, C.byref(t)) >= 6 * 29 * 4
    assert lib.jp_sino_osem_tof_workspace_bytes(off_dec, 2, 10, C.byref(t)) == 0
    assert lib.jp_sino_sens_tof(C.byref(l), off_ok, 2, None, C.byref(g), C.byref(t), None, None, 0, None) == -1
    assert lib.jp_osem_update(None, P, P, 1.0, C.byref(g), None) == -1
    assert lib.jp_lm_osem_planned_backratio(None, 0, P, P, P, 1 << 20, None) == -4
    assert lib.jp_fwd_tof_sino_host(None, P, C.byref(g), C.byref(t), P) == -1
    bad = binding.make_tof(17.0, 13.6, 3.0, 0)
    assert lib.jp_fwd_tof_sino_host(C.byref(l), P, C.byref(g), C.byref(bad), P) == -2


def test_no_cpu_fallback():
    import torch
    x = torch.zeros((3, 4))
    with pytest.raises(binding.JosephError):
        binding.jp_fwd(x, x, torch.zeros((4, 4, 4)), (0, 0, 0), (1, 1, 1))

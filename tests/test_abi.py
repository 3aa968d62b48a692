"""Host-side checks that need no GPU: the C-ABI library builds, loads, and exports every symbol that
include/slam.h declares; sizes and argument validation that happen before any launch."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2603_25834_b200 import build
    return ctypes.CDLL(build.build())


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "slam.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(slam_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    syms = declared_symbols()
    assert len(syms) >= 20
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in include/slam.h but not exported"


def test_binding_lists_every_symbol():
    src = open(os.path.join(ROOT, "paper_2603_25834_b200", "binding.py")).read()
    for s in declared_symbols():
        assert f'"{s}"' in src


def test_workspace_bytes_and_size_validation(lib):
    lib.slam_workspace_bytes.restype = ctypes.c_size_t
    lib.slam_workspace_bytes.argtypes = [ctypes.c_int] * 3
    assert lib.slam_workspace_bytes(0, 10, 0) == 0
    assert lib.slam_workspace_bytes(4, 1, 0) == 0
    assert lib.slam_workspace_bytes(4, 65, 0) == 0
    assert lib.slam_workspace_bytes(4, 10, 65) == 0
    small = lib.slam_workspace_bytes(4, 10, 0)
    big = lib.slam_workspace_bytes(16384, 20, 24)
    assert 0 < small < big
    # the prior is stored with worst-case capacity n(n+1)/2 floats per environment
    n = 3 * 20 + 2 * 24
    assert big >= 16384 * (n * (n + 1) // 2) * 4
    assert big < 16384 * 96 * 1024            # fp32 record + fp64 shadow record (slam_set_precision)
    # the largest supported window (W = 64, L = 64: n = 320) still fits the shared memory of one SM
    assert lib.slam_workspace_bytes(1, 64, 64) > 0
    # the largest BASELINE configuration fits the 180 GB of one B200 many times over
    assert lib.slam_workspace_bytes(65536, 50, 0) < 16 * 2 ** 30


def test_create_rejects_bad_arguments(lib):
    lib.slam_create.argtypes = [ctypes.POINTER(ctypes.c_void_p), ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p]
    h = ctypes.c_void_p()
    assert lib.slam_create(ctypes.byref(h), 4, 10, 0, None, None, 0, None) == 1      # NULL workspace
    assert lib.slam_create(ctypes.byref(h), 4, 10, 0, None, ctypes.c_void_p(128), 1 << 20, None) == 1  # misaligned
    assert lib.slam_create(None, 4, 10, 0, None, ctypes.c_void_p(256), 1 << 20, None) == 1
    assert not h.value


def test_default_config(lib):
    from harness import synth

    class Cfg(ctypes.Structure):
        _fields_ = [("p", ctypes.c_float * 3), ("o", ctypes.c_float * 3), ("l", ctypes.c_float * 3), ("r", ctypes.c_float * 2)]

    c = Cfg()
    lib.slam_default_config(ctypes.byref(c))
    assert tuple(round(x, 6) for x in c.p) == synth.PRIOR_SIGMA
    assert tuple(round(x, 6) for x in c.o) == synth.ODO_SIGMA
    assert tuple(round(x, 6) for x in c.l) == synth.LC_SIGMA
    assert tuple(round(x, 6) for x in c.r) == synth.RB_SIGMA

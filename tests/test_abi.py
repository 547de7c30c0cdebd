"""CPU checks of the boundary: the C-ABI library loads, exports every symbol include/lqcd.h
declares, and refuses to work without a device (no CPU fallback)."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "lqcd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lqcd_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2411_08461_b200 import build, lqcd
    build.build()
    L = ctypes.CDLL(build.SO)
    names = declared_symbols()
    assert len(names) >= 25
    for n in names:
        assert hasattr(L, n), n
    assert sorted(lqcd.SYMBOLS) == names      # the Python binding carries the same names


def test_error_strings_and_null_handling():
    from paper_2411_08461_b200 import lqcd
    L = lqcd.load()
    assert L.lqcd_strerror(0) == b"ok"
    assert b"singular" in L.lqcd_strerror(-6)
    assert L.lqcd_gauge_bytes(None) == 0 and L.lqcd_launch_count(None) == 0
    h = ctypes.c_void_p()
    dims = (ctypes.c_int * 4)(4, 4, 4, 8)
    assert L.lqcd_create(ctypes.byref(h), dims, 3, 18, -1, 0) == -1        # bad precision
    assert L.lqcd_create(ctypes.byref(h), (ctypes.c_int * 4)(4, 4, 3, 8), 8, 18, -1, 0) == -2  # odd extent
    assert L.lqcd_create(ctypes.byref(h), (ctypes.c_int * 4)(2, 4, 4, 8), 8, 18, -1, 0) == -2  # L < 4


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-device behaviour")
def test_no_cpu_fallback_without_device():
    from paper_2411_08461_b200 import lqcd
    with pytest.raises(lqcd.LqcdError):
        lqcd.Context((4, 4, 4, 8))

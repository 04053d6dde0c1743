"""The C-ABI library builds, loads and exports every symbol include/nmf.h declares (no GPU)."""
import ctypes
import os
import re

from paper_2309_04623_b200 import build as nmf_build
from paper_2309_04623_b200 import nmf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "nmf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nmf_[a-z_]+)\s*\(", src)))


def test_header_symbols_exported():
    path = nmf_build.build()
    L = ctypes.CDLL(path)
    names = _declared()
    assert len(names) >= 15
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/nmf.h but not exported"
    assert sorted(nmf.SYMBOLS) == names, "python binding and header disagree"


def test_status_strings_and_null_plan():
    L = nmf.lib()
    assert L.nmf_status_string(0) == b"NMF_OK"
    for code in range(-6, 0):
        assert L.nmf_status_string(code).startswith(b"NMF_ERR_")
    assert L.nmf_plan_workspace_bytes(None) == 0
    assert L.nmf_plan_destroy(None) == -1
    assert L.nmf_fit(None, None, None, None, None, 1) == -1
    h = ctypes.c_void_p()
    assert L.nmf_plan_create(ctypes.byref(h), 0, 64, 4, 1, 0) == -1       # N < 1
    assert L.nmf_plan_create(ctypes.byref(h), 4, 66, 4, 1, 0) == -2       # P % 4
    assert L.nmf_plan_create(ctypes.byref(h), 257, 64, 4, 1, 0) == -3     # N > 256
    assert L.nmf_plan_create(ctypes.byref(h), 4, 64, 129, 1, 0) == -3     # K > 128

"""CPU-side checks of the boundary: libwd.so builds, loads and exports every symbol include/wd.h
declares (no compute calls without a GPU), and the product never imports the oracle."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1009_5169_b200 import build, wd
    path = build.build()
    L = ctypes.CDLL(path)
    hdr = open(os.path.join(ROOT, "include", "wd.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(wd_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(wd.SYMBOLS), declared ^ set(wd.SYMBOLS)
    for name in declared:
        assert hasattr(L, name), name
    L.wd_version.restype = ctypes.c_char_p
    assert b"sm_100a" in L.wd_version()
    L.wd_strerror.restype = ctypes.c_char_p
    L.wd_strerror.argtypes = [ctypes.c_int]
    assert L.wd_strerror(-4) and L.wd_strerror(0) == b"ok"


def test_solve_info_struct_matches_header():
    from paper_1009_5169_b200 import wd
    # 4 ints, 2*16 doubles, 1 double
    assert ctypes.sizeof(wd.SolveInfo) == 16 + 8 * (2 * wd.MAX_RHS + 1)
    hdr = open(os.path.join(ROOT, "include", "wd.h")).read()
    assert f"#define WD_MAX_RHS {wd.MAX_RHS}" in hdr


def test_product_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1009_5169_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                for pat in ("import oracle", "from oracle", "wd_oracle", "libwd_oracle", "orc_"):
                    assert pat not in src, (f, pat)


def test_create_rejects_bad_arguments_without_a_gpu_call():
    from paper_1009_5169_b200 import wd
    L = wd.lib()
    h = ctypes.c_void_p()
    assert L.wd_create(None, (ctypes.c_int * 4)(4, 4, 4, 4), 0.1, 1, 5, None) == wd.EINVAL
    assert L.wd_create(ctypes.byref(h), (ctypes.c_int * 4)(4, 4, 5, 4), 0.1, 1, 5, None) == wd.EINVAL
    assert L.wd_create(ctypes.byref(h), (ctypes.c_int * 4)(4, 4, 4, 4), float("nan"), 1, 5, None) == wd.EINVAL
    assert L.wd_create(ctypes.byref(h), (ctypes.c_int * 4)(4, 4, 4, 4), 0.1, 7, 5, None) == wd.EINVAL
    assert L.wd_create(ctypes.byref(h), (ctypes.c_int * 4)(4, 4, 4, 4), 0.1, 1, 0, None) == wd.EINVAL
    assert L.wd_create(ctypes.byref(h), (ctypes.c_int * 4)(4, 4, 4, 2), 0.1, 1, 5, None) == wd.EINVAL
    assert L.wd_destroy(None) == wd.EINVAL
    assert L.wd_workspace_bytes(None) == 0

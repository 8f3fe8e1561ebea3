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
    # a library built with the ablation switches of csrc/wd_hop_zm.cu (build.py WD_NVCC_DEFINES) must never be tested or shipped
    assert b"MEASUREMENT BUILD" not in L.wd_version(), L.wd_version()
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


def test_option_and_enum_constants_match_header():
    """The binding's integer constants are the header's (the binding only marshals arguments)."""
    from paper_1009_5169_b200 import wd
    hdr = open(os.path.join(ROOT, "include", "wd.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    consts = {k: int(v) for k, v in re.findall(r"\b(WD_[A-Z0-9_]+)\s*=\s*(-?\d+)", hdr)}
    pairs = {"WD_OK": wd.OK, "WD_EINVAL": wd.EINVAL, "WD_ENOCONV": wd.ENOCONV, "WD_BC_PERIODIC": wd.BC_PERIODIC,
             "WD_BC_SF": wd.BC_SF, "WD_OP_D": wd.OP_D, "WD_OP_DDAG": wd.OP_DDAG, "WD_F64": wd.F64, "WD_F32": wd.F32,
             "WD_LINK18": wd.LINK18, "WD_LINK12": wd.LINK12, "WD_ORDER_LINEAR": wd.ORDER_LINEAR,
             "WD_ORDER_TILED": wd.ORDER_TILED, "WD_OPT_HOP32_SITES": wd.OPT_HOP32_SITES,
             "WD_OPT_HOP64_SITES": wd.OPT_HOP64_SITES, "WD_OPT_HOP32_REGS": wd.OPT_HOP32_REGS,
             "WD_OPT_HOP64_REGS": wd.OPT_HOP64_REGS, "WD_OPT_POLL_EVERY": wd.OPT_POLL_EVERY,
             "WD_OPT_HOP_IMPL": wd.OPT_HOP_IMPL, "WD_OPT_ALTERNATE_SWEEP": wd.OPT_ALTERNATE_SWEEP,
             "WD_OPT_HOP_ROWS": wd.OPT_HOP_ROWS, "WD_OPT_SOLVER": wd.OPT_SOLVER, "WD_OPT_PAIRED": wd.OPT_PAIRED, "WD_OPT_GRAPH": wd.OPT_GRAPH, "WD_OPT_MERGE": wd.OPT_MERGE, "WD_F32P": wd.F32P, "WD_SOLVER_DC_F32": wd.SOLVER_DC_F32,
             "WD_SOLVER_RELIABLE_H16": wd.SOLVER_RELIABLE_H16, "WD_SOLVER_GL_FLEX": wd.SOLVER_GL_FLEX,
             "WD_SOLVER_GL_F64": wd.SOLVER_GL_F64, "WD_SOLVER_BL_F64": wd.SOLVER_BL_F64, "WD_ACTION_FULL": wd.ACTION_FULL, "WD_ACTION_EO": wd.ACTION_EO,
             "WD_PARITY_EVEN": wd.PARITY_EVEN, "WD_PARITY_ODD": wd.PARITY_ODD, "WD_PARITY_BOTH": wd.PARITY_BOTH}
    for name, val in pairs.items():
        assert consts[name] == val, name
    assert len(wd.PROF_NAMES) == consts["WD_PROF_N"]


def test_set_option_rejects_null_context():
    from paper_1009_5169_b200 import wd
    L = wd.lib()
    assert L.wd_set_option(None, 0, 1) == wd.EINVAL
    v = ctypes.c_int()
    assert L.wd_get_option(None, 0, ctypes.byref(v)) == wd.EINVAL


def test_round3_entry_points_reject_null_context():
    """wd_inner_plan and wd_set_residual_history are host-only calls on a context: without one they return WD_EINVAL
    (checked here on the CPU box; their behaviour on a context is in tests/test_gpu_parity.py)."""
    from paper_1009_5169_b200 import wd
    L = wd.lib()
    plan = (ctypes.c_int * 4)()
    assert L.wd_inner_plan(None, 5, wd.LINK18, plan) == wd.EINVAL
    assert L.wd_set_residual_history(None, None, 0) == wd.EINVAL
    hdr = open(os.path.join(ROOT, "include", "wd.h")).read()
    assert "WD_PLAN_N = 4" in hdr and len(wd.HOP_KERNEL_NAMES) == 3

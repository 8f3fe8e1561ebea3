"""Thin Python binding of the C-ABI library declared in include/wd.h (same names, argument
marshalling only).  PyTorch supplies device memory and the CUDA stream; every step of the hot
path runs in the library's CUDA kernels.  There is no CPU fallback: if libwd.so is missing or
cannot be loaded, importing this module's `lib()` raises.

    ctx = Context(dims, kappa, bc=BC_SF, max_rhs=5)
    ctx.set_gauge(U_canon)                       # torch.float64 cuda tensor [4,T,Lz,Ly,Lx,3,3,2]
    Phi = ctx.pack(Phi_canon)                    # native fp64 block
    X, info = ctx.solve_block(OP_D, Phi, tol=1e-12)
    Y, info = ctx.solve_block(OP_DDAG, X, tol=1e-12)
    F = ctx.force(X, Y)                          # canonical [4,T,Lz,Ly,Lx,3,3,2]
"""
from __future__ import annotations

import ctypes
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libwd.so")

OK, EINVAL, ENOMEM, ECUDA, ENOCONV, ESTATE = 0, -1, -2, -3, -4, -5
BC_PERIODIC, BC_SF = 0, 1
OP_D, OP_DDAG = 0, 1
F64, F32, F32P = 0, 1, 2
LINK18, LINK12 = 0, 1
ORDER_LINEAR, ORDER_TILED = 0, 1
ACTION_FULL, ACTION_EO = 0, 1
PARITY_EVEN, PARITY_ODD, PARITY_BOTH = 0, 1, 2
MAX_RHS = 16
OPT_HOP32_SITES, OPT_HOP64_SITES, OPT_HOP32_REGS, OPT_HOP64_REGS, OPT_POLL_EVERY, OPT_HOP_IMPL, OPT_ALTERNATE_SWEEP, OPT_HOP_ROWS, OPT_SOLVER, OPT_PAIRED, OPT_GRAPH, OPT_MERGE = 0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11
SOLVER_DC_F32, SOLVER_RELIABLE_H16, SOLVER_GL_FLEX, SOLVER_GL_F64, SOLVER_BL_F64 = 0, 1, 2, 3, 4
PROF_NAMES = ("hop32", "hop64", "blas", "force", "layout")
PROF_N = len(PROF_NAMES)

# every symbol include/wd.h declares (tests check that the library exports each one)
SYMBOLS = ["wd_create", "wd_destroy", "wd_site_order", "wd_workspace_bytes", "wd_set_workspace",
           "wd_set_option", "wd_get_option", "wd_set_gauge", "wd_native_bytes", "wd_pack", "wd_unpack", "wd_apply", "wd_hop",
           "wd_solve_block", "wd_force", "wd_md_force_host", "wd_md_force_host_gauge", "wd_refresh", "wd_action",
           "wd_project_parity", "wd_md_force", "wd_profile", "wd_profile_read", "wd_launch_count", "wd_strerror",
           "wd_last_error", "wd_version", "wd_action_static", "wd_action_static_error", "wd_inner_plan", "wd_set_residual_history"]
HOP_KERNEL_NAMES = ("register", "ring", "zmarch")   # WD_HOP_KERNEL_*
STATIC_MAX_ROWS = 1 << 25          # WD_STATIC_MAX_ROWS
STATIC_SCRATCH_BYTES = 2097408     # WD_STATIC_SCRATCH_BYTES


class SolveInfo(ctypes.Structure):
    _fields_ = [("n_rhs", ctypes.c_int), ("outer_steps", ctypes.c_int),
                ("inner_iters_total", ctypes.c_int), ("converged", ctypes.c_int),
                ("relres", ctypes.c_double * MAX_RHS), ("bnorm", ctypes.c_double * MAX_RHS),
                ("seconds", ctypes.c_double)]

    def as_dict(self):
        n = self.n_rhs
        return dict(n_rhs=n, outer_steps=self.outer_steps, inner_iters_total=self.inner_iters_total,
                    converged=bool(self.converged), relres=[self.relres[i] for i in range(n)],
                    bnorm=[self.bnorm[i] for i in range(n)], seconds=self.seconds)


class WdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"wd error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libwd.so (built by paper_1009_5169_b200.build).  Raises if it is absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1009_5169_b200.build` "
                           "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, ci, cd, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    ip = ctypes.POINTER(ctypes.c_int)
    L.wd_create.argtypes = [ctypes.POINTER(vp), ip, cd, ci, ci, vp]
    L.wd_destroy.argtypes = [vp]
    L.wd_site_order.argtypes = [vp, ci, ip]
    L.wd_set_option.argtypes = [vp, ci, ci]
    L.wd_get_option.argtypes = [vp, ci, ip]
    L.wd_workspace_bytes.argtypes = [vp]
    L.wd_workspace_bytes.restype = sz
    L.wd_set_workspace.argtypes = [vp, vp, sz]
    L.wd_set_gauge.argtypes = [vp, vp]
    L.wd_native_bytes.argtypes = [vp, ci, ci]
    L.wd_native_bytes.restype = sz
    L.wd_pack.argtypes = [vp, ci, ci, vp, vp]
    L.wd_unpack.argtypes = [vp, ci, ci, vp, vp]
    L.wd_apply.argtypes = [vp, ci, ci, ci, ci, vp, vp]
    L.wd_hop.argtypes = [vp, ci, ci, ci, ci, ci, vp, vp]
    L.wd_solve_block.argtypes = [vp, ci, ci, vp, vp, cd, ci, ci, cd, ci, ctypes.POINTER(SolveInfo)]
    L.wd_force.argtypes = [vp, ci, vp, vp, vp]
    L.wd_md_force_host.argtypes = [vp, ci, vp, vp, cd, ci, ci, cd, ci, ctypes.POINTER(SolveInfo)]
    L.wd_md_force_host_gauge.argtypes = [vp, ci, vp, vp, vp, cd, ci, ci, cd, ci, ctypes.POINTER(SolveInfo)]
    L.wd_refresh.argtypes = [vp, ci, ci, vp, vp]
    L.wd_action.argtypes = [vp, ci, ci, vp, ctypes.POINTER(cd)]
    L.wd_project_parity.argtypes = [vp, ci, ci, ci, vp]
    L.wd_md_force.argtypes = [vp, ci, ci, vp, vp, vp, vp, ctypes.POINTER(cd), cd, ci, ci, cd, ci, ctypes.POINTER(SolveInfo)]
    L.wd_profile.argtypes = [vp, ci]
    L.wd_profile_read.argtypes = [vp, ctypes.POINTER(cd), ctypes.POINTER(ctypes.c_longlong)]
    L.wd_launch_count.argtypes = [vp]
    L.wd_launch_count.restype = ctypes.c_longlong
    L.wd_strerror.argtypes = [ci]
    L.wd_strerror.restype = ctypes.c_char_p
    L.wd_last_error.argtypes = [vp]
    L.wd_last_error.restype = ctypes.c_char_p
    L.wd_version.restype = ctypes.c_char_p
    if b"MEASUREMENT BUILD" in L.wd_version() and os.environ.get("WD_ALLOW_MEASUREMENT_BUILD") != "1":
        raise RuntimeError(f"{LIB_PATH} is a measurement build ({L.wd_version().decode()}): its results are wrong on purpose. "
                           "Rebuild with `python -m paper_1009_5169_b200.build --force` (WD_NVCC_DEFINES unset), or set "
                           "WD_ALLOW_MEASUREMENT_BUILD=1 for a timing run")
    L.wd_set_residual_history.argtypes = [vp, vp, ci]
    L.wd_set_residual_history.restype = ci
    L.wd_inner_plan.argtypes = [vp, ci, ci, ip]
    L.wd_inner_plan.restype = ci
    L.wd_action_static.argtypes = [ci, sz, vp, vp, vp]
    L.wd_action_static.restype = ci
    L.wd_action_static_error.restype = ctypes.c_char_p
    for name in ("wd_create", "wd_destroy", "wd_site_order", "wd_set_option", "wd_get_option", "wd_set_workspace", "wd_set_gauge", "wd_pack",
                 "wd_unpack", "wd_apply", "wd_hop", "wd_solve_block", "wd_force", "wd_md_force_host", "wd_md_force_host_gauge", "wd_refresh", "wd_action",
           "wd_project_parity", "wd_md_force", "wd_profile",
                 "wd_profile_read"):
        getattr(L, name).restype = ci
    _lib = L
    return L


def _dims(dims):
    return (ctypes.c_int * 4)(*[int(d) for d in dims])


def action_static(X_native, n_rhs, parity_sel=PARITY_BOTH, out=None, stream=None):
    """wd_action_static: per-column |x_i|^2 of a native fp64 block WITHOUT a Context -- for callers that cannot
    allocate device memory (all of it is in their own arena, or a cudaMalloc would stall their other streams).  The
    library allocates nothing: its scratch is a fixed array inside libwd.so, which limits the input to
    STATIC_MAX_ROWS * n_rhs complex numbers and means two calls that overlap on the GPU race (calls on one stream are
    fine).  `out` is the caller's n_rhs-double CUDA tensor (made here with torch only if omitted); the result is
    stream-ordered on `stream` (default: torch's current stream), nothing is synchronised or copied to the host.
    parity_sel picks the even half, the odd half or the whole block, as in Context.action."""
    assert X_native.is_cuda and X_native.dtype == torch.float64 and X_native.is_contiguous()
    n = int(n_rhs)
    total = X_native.numel() // 2   # complex numbers in the whole block
    half = total // 2
    offset, count = {PARITY_BOTH: (0, total), PARITY_EVEN: (0, half), PARITY_ODD: (half, half)}[int(parity_sel)]
    if out is None:
        out = torch.empty(n, dtype=torch.float64, device=X_native.device)
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= n
    if stream is None:
        stream = torch.cuda.current_stream(X_native.device)
    L = lib()
    with torch.cuda.device(X_native.device):   # the library uses the current device's copy of its scratch array
        rc = L.wd_action_static(n, count, ctypes.c_void_p(X_native.data_ptr() + 16 * offset),
                                ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(stream.cuda_stream))
    if rc != OK:
        raise WdError(rc, f"{L.wd_strerror(rc).decode()}: {L.wd_action_static_error().decode()}")
    return out


class Context:
    """Owns a wd_ctx and the torch workspace tensor it points into."""

    def __init__(self, dims, kappa, bc=BC_SF, max_rhs=5, device="cuda:0", order=ORDER_LINEAR, tile=None,
                 stream=None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1009_5169_b200 needs a CUDA device (no CPU fallback)")
        self.L = lib()
        self.dims = tuple(int(d) for d in dims)
        self.kappa = float(kappa)
        self.bc = int(bc)
        self.max_rhs = int(max_rhs)
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = ctypes.c_void_p()
        rc = self.L.wd_create(ctypes.byref(self._h), _dims(self.dims), self.kappa, self.bc, self.max_rhs,
                              ctypes.c_void_p(self.stream.cuda_stream))
        if rc != OK:
            raise WdError(rc, self.L.wd_strerror(rc).decode())
        if order != ORDER_LINEAR:
            self._check(self.L.wd_site_order(self._h, int(order), _dims(tile)))
        nbytes = int(self.L.wd_workspace_bytes(self._h))
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        aligned = (base + 255) // 256 * 256
        self._check(self.L.wd_set_workspace(self._h, ctypes.c_void_p(aligned), nbytes))
        self.V = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]

    # -- helpers ------------------------------------------------------------------------------
    def _check(self, rc, allow=()):
        if rc != OK and rc not in allow:
            raise WdError(rc, f"{self.L.wd_strerror(rc).decode()}: {self.L.wd_last_error(self._h).decode()}")
        return rc

    def close(self):
        if self._h:
            self.stream.synchronize()
            self.L.wd_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @staticmethod
    def _ptr(t):
        return ctypes.c_void_p(t.data_ptr())

    def _canon_spinor_check(self, t):
        lx, ly, lz, lt = self.dims
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
        assert tuple(t.shape[1:]) == (lt, lz, ly, lx, 4, 3, 2), t.shape
        return int(t.shape[0])

    def native_numel(self, prec, n_rhs):
        return int(self.L.wd_native_bytes(self._h, int(prec), int(n_rhs))) // (8 if prec == F64 else 4)

    def empty_native(self, prec, n_rhs):
        """Uninitialised native full-lattice block: flat tensor of reals with attribute n_rhs."""
        t = torch.empty(self.native_numel(prec, n_rhs), dtype=torch.float64 if prec == F64 else torch.float32,
                        device=self.device)
        return t

    # -- the calls of include/wd.h ---------------------------------------------------------------
    def set_gauge(self, U):
        lx, ly, lz, lt = self.dims
        assert U.is_cuda and U.dtype == torch.float64 and U.is_contiguous()
        assert tuple(U.shape) == (4, lt, lz, ly, lx, 3, 3, 2), U.shape
        self._check(self.L.wd_set_gauge(self._h, self._ptr(U)))

    def pack(self, canon, prec=F64):
        n = self._canon_spinor_check(canon)
        out = self.empty_native(prec, n)
        self._check(self.L.wd_pack(self._h, int(prec), n, self._ptr(canon), self._ptr(out)))
        return out

    def unpack(self, native, n_rhs, prec=F64):
        lx, ly, lz, lt = self.dims
        out = torch.empty((n_rhs, lt, lz, ly, lx, 4, 3, 2), dtype=torch.float64, device=self.device)
        self._check(self.L.wd_unpack(self._h, int(prec), int(n_rhs), self._ptr(native), self._ptr(out)))
        return out

    def apply(self, op, native_in, n_rhs, prec=F64, recon=LINK18, out=None):
        if out is None:
            out = torch.empty_like(native_in)
        self._check(self.L.wd_apply(self._h, int(op), int(prec), int(recon), int(n_rhs), self._ptr(native_in),
                                    self._ptr(out)))
        return out

    def hop(self, op, half_in, n_rhs, out_parity, prec=F64, recon=LINK18, out=None):
        if out is None:
            out = torch.empty_like(half_in)
        self._check(self.L.wd_hop(self._h, int(op), int(prec), int(recon), int(n_rhs), int(out_parity),
                                  self._ptr(half_in), self._ptr(out)))
        return out

    def solve_block(self, op, Phi_native, n_rhs, tol=1e-12, max_outer=20, max_inner=1000, inner_tol=0.0,
                    recon=LINK18, out=None, raise_on_noconv=True):
        if out is None:
            out = torch.empty_like(Phi_native)
        info = SolveInfo()
        rc = self.L.wd_solve_block(self._h, int(op), int(n_rhs), self._ptr(Phi_native), self._ptr(out), float(tol),
                                   int(max_outer), int(max_inner), float(inner_tol), int(recon), ctypes.byref(info))
        self._check(rc, allow=() if raise_on_noconv else (ENOCONV,))
        return out, info.as_dict()

    def force(self, X_native, Y_native, n_rhs, F=None):
        lx, ly, lz, lt = self.dims
        if F is None:
            F = torch.zeros((4, lt, lz, ly, lx, 3, 3, 2), dtype=torch.float64, device=self.device)
        self._check(self.L.wd_force(self._h, int(n_rhs), self._ptr(X_native), self._ptr(Y_native), self._ptr(F)))
        return F

    def md_force_host(self, Phi_host, F_host=None, tol=1e-12, max_outer=20, max_inner=1000, inner_tol=0.0,
                      recon=LINK18):
        """Whole MD force evaluation from HOST (ideally pinned) canonical tensors."""
        lx, ly, lz, lt = self.dims
        assert (not Phi_host.is_cuda) and Phi_host.dtype == torch.float64 and Phi_host.is_contiguous()
        n = int(Phi_host.shape[0])
        if F_host is None:
            F_host = torch.empty((4, lt, lz, ly, lx, 3, 3, 2), dtype=torch.float64).pin_memory()
        infos = (SolveInfo * 2)()
        rc = self.L.wd_md_force_host(self._h, n, self._ptr(Phi_host), self._ptr(F_host), float(tol), int(max_outer),
                                     int(max_inner), float(inner_tol), int(recon), infos)
        self._check(rc)
        return F_host, [infos[0].as_dict(), infos[1].as_dict()]

    def md_force_host_gauge(self, U_host, Phi_host, F_host=None, tol=1e-12, max_outer=20, max_inner=1000, inner_tol=0.0,
                            recon=LINK18):
        """Whole MD force evaluation from HOST canonical tensors including the gauge field (upload + ingest)."""
        lx, ly, lz, lt = self.dims
        assert (not Phi_host.is_cuda) and Phi_host.dtype == torch.float64 and Phi_host.is_contiguous()
        assert (not U_host.is_cuda) and U_host.dtype == torch.float64 and U_host.is_contiguous()
        assert tuple(U_host.shape) == (4, lt, lz, ly, lx, 3, 3, 2), U_host.shape
        n = int(Phi_host.shape[0])
        if F_host is None:
            F_host = torch.empty((4, lt, lz, ly, lx, 3, 3, 2), dtype=torch.float64).pin_memory()
        infos = (SolveInfo * 2)()
        rc = self.L.wd_md_force_host_gauge(self._h, n, self._ptr(U_host), self._ptr(Phi_host), self._ptr(F_host), float(tol),
                                           int(max_outer), int(max_inner), float(inner_tol), int(recon), infos)
        self._check(rc)
        return F_host, [infos[0].as_dict(), infos[1].as_dict()]

    def refresh(self, eta_native, n_rhs, variant=ACTION_FULL, out=None):
        """phi = D eta (ACTION_FULL) or phi_e = Dhat eta_e, phi_o = 0 (ACTION_EO); native fp64 blocks."""
        if out is None:
            out = torch.empty_like(eta_native)
        self._check(self.L.wd_refresh(self._h, int(variant), int(n_rhs), self._ptr(eta_native), self._ptr(out)))
        return out

    def action(self, X_native, n_rhs, parity_sel=PARITY_BOTH):
        """Per-column |x_i|^2 over the selected sites, as a list of floats (synchronises)."""
        S = (ctypes.c_double * int(n_rhs))()
        self._check(self.L.wd_action(self._h, int(n_rhs), int(parity_sel), self._ptr(X_native), S))
        return [S[i] for i in range(int(n_rhs))]

    def project_parity(self, native, n_rhs, parity, prec=F64):
        """In place: zero the sites of the other parity."""
        self._check(self.L.wd_project_parity(self._h, int(prec), int(n_rhs), int(parity), self._ptr(native)))
        return native

    def md_force(self, Phi_native, n_rhs, variant=ACTION_FULL, F=None, tol=1e-12, max_outer=20, max_inner=1000,
                 inner_tol=0.0, recon=LINK18, want_action=True):
        """Algorithm 2 on device-resident fields: returns (X, Y, F, S per column or None, [info_X, info_Y])."""
        lx, ly, lz, lt = self.dims
        if F is None:
            F = torch.zeros((4, lt, lz, ly, lx, 3, 3, 2), dtype=torch.float64, device=self.device)
        X = torch.empty_like(Phi_native)
        Y = torch.empty_like(Phi_native)
        S = (ctypes.c_double * int(n_rhs))() if want_action else None
        infos = (SolveInfo * 2)()
        rc = self.L.wd_md_force(self._h, int(variant), int(n_rhs), self._ptr(Phi_native), self._ptr(X), self._ptr(Y),
                                self._ptr(F), S, float(tol), int(max_outer), int(max_inner), float(inner_tol), int(recon),
                                infos)
        self._check(rc)
        return X, Y, F, ([S[i] for i in range(int(n_rhs))] if want_action else None), [infos[0].as_dict(), infos[1].as_dict()]

    def profile(self, enable=True):
        self._check(self.L.wd_profile(self._h, 1 if enable else 0))

    def profile_read(self):
        """{class name: (milliseconds, launch groups)} since the previous read; synchronises."""
        ms = (ctypes.c_double * PROF_N)()
        cnt = (ctypes.c_longlong * PROF_N)()
        self._check(self.L.wd_profile_read(self._h, ms, cnt))
        return {name: (ms[i], int(cnt[i])) for i, name in enumerate(PROF_NAMES)}

    def set_option(self, key, value):
        self._check(self.L.wd_set_option(self._h, int(key), int(value)))

    def get_option(self, key):
        v = ctypes.c_int()
        self._check(self.L.wd_get_option(self._h, int(key), ctypes.byref(v)))
        return v.value

    def set_residual_history(self, hist):
        """wd_set_residual_history: `hist` is a CUDA float64 tensor [capacity, MAX_RHS] (kept alive here), or None to
        switch the record off.  After a solve, hist[:info['inner_iters_total'], :n_rhs] is the residual curve per column."""
        if hist is None:
            self._check(self.L.wd_set_residual_history(self._h, None, 0))
        else:
            assert hist.is_cuda and hist.dtype == torch.float64 and hist.is_contiguous() and hist.shape[1] == MAX_RHS
            self._check(self.L.wd_set_residual_history(self._h, self._ptr(hist), int(hist.shape[0])))
        self._hist = hist

    def inner_plan(self, n_rhs, recon=LINK18):
        """What the fp32 inner solver will run for (n_rhs, recon) under the current options (wd_inner_plan)."""
        plan = (ctypes.c_int * 4)()
        self._check(self.L.wd_inner_plan(self._h, int(n_rhs), int(recon), plan))
        return dict(hop_kernel=HOP_KERNEL_NAMES[plan[0]], merged=bool(plan[1]), paired=bool(plan[2]),
                    kernels_per_iter=int(plan[3]))

    def launch_count(self):
        return int(self.L.wd_launch_count(self._h))

"""ctypes loader for the fp64 CPU oracle (oracle/wd_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  The product (paper_1009_5169_b200) never does.  Argument marshalling for everything in
wd_oracle.cpp, which cites the passages it follows; two functions hold arithmetic of their own in numpy, both pinned
in tests/test_oracle_pins.py: action() (a sum of squares, eq. 2.2) and eo_md_force() (a composition of the pinned
solve, project_parity and force for the even/odd-preconditioned action).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wd_oracle.cpp")
_LIB = os.path.join(_HERE, "libwd_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile wd_oracle.cpp with g++ (OpenMP over sites, as the paper's CPU code)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-fopenmp", "-fcx-limited-range", "-fPIC", "-shared", "-std=c++17",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        L.orc_max_threads.restype = ctypes.c_int
        L.orc_set_threads.argtypes = [ctypes.c_int]
        L.orc_gamma.argtypes = [ctypes.c_int, dp]
        L.orc_apply.argtypes = [ip, ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp]
        L.orc_solve.argtypes = [ip, ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp,
                                ctypes.c_double, ctypes.c_int, dp, ip]
        L.orc_solve_cgne.argtypes = L.orc_solve.argtypes
        L.orc_project_parity.argtypes = [ip, ctypes.c_int, ctypes.c_int, dp, dp]
        L.orc_force.argtypes = [ip, ctypes.c_double, ctypes.c_int, ctypes.c_int, dp, dp, dp, dp]
        L.orc_dense_dim.argtypes = [ip, ctypes.c_int]
        L.orc_dense_dim.restype = ctypes.c_long
        L.orc_dense_matrix.argtypes = [ip, ctypes.c_double, ctypes.c_int, ctypes.c_int, dp, dp]
        L.orc_lu_solve.argtypes = [ctypes.c_long, dp, dp, ctypes.c_int]
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _dims(dims):
    return (ctypes.c_int * 4)(*[int(d) for d in dims])


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def max_threads() -> int:
    return int(lib().orc_max_threads())


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def gamma(mu: int) -> np.ndarray:
    """gamma_mu for mu = 0..3 (x,y,z,t), gamma5 for mu = 4, as a complex [4][4] array."""
    out = np.zeros((4, 4, 2), dtype=np.float64)
    rc = lib().orc_gamma(int(mu), _dp(out))
    assert rc == 0
    return out[..., 0] + 1j * out[..., 1]


def apply(dims, kappa, bc, dag, U, psi) -> np.ndarray:
    """D psi (dag=0) or D^dag psi (dag=1) on a canonical block [n_rhs][T][Lz][Ly][Lx][4][3][2]."""
    U = _f64(U)
    psi = _f64(psi)
    n_rhs = psi.shape[0]
    out = np.empty_like(psi)
    rc = lib().orc_apply(_dims(dims), float(kappa), int(bc), int(dag), n_rhs, _dp(U), _dp(psi), _dp(out))
    assert rc == 0
    return out


def solve(dims, kappa, bc, dag, U, B, tol=1e-14, max_iter=5000):
    """Solve D X = B / D^dag X = B.  Returns (X, true relative residuals, iteration counts, rc)."""
    U = _f64(U)
    B = _f64(B)
    n_rhs = B.shape[0]
    X = np.zeros_like(B)
    relres = np.zeros(n_rhs, dtype=np.float64)
    iters = np.zeros(n_rhs, dtype=np.int32)
    rc = lib().orc_solve(_dims(dims), float(kappa), int(bc), int(dag), n_rhs, _dp(U), _dp(B), _dp(X),
                         float(tol), int(max_iter), _dp(relres),
                         iters.ctypes.data_as(ctypes.POINTER(ctypes.c_int)))
    assert rc >= 0
    return X, relres, iters, rc


def solve_cgne(dims, kappa, bc, dag, U, B, tol=1e-14, max_iter=100000):
    """The CG-on-normal-equations fallback of `solve`, on its own.  Same returns as `solve`."""
    U = _f64(U)
    B = _f64(B)
    n_rhs = B.shape[0]
    X = np.zeros_like(B)
    relres = np.zeros(n_rhs, dtype=np.float64)
    iters = np.zeros(n_rhs, dtype=np.int32)
    rc = lib().orc_solve_cgne(_dims(dims), float(kappa), int(bc), int(dag), n_rhs, _dp(U), _dp(B), _dp(X),
                              float(tol), int(max_iter), _dp(relres),
                              iters.ctypes.data_as(ctypes.POINTER(ctypes.c_int)))
    assert rc >= 0
    return X, relres, iters, rc


def project_parity(dims, parity, psi) -> np.ndarray:
    """P_parity psi: the sites with (x+y+z+t) mod 2 == parity kept, the others zero."""
    psi = _f64(psi)
    out = np.empty_like(psi)
    rc = lib().orc_project_parity(_dims(dims), int(parity), psi.shape[0], _dp(psi), _dp(out))
    assert rc == 0
    return out


def action(X) -> np.ndarray:
    """Pseudo-fermion action per column, S_i = |x_i|^2 with x_i = D^-1 phi_i (eq. 2.2)."""
    X = _f64(X)
    return np.sum(X.reshape(X.shape[0], -1) ** 2, axis=1)


def eo_md_force(dims, kappa, bc, U, Phi_e, tol=1e-14):
    """Even/odd-preconditioned-action variant: phi lives on even sites,
    S = sum_i |Dhat^-1 phi_i|^2 with Dhat = 1 - kappa^2 H_eo H_oe the Schur complement of D on the even sites.
    Because D (x_e, kappa H_oe x_e) = (Dhat x_e, 0), Dhat^-1 phi_e = P_e D^-1 (phi_e, 0); so with
        X = D^-1 (phi_e, 0),   Y = D^dag^-1 (P_e X),
    S_i = |P_e x_i|^2 and dS = -2 Re(y^dag dD x): the SAME functional f[x, y] as the full action.  Composition of the
    pinned pieces only.  Returns (X, Y, S per column, F)."""
    Phi = project_parity(dims, 0, Phi_e)
    X, r1, _, rc1 = solve(dims, kappa, bc, 0, U, Phi, tol=tol)
    Xe = project_parity(dims, 0, X)
    Y, r2, _, rc2 = solve(dims, kappa, bc, 1, U, Xe, tol=tol)
    assert rc1 == 0 and rc2 == 0, (r1, r2)
    return X, Y, action(Xe), force(dims, kappa, bc, U, X, Y)


def force(dims, kappa, bc, U, X, Y, F=None) -> np.ndarray:
    """F += sum_i f[x_i, y_i]; F canonical [4][T][Lz][Ly][Lx][3][3][2] (allocated as zero if None)."""
    U = _f64(U)
    X = _f64(X)
    Y = _f64(Y)
    if F is None:
        F = np.zeros(U.shape, dtype=np.float64)
    assert F.dtype == np.float64 and F.flags["C_CONTIGUOUS"]
    rc = lib().orc_force(_dims(dims), float(kappa), int(bc), X.shape[0], _dp(U), _dp(X), _dp(Y), _dp(F))
    assert rc == 0
    return F


def dense_matrix(dims, kappa, bc, dag, U) -> np.ndarray:
    """The dynamical block of D (or D^dag) as a complex [N][N] array, built from unit vectors."""
    U = _f64(U)
    n = int(lib().orc_dense_dim(_dims(dims), int(bc)))
    A = np.zeros((n, n, 2), dtype=np.float64)
    rc = lib().orc_dense_matrix(_dims(dims), float(kappa), int(bc), int(dag), _dp(U), _dp(A))
    assert rc == 0
    return A[..., 0] + 1j * A[..., 1]


def lu_solve(A: np.ndarray, b: np.ndarray) -> np.ndarray:
    """Solve A x = b with the oracle's own partial-pivot LU.  A complex [N][N]; b complex [nrhs][N]."""
    n = A.shape[0]
    Ar = np.ascontiguousarray(np.stack([A.real, A.imag], axis=-1), dtype=np.float64)
    br = np.ascontiguousarray(np.stack([b.real, b.imag], axis=-1), dtype=np.float64)
    rc = lib().orc_lu_solve(n, _dp(Ar), _dp(br), int(b.shape[0]))
    assert rc == 0, "singular matrix"
    return br[..., 0] + 1j * br[..., 1]

"""Seeded synthetic inputs for the Wilson-Dirac hot path (BASELINE.json configs).

This module is the ONLY code shared by the oracle side (``oracle/``) and the CUDA side
(``paper_1009_5169_b200/``).  It holds none of the method's arithmetic: no Dirac operator, no
solver, no force.  It produces, on the host in fp64 numpy,

* gauge links ``U = exp(i eps H)`` with ``H = sum_a eta_a lambda_a / 2`` Gaussian Hermitian
  traceless, reunitarised (configs[0]: "links = exp(i eps H) with H Gaussian Hermitian traceless,
  eps=0.2, reunitarised"), spatial links on the t=0 slice set to the identity in SF mode;
* right-hand sides: unit Gaussian complex spinors (4 spin x 3 colour), zero on t=0 in SF mode;
* the named configurations of BASELINE.json.

They stand in for the paper's thermalised 16^4, beta=4.52, kappa=0.15805 configuration
(PAPER.md:96), which is not available.

Random numbers come from a counter-based generator keyed by (seed, stream, index), so a field does
not depend on loop order, chunking or thread count.

Canonical layouts (what both sides receive):
  gauge   float64 [mu=4][T][Lz][Ly][Lx][3][3][2]   row-major colour matrix, (re, im)
  spinor  float64 [n_rhs][T][Lz][Ly][Lx][4][3][2]   spin, colour, (re, im)
with mu = 0,1,2,3 = x,y,z,t and dims = (Lx, Ly, Lz, T).
"""
from __future__ import annotations

import numpy as np

BC_PERIODIC = 0
BC_SF = 1

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLD = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)
_C3 = np.uint64(0xD1B54A32D192ED03)

STREAM_LINKS = 0
STREAM_RHS = 1
STREAM_AUX = 2  # gauge transformations, probe directions etc. used by tests


def _mix64(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on uint64 arrays (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * _C1
        z = (z ^ (z >> np.uint64(27))) * _C2
        return z ^ (z >> np.uint64(31))


def uniform_pair(seed: int, stream: int, index: np.ndarray):
    """Two independent uniforms in (0,1) per counter ``index`` (uint64 array)."""
    index = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        key = _mix64(np.uint64(seed) * _GOLD + np.uint64(stream) * _C3 + np.uint64(1))
        a = _mix64(key + index * _GOLD)
        b = _mix64(a ^ _C3)
    scale = 1.0 / 9007199254740992.0  # 2^-53
    u1 = ((a >> np.uint64(11)).astype(np.float64) + 0.5) * scale
    u2 = ((b >> np.uint64(11)).astype(np.float64) + 0.5) * scale
    return u1, u2


def normal_pair(seed: int, stream: int, index: np.ndarray):
    """Two independent N(0,1) per counter (Box-Muller)."""
    u1, u2 = uniform_pair(seed, stream, index)
    r = np.sqrt(-2.0 * np.log(u1))
    ang = 2.0 * np.pi * u2
    return r * np.cos(ang), r * np.sin(ang)


def volume(dims) -> int:
    lx, ly, lz, lt = dims
    return int(lx) * int(ly) * int(lz) * int(lt)


def gell_mann() -> np.ndarray:
    """The eight Gell-Mann matrices, [8][3][3] complex."""
    lam = np.zeros((8, 3, 3), dtype=np.complex128)
    lam[0, 0, 1] = lam[0, 1, 0] = 1
    lam[1, 0, 1] = -1j
    lam[1, 1, 0] = 1j
    lam[2, 0, 0] = 1
    lam[2, 1, 1] = -1
    lam[3, 0, 2] = lam[3, 2, 0] = 1
    lam[4, 0, 2] = -1j
    lam[4, 2, 0] = 1j
    lam[5, 1, 2] = lam[5, 2, 1] = 1
    lam[6, 1, 2] = -1j
    lam[6, 2, 1] = 1j
    lam[7, 0, 0] = lam[7, 1, 1] = 1 / np.sqrt(3.0)
    lam[7, 2, 2] = -2 / np.sqrt(3.0)
    return lam


def su3_exp(a: np.ndarray, terms: int = 40) -> np.ndarray:
    """exp(A) for a batch [...,3,3] by the Taylor series summed to fp64 convergence."""
    out = np.zeros_like(a)
    out[..., 0, 0] = out[..., 1, 1] = out[..., 2, 2] = 1.0
    term = out.copy()
    for k in range(1, terms + 1):
        term = np.matmul(term, a) / k
        out = out + term
        if np.max(np.abs(term)) < 1e-18:
            break
    return out


def reunitarise(u: np.ndarray) -> np.ndarray:
    """Row 1 normalised; row 2 Gram-Schmidt against row 1, normalised; row 3 = conj(row1 x row2)."""
    r1 = u[..., 0, :]
    r1 = r1 / np.linalg.norm(r1, axis=-1, keepdims=True)
    r2 = u[..., 1, :]
    r2 = r2 - r1 * np.sum(np.conj(r1) * r2, axis=-1, keepdims=True)
    r2 = r2 / np.linalg.norm(r2, axis=-1, keepdims=True)
    r3 = np.conj(np.cross(r1, r2))
    return np.stack([r1, r2, r3], axis=-2)


def random_algebra(seed: int, stream: int, count: int, offset: int = 0) -> np.ndarray:
    """``count`` Hermitian traceless matrices H = sum_a eta_a lambda_a / 2, eta_a ~ N(0,1)."""
    idx = (np.arange(count * 8, dtype=np.uint64) + np.uint64(offset * 8))
    eta, _ = normal_pair(seed, stream, idx)
    eta = eta.reshape(count, 8)
    return np.einsum("na,aij->nij", eta, gell_mann() / 2.0)


def random_su3(seed: int, stream: int, count: int, eps: float, offset: int = 0,
               chunk: int = 1 << 18) -> np.ndarray:
    """``count`` SU(3) matrices exp(i eps H), reunitarised; [count][3][3] complex."""
    out = np.empty((count, 3, 3), dtype=np.complex128)
    for lo in range(0, count, chunk):
        hi = min(count, lo + chunk)
        h = random_algebra(seed, stream, hi - lo, offset + lo)
        out[lo:hi] = reunitarise(su3_exp(1j * eps * h))
    return out


def gauge_field(dims, eps: float, seed: int, bc: int = BC_SF) -> np.ndarray:
    """Canonical gauge field, float64 [4][T][Lz][Ly][Lx][3][3][2].

    Link (mu, site) uses counters (mu*V + site)*8 + a of stream 0.  In SF mode the spatial links on
    the t=0 slice are set to the identity afterwards (configs[0]: "boundary spatial links identity").
    """
    lx, ly, lz, lt = (int(d) for d in dims)
    v = lx * ly * lz * lt
    u = random_su3(seed, STREAM_LINKS, 4 * v, eps).reshape(4, lt, lz, ly, lx, 3, 3)
    if bc == BC_SF:
        u[0:3, 0] = np.eye(3, dtype=np.complex128)
    return np.ascontiguousarray(np.stack([u.real, u.imag], axis=-1))


def unit_gauge(dims) -> np.ndarray:
    lx, ly, lz, lt = (int(d) for d in dims)
    u = np.zeros((4, lt, lz, ly, lx, 3, 3, 2), dtype=np.float64)
    for a in range(3):
        u[..., a, a, 0] = 1.0
    return u


def spinor_field(dims, n_rhs: int, seed: int, bc: int = BC_SF, stream: int = STREAM_RHS) -> np.ndarray:
    """Canonical block of right-hand sides, float64 [n_rhs][T][Lz][Ly][Lx][4][3][2].

    re, im ~ N(0,1) independently from counter (rhs*V + site)*12 + (spin*3 + colour); zero on t=0
    in SF mode.
    """
    lx, ly, lz, lt = (int(d) for d in dims)
    v = lx * ly * lz * lt
    idx = np.arange(n_rhs * v * 12, dtype=np.uint64)
    re, im = normal_pair(seed, stream, idx)
    phi = np.stack([re, im], axis=-1).reshape(n_rhs, lt, lz, ly, lx, 4, 3, 2)
    if bc == BC_SF:
        phi[:, 0] = 0.0
    return np.ascontiguousarray(phi)


def to_complex(a: np.ndarray) -> np.ndarray:
    """View a (..., 2) float64 array as complex128 (...)."""
    a = np.ascontiguousarray(a)
    return a.view(np.complex128)[..., 0]


def from_complex(c: np.ndarray) -> np.ndarray:
    c = np.ascontiguousarray(c, dtype=np.complex128)
    return np.ascontiguousarray(np.stack([c.real, c.imag], axis=-1))


# BASELINE.json `configs`, made concrete.  seed 1 throughout.
CONFIGS = {
    0: dict(name="4^3x4 SF", dims=(4, 4, 4, 4), eps=0.2, kappa=0.125, n_rhs=5, seed=1, bc=BC_SF),
    1: dict(name="8^3x8 SF", dims=(8, 8, 8, 8), eps=0.3, kappa=0.13, n_rhs=5, seed=1, bc=BC_SF),
    2: dict(name="12^3x12 SF", dims=(12, 12, 12, 12), eps=0.4, kappa=0.135, n_rhs=5, seed=1, bc=BC_SF),
    3: dict(name="16^3x16 SF", dims=(16, 16, 16, 16), eps=0.4, kappa=0.135, n_rhs=5, seed=1, bc=BC_SF),
    4: dict(name="24^3x24 SF", dims=(24, 24, 24, 24), eps=0.4, kappa=0.135, n_rhs=5, seed=1, bc=BC_SF),
}


def make_config(idx: int, n_rhs: int | None = None):
    """(cfg dict, U canonical, Phi canonical) for BASELINE.json configs[idx]."""
    cfg = dict(CONFIGS[idx])
    if n_rhs is not None:
        cfg["n_rhs"] = int(n_rhs)
    u = gauge_field(cfg["dims"], cfg["eps"], cfg["seed"], cfg["bc"])
    phi = spinor_field(cfg["dims"], cfg["n_rhs"], cfg["seed"], cfg["bc"])
    return cfg, u, phi

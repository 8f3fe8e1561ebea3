"""The merged-update schedule of the fp32 inner solver (csrc/wd_solve.cu, WD_OPT_MERGE) restated in
numpy and checked against textbook BiCGStab on a random well-conditioned system: same iterates in fp64, and in fp32 the
recursive residual falls to the fp32 floor in as many iterations.  CPU only: this pins the recurrence the kernels implement, not the kernels."""
import numpy as np


def system(n=96, seed=3, dtype=np.complex128):
    rng = np.random.default_rng(seed)
    A = np.eye(n) + 0.35 * (rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))) / np.sqrt(n)
    b = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    return A.astype(dtype), (b / np.linalg.norm(b)).astype(dtype)


def textbook(A, b, iters, floor=0.0):
    x = np.zeros_like(b); r = b.copy(); rt = b.copy(); p = np.zeros_like(b); v = np.zeros_like(b)
    rho = np.vdot(rt, r); alpha = omega = 1.0; beta = 0.0
    hist = []
    for _ in range(iters):
        p = r + beta * (p - omega * v)
        v = A @ p
        alpha = rho / np.vdot(rt, v)
        s = r - alpha * v
        t = A @ s
        omega = np.vdot(t, s) / np.vdot(t, t)
        x = x + alpha * p + omega * s
        r = s - omega * t
        rho1 = np.vdot(rt, r)
        beta = (rho1 / rho) * (alpha / omega)
        rho = rho1
        hist.append((x.copy(), np.linalg.norm(r)))
        if hist[-1][1] <= floor:
            break
    return hist


def merged(A, b, iters, keep_rts=True, floor=0.0):
    """p starts as r; rho' comes from <rt,s> - omega <rt,t> (both available when t is), so that the new p is formed in the
    same pass as the new r."""
    x = np.zeros_like(b); r = b.copy(); rt = b.copy(); p = r.copy()
    rho = np.vdot(rt, r)
    hist = []
    for _ in range(iters):
        v = A @ p
        alpha = rho / np.vdot(rt, v)
        s = r - alpha * v
        t = A @ s
        omega = np.vdot(t, s) / np.vdot(t, t)
        rho1 = (np.vdot(rt, s) if keep_rts else 0.0) - omega * np.vdot(rt, t)
        beta = (rho1 / rho) * (alpha / omega)
        rho = rho1
        x = x + alpha * p + omega * s          # one pass: x, r, p
        r = s - omega * t
        p = r + beta * (p - omega * v)
        hist.append((x.copy(), np.linalg.norm(r)))
        if hist[-1][1] <= floor:
            break
    return hist


def test_merged_schedule_reproduces_textbook_bicgstab_in_fp64():
    A, b = system()
    h0, h1 = textbook(A, b, 30, floor=1e-13), merged(A, b, 30, floor=1e-13)
    for (x0, r0), (x1, r1) in zip(h0, h1):
        if r0 < 1e-11:
            break   # at the rounding floor the two orders of the same arithmetic drift apart
        assert np.linalg.norm(x0 - x1) <= 1e-8 * np.linalg.norm(x0)
        assert abs(r0 - r1) <= 1e-6 * r0 + 1e-14
    xs = np.linalg.solve(A, b)
    assert np.linalg.norm(h1[-1][0] - xs) < 1e-10 * np.linalg.norm(xs)


def test_merged_schedule_converges_in_fp32_like_the_textbook_order():
    """In fp32 the recursive residual of the merged schedule falls to the fp32 floor in as many iterations as the textbook
    order takes (the <rt,s> term, zero in exact arithmetic, is kept as computed: the kernels do the same)."""
    A, b = system(dtype=np.complex64)
    mg = merged(A, b, 40, keep_rts=True, floor=2e-7)
    tb = textbook(A, b, 40, floor=2e-7)
    assert mg[-1][1] <= 2e-7 and tb[-1][1] <= 2e-7
    assert abs(len(mg) - len(tb)) <= 1
    xs = np.linalg.solve(A.astype(np.complex128), b.astype(np.complex128))
    assert np.linalg.norm(mg[-1][0] - xs) < 1e-5 * np.linalg.norm(xs)

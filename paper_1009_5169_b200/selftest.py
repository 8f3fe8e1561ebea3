"""Run every kernel class of libwd.so once on a small lattice (no oracle: results are only checked for finiteness and
convergence).  Meant for `compute-sanitizer --tool memcheck|racecheck python -m paper_1009_5169_b200.selftest` and as a
quick installation check.

    python -m paper_1009_5169_b200.selftest [--dims 8 4 4 6] [--n-rhs 5]
"""
from __future__ import annotations

import argparse

import torch

import wd_inputs as wi

from . import wd as pkg


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--dims", type=int, nargs=4, default=[8, 4, 4, 6])   # Lx/2 = 4: row-major layout, staged kernels run
    ap.add_argument("--n-rhs", type=int, default=5)
    a = ap.parse_args()
    dims, n, bc, kappa = tuple(a.dims), a.n_rhs, wi.BC_SF, 0.125
    U = torch.from_numpy(wi.gauge_field(dims, 0.3, 1, bc)).cuda()
    Phi = torch.from_numpy(wi.spinor_field(dims, n, 1, bc)).cuda()
    ctx = pkg.Context(dims, kappa, bc=bc, max_rhs=n)
    ctx.set_gauge(U)
    done = []
    for prec in (pkg.F64, pkg.F32):
        P = ctx.pack(Phi, prec)
        for impl in (0, 1, 2):
            ctx.set_option(pkg.OPT_HOP_IMPL, impl)
            for recon in (pkg.LINK18, pkg.LINK12):
                for op in (pkg.OP_D, pkg.OP_DDAG):
                    out = ctx.apply(op, P, n, prec, recon)
                    assert bool(torch.isfinite(out).all())
        assert bool(torch.isfinite(ctx.unpack(P, n, prec)).all())
        done.append(f"apply prec {prec}: 3 hop kernels x 2 link forms x D, D^dag")
    P = ctx.pack(Phi)
    for impl in (0, 1, 2):
        ctx.set_option(pkg.OPT_HOP_IMPL, impl)
        for solver in (pkg.SOLVER_DC_F32, pkg.SOLVER_RELIABLE_H16, pkg.SOLVER_GL_FLEX, pkg.SOLVER_GL_F64, pkg.SOLVER_BL_F64):
            ctx.set_option(pkg.OPT_SOLVER, solver)
            X, info = ctx.solve_block(pkg.OP_D, P, n, tol=1e-12, max_outer=500)
            assert info["converged"], (impl, solver, info)
        done.append(f"hop impl {impl}: 5 solvers")
    ctx.set_option(pkg.OPT_SOLVER, pkg.SOLVER_DC_F32)
    for variant in (pkg.ACTION_FULL, pkg.ACTION_EO):
        phi = ctx.refresh(P, n, variant)
        X, Y, F, S, infos = ctx.md_force(phi, n, variant)
        assert bool(torch.isfinite(F).all()) and all(s > 0 for s in S)
    done.append("refresh + md_force, full and even/odd action")
    Fh, infos = ctx.md_force_host_gauge(U.cpu().pin_memory(), Phi.cpu().pin_memory())
    assert bool(torch.isfinite(Fh).all())
    done.append("md_force_host_gauge")
    launches = ctx.launch_count()
    ctx.close()
    for d in done:
        print("ok:", d)
    print(f"selftest passed: {launches} kernel launches on {dims}, n_rhs = {n}")


if __name__ == "__main__":
    main()

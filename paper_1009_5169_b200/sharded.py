"""RHS-sharded multi-GPU form of the path.

The N_f/2 pseudo-fermion columns are independent ("the force contribution F_mu,i can be computed independently",
PAPER.md:60-64); the paper deals its five equations 2:3 to two GTX 285 cards.  Here: one process per GPU, column i goes
to rank i mod G, the gauge field is replicated, every rank runs Algorithm 2 (wd_md_force) on its columns with the same
kernels, and ONE exchange step follows: allReduce(sum) of F (4 V 18 doubles; NCCL over NVLink / NVSwitch -- every peer at
full bandwidth, so no topology-aware split like the paper's 2:3 is needed) and an all-gather of the per-column actions.
Cost of sharding: each GPU amortises a link over fewer columns.

The collective plumbing is torch.distributed (backend nccl on GPUs; the same code runs over gloo on CPU tensors in
tests/test_sharded_gloo.py, with the per-rank computation injected).  This module holds no arithmetic of the method.
"""
from __future__ import annotations

import torch


def columns_of_rank(n_rhs: int, world: int, rank: int) -> list[int]:
    """Columns dealt round-robin: rank r owns i = r, r + G, r + 2G, ...  (loads differ by at most one column)."""
    return list(range(rank, n_rhs, world))


def max_columns_per_rank(n_rhs: int, world: int) -> int:
    return (n_rhs + world - 1) // world


def allreduce_force(dist, F: torch.Tensor, world: int) -> torch.Tensor:
    """F <- sum over ranks of the per-rank force contributions (Algorithm 2 line 5 across GPUs), in place."""
    if world > 1:
        dist.all_reduce(F, op=dist.ReduceOp.SUM)
    return F


def gather_actions(dist, S_local, cols, n_rhs: int, world: int, device) -> list[float]:
    """Per-column actions of all ranks, in column order."""
    S = torch.zeros(n_rhs, dtype=torch.float64, device=device)
    for s, i in zip(S_local, cols):
        S[i] = float(s)
    if world > 1:
        dist.all_reduce(S, op=dist.ReduceOp.SUM)   # disjoint supports: the sum is the gather
    return [float(x) for x in S.cpu()]


def sharded_md_force(dist, world: int, rank: int, n_rhs: int, local_force, F_shape, device):
    """One MD force evaluation over `world` ranks.  `local_force(cols)` runs Algorithm 2 on this rank's columns and
    returns (F_local tensor of shape F_shape on `device`, list of per-column actions or None); a rank without columns
    contributes zeros.  Returns (F summed over ranks, actions in column order or None)."""
    cols = columns_of_rank(n_rhs, world, rank)
    if cols:
        F, S = local_force(cols)
    else:
        F, S = torch.zeros(F_shape, dtype=torch.float64, device=device), []
    allreduce_force(dist, F, world)
    actions = gather_actions(dist, S, cols, n_rhs, world, device) if S is not None else None
    return F, actions


class ShardedContext:
    """The library context of one rank of an RHS-sharded job: gauge replicated, columns i = rank mod world."""

    def __init__(self, pkg, dist, dims, kappa, bc, n_rhs, world, rank, device):
        self.pkg, self.dist, self.world, self.rank, self.n_rhs = pkg, dist, world, rank, n_rhs
        self.cols = columns_of_rank(n_rhs, world, rank)
        self.device = torch.device(device)
        self.dims = tuple(dims)
        self.ctx = pkg.Context(dims, kappa, bc=bc, max_rhs=max(1, len(self.cols)), device=device) if self.cols else None

    def set_gauge(self, U_dev):
        if self.ctx is not None:
            self.ctx.set_gauge(U_dev)

    def pack_local(self, Phi_canon_dev):
        """Phi_canon_dev: canonical block of ALL columns (replicated input); packs this rank's columns."""
        if self.ctx is None:
            return None
        idx = torch.tensor(self.cols, device=Phi_canon_dev.device)
        return self.ctx.pack(Phi_canon_dev.index_select(0, idx).contiguous())

    def md_force(self, P_local, variant=0, **kw):
        lx, ly, lz, lt = self.dims
        shape = (4, lt, lz, ly, lx, 3, 3, 2)
        infos = []

        def local(cols):
            X, Y, F, S, inf = self.ctx.md_force(P_local, len(cols), variant, **kw)
            infos.extend(inf)
            return F, S

        F, S = sharded_md_force(self.dist, self.world, self.rank, self.n_rhs, local, shape, self.device)
        return F, S, infos

    def close(self):
        if self.ctx is not None:
            self.ctx.close()

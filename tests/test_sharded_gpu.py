"""The RHS-sharded form (paper_1009_5169_b200/sharded.py) with the library's own
kernels as the per-rank compute.  tests/test_sharded_gloo.py covers the deal and the exchange step on CPU with the oracle
injected; here ShardedContext itself runs on a GPU: pack_local's column selection, contexts sized for a rank's own
columns (one or two columns put a rank in the chunk-major layout, max_rhs < 3), a rank that owns no column, and the sum
of the per-rank forces against the unsharded wd_md_force and the oracle.

One GPU is all the test boxes have, so the ranks of a world of G are run ONE AFTER THE OTHER on cuda:0 (they are
independent up to the final sum: no rank ever waits for another) with a stand-in for torch.distributed that records the
tensors handed to all_reduce; the test adds them up itself.  With two or more GPUs the last test runs world size 2 for
real under NCCL."""
import os
import socket
import sys

import numpy as np
import pytest
import torch

import wd_inputs as wi
from oracle import wd_oracle as orc

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _wd():
    import paper_1009_5169_b200 as pkg
    return pkg


class _RecordingDist:
    """all_reduce of a one-rank-at-a-time run: remembers what each rank contributed, leaves the tensor alone."""

    class ReduceOp:
        SUM = "sum"

    def __init__(self):
        self.seen = []

    def all_reduce(self, t, op=None):
        assert op == self.ReduceOp.SUM
        self.seen.append(t.detach().clone())


def _reference(cfg_idx, n):
    cfg, U, Phi = wi.make_config(cfg_idx, n)
    dims, kappa, bc = cfg["dims"], cfg["kappa"], cfg["bc"]
    X, r1, _, rc1 = orc.solve(dims, kappa, bc, 0, U, Phi, tol=1e-14)
    Y, r2, _, rc2 = orc.solve(dims, kappa, bc, 1, U, X, tol=1e-14)
    assert rc1 == 0 and rc2 == 0 and max(r1.max(), r2.max()) < 1e-13
    return cfg, U, Phi, orc.force(dims, kappa, bc, U, X, Y), orc.action(X)


def test_sharded_context_world_1_equals_plain_md_force_and_the_oracle():
    pkg = _wd()
    from paper_1009_5169_b200 import sharded as sh
    n = 5
    cfg, U, Phi, Fr, Sr = _reference(1, n)
    dims, kappa, bc = cfg["dims"], cfg["kappa"], cfg["bc"]
    Ud, Pd = torch.from_numpy(U).cuda(), torch.from_numpy(Phi).cuda()
    sc = sh.ShardedContext(pkg, None, dims, kappa, bc, n, 1, 0, "cuda:0")     # world 1: torch.distributed is never touched
    sc.set_gauge(Ud)
    F, S, infos = sc.md_force(sc.pack_local(Pd), tol=1e-12)
    assert len(infos) == 2 and all(i["converged"] for i in infos)
    ctx = pkg.Context(dims, kappa, bc=bc, max_rhs=n)
    ctx.set_gauge(Ud)
    _, _, F0, S0, _ = ctx.md_force(ctx.pack(Pd), n, tol=1e-12)
    assert torch.equal(F, F0) and S == S0                                     # same kernels, same columns: same bits
    Fn = F.cpu().numpy()
    assert np.linalg.norm(Fn - Fr) / np.linalg.norm(Fr) < 1e-9
    assert np.allclose(S, Sr, rtol=1e-9)
    sc.close()
    ctx.close()


@pytest.mark.parametrize("world", [2, 3, 6])
def test_sharded_context_ranks_run_in_turn_sum_to_the_unsharded_force(world):
    """n_rhs = 5 over 2 ranks (3 + 2 columns, the paper's 2:3 deal), 3 ranks (2 + 2 + 1: every rank in the chunk-major
    layout) and 6 ranks (one column each, the last rank none)."""
    pkg = _wd()
    from paper_1009_5169_b200 import sharded as sh
    n = 5
    cfg, U, Phi, Fr, Sr = _reference(1, n)
    dims, kappa, bc = cfg["dims"], cfg["kappa"], cfg["bc"]
    Ud, Pd = torch.from_numpy(U).cuda(), torch.from_numpy(Phi).cuda()
    F_sum = torch.zeros(U.shape, dtype=torch.float64, device="cuda")
    S_sum = torch.zeros(n, dtype=torch.float64, device="cuda")
    for rank in range(world):
        rec = _RecordingDist()
        sc = sh.ShardedContext(pkg, rec, dims, kappa, bc, n, world, rank, "cuda:0")
        assert sc.cols == sh.columns_of_rank(n, world, rank)
        if sc.cols:
            assert sc.ctx.max_rhs == len(sc.cols)
        else:
            assert sc.ctx is None and sc.pack_local(Pd) is None
        sc.set_gauge(Ud)
        F, S, infos = sc.md_force(sc.pack_local(Pd), tol=1e-12)
        assert len(rec.seen) == 2 and rec.seen[0].shape == F_sum.shape and rec.seen[1].shape == S_sum.shape
        if not sc.cols:
            assert not rec.seen[0].any() and not rec.seen[1].any()            # a rank without columns contributes zeros
        else:
            assert all(i["converged"] for i in infos)
            assert sorted(torch.nonzero(rec.seen[1]).flatten().tolist()) == sc.cols
        F_sum += rec.seen[0]
        S_sum += rec.seen[1]
        sc.close()
    Fn = F_sum.cpu().numpy()
    assert np.linalg.norm(Fn - Fr) / np.linalg.norm(Fr) < 1e-9
    assert np.allclose(S_sum.cpu().numpy(), Sr, rtol=1e-9)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _nccl_worker(rank, world, port, n, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank),
                      LOCAL_RANK=str(rank))
    if ROOT not in sys.path:
        sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import paper_1009_5169_b200 as pkg
    from paper_1009_5169_b200 import sharded as sh
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device(f"cuda:{rank}"))
    cfg, U, Phi = wi.make_config(1, n)
    sc = sh.ShardedContext(pkg, dist, cfg["dims"], cfg["kappa"], cfg["bc"], n, world, rank, f"cuda:{rank}")
    sc.set_gauge(torch.from_numpy(U).cuda())
    F, S, _ = sc.md_force(sc.pack_local(torch.from_numpy(Phi).cuda()), tol=1e-12)
    out[rank] = (F.cpu().numpy(), S)
    sc.close()
    dist.destroy_process_group()


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two GPUs (the test boxes have one)")
def test_sharded_context_world_2_over_nccl():
    import torch.multiprocessing as mp
    n = 5
    _, _, _, Fr, Sr = _reference(1, n)
    out = mp.Manager().dict()
    mp.spawn(_nccl_worker, args=(2, _free_port(), n, out), nprocs=2, join=True)
    for rank in range(2):
        F, S = out[rank]
        assert np.linalg.norm(F - Fr) / np.linalg.norm(Fr) < 1e-9
        assert np.allclose(S, Sr, rtol=1e-9)
    assert np.array_equal(out[0][0], out[1][0])

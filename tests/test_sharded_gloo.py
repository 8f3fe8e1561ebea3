"""RHS-sharded multi-GPU form of the path (paper_1009_5169_b200/sharded.py): columns
dealt round-robin to the ranks, gauge replicated, one allReduce(sum) of F.  Run here with world sizes 2 and 3 on CPU over
gloo; the per-rank Algorithm 2 is the ORACLE's (the kernels need a GPU), so what is tested is the sharding logic: the
deal, the exchange step, and that the sharded force and actions equal the unsharded ones (Alg. 1 = Alg. 2 additivity)."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_rhs, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank),
                      LOCAL_RANK=str(rank))
    from paper_1009_5169_b200 import sharded as sh
    import wd_inputs as wi
    from oracle import wd_oracle as orc
    orc.set_threads(2)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg, U, Phi = wi.make_config(0, n_rhs)
    dims, kappa, bc = cfg["dims"], cfg["kappa"], cfg["bc"]

    def local_force(cols):
        P = np.ascontiguousarray(Phi[cols])
        X, r1, _, rc1 = orc.solve(dims, kappa, bc, 0, U, P, tol=1e-14)
        Y, r2, _, rc2 = orc.solve(dims, kappa, bc, 1, U, X, tol=1e-14)
        assert rc1 == 0 and rc2 == 0
        return torch.from_numpy(orc.force(dims, kappa, bc, U, X, Y)), list(orc.action(X))

    F, S = sh.sharded_md_force(dist, world, rank, n_rhs, local_force, U.shape, "cpu")
    out[rank] = (F.numpy().copy(), S, sh.columns_of_rank(n_rhs, world, rank))
    dist.destroy_process_group()


def _run(world, n_rhs):
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), n_rhs, out), nprocs=world, join=True)
    return [out[r] for r in range(world)]


def _unsharded(n_rhs):
    import wd_inputs as wi
    from oracle import wd_oracle as orc
    cfg, U, Phi = wi.make_config(0, n_rhs)
    dims, kappa, bc = cfg["dims"], cfg["kappa"], cfg["bc"]
    X, _, _, _ = orc.solve(dims, kappa, bc, 0, U, Phi, tol=1e-14)
    Y, _, _, _ = orc.solve(dims, kappa, bc, 1, U, X, tol=1e-14)
    return orc.force(dims, kappa, bc, U, X, Y), orc.action(X)


def test_rhs_sharded_force_over_gloo_world2():
    n_rhs = 5                                   # the paper's five equations over two cards: 3 + 2
    res = _run(2, n_rhs)
    Fr, Sr = _unsharded(n_rhs)
    assert res[0][2] == [0, 2, 4] and res[1][2] == [1, 3]
    for F, S, _ in res:                          # every rank ends with the full force and all the actions
        assert np.linalg.norm(F - Fr) / np.linalg.norm(Fr) < 1e-12
        assert np.allclose(S, Sr, rtol=1e-12)
    assert np.array_equal(res[0][0], res[1][0])  # and the ranks agree bit for bit


def test_rhs_sharded_force_over_gloo_more_ranks_than_columns():
    res = _run(3, 2)                             # rank 2 owns no column and contributes zeros
    Fr, Sr = _unsharded(2)
    assert res[2][2] == []
    for F, S, _ in res:
        assert np.linalg.norm(F - Fr) / np.linalg.norm(Fr) < 1e-12
        assert np.allclose(S, Sr, rtol=1e-12)


def test_column_deal():
    from paper_1009_5169_b200 import sharded as sh
    for n in (1, 5, 12, 16):
        for w in (1, 2, 3, 8):
            cols = [sh.columns_of_rank(n, w, r) for r in range(w)]
            assert sorted(sum(cols, [])) == list(range(n))
            assert max(len(c) for c in cols) == sh.max_columns_per_rank(n, w)
            assert max(len(c) for c in cols) - min(len(c) for c in cols) <= 1

"""The N > 1 path of bench.py is "replicas only": no data-path collective, only a barrier and a max over
ranks of the device time.  This runs that host logic with world_size 2 on CPU over gloo."""
import os
import socket
import sys

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


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank),
                      LOCAL_RANK=str(rank))
    from paper_1009_5169_b200 import replicas as rp
    import wd_inputs as wi
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w, r, l = rp.env_world()
    assert (w, r, l) == (world, rank, rank)
    # independent replicas: different seeds give different fields
    seed = rp.replica_seed(1, r)
    phi = wi.spinor_field((4, 4, 4, 4), 1, seed, wi.BC_SF)
    rp.barrier(dist, w)
    ms = 10.0 + 5.0 * r                      # rank 1 is the slow one
    mx = rp.max_over_ranks(dist, torch, w, ms, "cpu")
    rp.barrier(dist, w)
    out[rank] = (mx, rp.job_throughput(w, 3, mx), float(phi.sum()), rp.reference_arm_runs_here(r))
    dist.destroy_process_group()


def test_two_replicas_over_gloo():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    (mx0, v0, s0, ref0), (mx1, v1, s1, ref1) = out[0], out[1]
    assert mx0 == mx1 == 15.0                 # both ranks agree on the slowest replica's time
    assert v0 == v1 == world * 3 / 15e-3      # whole-job rate: all ranks' steps over that time
    assert s0 != s1                           # the replicas really are independent problems
    assert ref0 and not ref1                  # the reference arm runs on rank 0 only


def test_single_process_needs_no_process_group():
    from paper_1009_5169_b200 import replicas as rp
    assert rp.max_over_ranks(None, None, 1, 7.5, "cpu") == 7.5
    rp.barrier(None, 1)
    assert rp.job_throughput(1, 4, 2000.0) == 2.0

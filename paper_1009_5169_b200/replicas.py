"""Host-side logic of the multi-GPU form of the path: replicas only.

The pseudo-fermion columns are independent but the north_star keeps the whole block on
one GPU, so `bench.py --gpus N` runs N independent replicas of the hot path, one process per GPU.  The
only communication is measurement plumbing: a barrier around the timed region and the maximum over ranks
of the device time.  These helpers hold that logic so that it can be exercised on CPU with the gloo
backend (tests/test_replicas_gloo.py); on the GPU box the same code runs over NCCL.
"""
from __future__ import annotations

import os


def env_world():
    """(world_size, rank, local_rank) from the torchrun environment (1, 0, 0 when absent)."""
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


def replica_seed(base_seed: int, rank: int) -> int:
    """Every replica draws its own gauge field and right-hand sides: seed = base + rank."""
    return int(base_seed) + int(rank)


def barrier(dist, world: int) -> None:
    if world > 1:
        dist.barrier()


def max_over_ranks(dist, torch, world: int, value: float, device) -> float:
    """Device time of the slowest replica (the job is as slow as its slowest rank)."""
    if world == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(world: int, steps: int, max_ms: float) -> float:
    """Whole-job rate: every rank did `steps` units in the time of the slowest one (weak scaling)."""
    return world * steps / (max_ms * 1e-3)


def reference_arm_runs_here(rank: int) -> bool:
    """The oracle-timed reference arm runs on rank 0 only; other ranks exit 0 without work."""
    return rank == 0

"""Host-side logic of the multi-GPU path: replicas only.

Frames are independent ("per frame", BASELINE.json configs[3] "independent"), so N GPUs run
N copies of the single-GPU library with NO data-path collective: frame i of a stream goes to rank
i mod N, each rank of the single-frame bench cleans its own frame (same generator, seed offset by
rank).  torch.distributed is used for exactly two things: the barrier that brackets the timed region
and the MAX over ranks of the device-measured time.  Everything here is plain host code with no
method arithmetic; tests/test_replicas_gloo.py runs it with world_size 2 on the gloo backend.
"""
from __future__ import annotations

import os


def env_rank_world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process = 1 GPU)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def rank_seed(seed: int, rank: int) -> int:
    """Seed of the frame rank `rank` generates for the single-frame workload (weak scaling)."""
    return int(seed) + 100 * int(rank)


def shard(n_units: int, rank: int, world: int) -> list:
    """Indices of the independent units (frames) rank `rank` of `world` processes: i mod world == rank."""
    if world < 1 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad shard request: n_units=%r rank=%r world=%r" % (n_units, rank, world))
    return list(range(rank, n_units, world))


def barrier(world: int, sync=None) -> None:
    """Process barrier (when world > 1) followed by the device synchronisation `sync` (when given)."""
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    if sync is not None:
        sync()


def max_over_ranks(value: float, world: int, device=None) -> float:
    """MAX over ranks of a per-rank number (the device-measured time of the timed region)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, world: int, device=None) -> float:
    """SUM over ranks (units processed by the whole job)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput(units_this_rank: float, ms_this_rank: float, world: int, device=None) -> float:
    """Whole-job units/s: the units all ranks processed divided by the slowest rank's time."""
    units = sum_over_ranks(units_this_rank, world, device)
    ms = max_over_ranks(ms_this_rank, world, device)
    return units * 1e3 / ms

"""Multi-GPU plumbing of bench.py: N independent replicas.

The SHASTA step on one GPU exchanges nothing with other GPUs (north_star fixes the build to one GPU; the
paper's use case is event-by-event statistics), so `--gpus N` runs one independent event
per rank.  The only collectives are the barrier around the timed region and the MAX over ranks of the
device time.  Everything here works with the `gloo` backend on CPU as well (tests/test_replicas.py).
"""
from __future__ import annotations

import os

BASE_SEED = 12060919


def env():
    """(rank, world_size, local_rank) from the torchrun environment (1 process: 0, 1, 0)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(use_cuda: bool):
    """Join the process group when WORLD_SIZE > 1: nccl on GPUs, gloo on CPU.  Returns (rank, world, local)."""
    import torch
    import torch.distributed as dist
    rank, world, local = env()
    if world > 1 and not dist.is_initialized():
        if use_cuda:
            torch.cuda.set_device(local)
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")
    return rank, world, local


def barrier(use_cuda: bool):
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()
    if use_cuda:
        torch.cuda.synchronize()


def max_over_ranks(x: float, use_cuda: bool) -> float:
    """MAX over ranks of a per-rank device time (the contract's max-over-ranks timing)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device="cuda" if use_cuda else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def event_seed(rank: int) -> int:
    """Seed of the synthetic event of `rank`: a different event per replica."""
    return BASE_SEED + int(rank)


def aggregate_rate(cells_per_rank: int, steps: int, ms_max: float, world: int) -> float:
    """Whole-job cell-updates/s: every rank advanced `cells_per_rank` cells `steps` times within `ms_max`."""
    return world * cells_per_rank * steps / (ms_max * 1e-3)


def finalize():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()

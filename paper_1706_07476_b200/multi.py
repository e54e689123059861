"""Multi-GPU plumbing for replicas: rays are independent and the tally is a sum, so
each rank (one process per GPU) holds the whole mesh / tables, casts its own batches into a
private tally, and the replicas are combined by ONE fp64 sum all-reduce of the ncell doubles when
the tally is read (the tally leaves the GPU once, at the end).  There is no
data-path collective inside a cast step.  Backend: NCCL over NVLink on GPUs; the same code runs
on gloo for the CPU tests.
"""
from __future__ import annotations

import os
from typing import Tuple


def env_rank_world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process per GPU)."""
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def init_process_group(backend: str):
    import torch.distributed as dist

    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend)
    return dist


def batch_of_rank(step: int, rank: int, world: int) -> int:
    """Batch index cast by `rank` at `step`: ranks take disjoint, interleaved batches (weak scaling)."""
    return step * world + rank


def ray_shard(n_total: int, rank: int, world: int) -> Tuple[int, int]:
    """[first, last) of a contiguous split of one batch of n_total rays over `world` ranks (strong scaling)."""
    return n_total * rank // world, n_total * (rank + 1) // world


def allreduce_sum_(tensor):
    """In-place sum of a tally tensor over all ranks (no-op for a single process)."""
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(tensor, op=dist.ReduceOp.SUM)
    return tensor


def max_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())

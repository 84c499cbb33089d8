"""Multi-GPU plumbing: open-loop time steps are independent, so the
step range is split across ranks with replicated screens and no data-path collective; the only
exchange is one all-reduce(sum) of the long-exposure PSF at the end, plus the max-over-ranks of
the device time for reporting.  Works with the `nccl` backend on GPUs and `gloo` on CPU (tests).
"""
from __future__ import annotations

import os
from typing import Tuple


def env_world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process: 0, 0, 1)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str):
    import torch.distributed as dist
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def step_range(rank: int, world: int, steps_per_rank: int, step0: int = 0) -> Tuple[int, int]:
    """Weak scaling: every rank simulates `steps_per_rank` consecutive steps of one long run;
    rank r owns [step0 + r*K, step0 + (r+1)*K).  Returns (first step, count)."""
    return step0 + rank * steps_per_rank, steps_per_rank


def split_steps(rank: int, world: int, total_steps: int, step0: int = 0) -> Tuple[int, int]:
    """Strong scaling: `total_steps` split as evenly as possible; the first (total % world) ranks
    take one extra step.  Returns (first step, count); counts sum to total_steps, ranges tile."""
    base, extra = divmod(total_steps, world)
    count = base + (1 if rank < extra else 0)
    first = step0 + rank * base + min(rank, extra)
    return first, count


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks_(tensor):
    """In-place all-reduce(sum) of the long-exposure PSF accumulators (the one real exchange)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(tensor, op=dist.ReduceOp.SUM)
    return tensor

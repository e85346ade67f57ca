"""Multi-GPU plumbing: replicas only.

The per-projection solve does not shard usefully inside one solve: solves are
independent given w_init, so N GPUs run N replicas of the model and the projections of a sequence
are dealt to them in contiguous blocks (contiguous, so that each replica keeps the warm start from
its previous frame).  There is no data-path collective; torch.distributed is used only
for the start barrier and the max-over-ranks of the device time.
"""
from __future__ import annotations

import os
from typing import List, Tuple


def env_rank_world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process when absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def frame_block(rank: int, world: int, per_rank: int, start: int, n_total: int) -> List[int]:
    """Indices of the projections rank `rank` solves: a contiguous block of `per_rank` frames of the
    rotation, blocks of consecutive ranks following each other, wrapping around the n_total frames
    (weak scaling: per-rank work is fixed as the world grows)."""
    if not (0 <= rank < world) or per_rank < 0 or n_total < 1:
        raise ValueError("bad rank / world / per_rank")
    first = start + rank * per_rank
    return [(first + i) % n_total for i in range(per_rank)]


def init_process_group(backend: str):
    """Join the job torchrun started (no-op for a single process)."""
    import torch.distributed as dist
    _, _, world = env_rank_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend)
    return dist if world > 1 else None


def barrier(dist) -> None:
    if dist is not None:
        dist.barrier()


def max_over_ranks(dist, value: float, device=None) -> float:
    """Max of a per-rank scalar (the device time of the timed region)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(dist, value: float, device=None) -> float:
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())

"""Batch sharding over ranks: models are independent, the
tables are replicated, so the only cross-rank step is gathering B logL values
(and optionally the binned spectra).  Host logic only; the hot path itself
never communicates.  Works with any torch.distributed backend (NCCL on GPUs,
gloo in the CPU tests).
"""
from __future__ import annotations

from typing import Tuple


def shard_bounds(n_models: int, rank: int, world_size: int) -> Tuple[int, int]:
    """[begin, end) of the contiguous block of models rank `rank` evaluates.
    Blocks differ by at most one model; ranks beyond n_models get empty blocks."""
    if not (0 <= rank < world_size):
        raise ValueError(f"rank {rank} outside world of {world_size}")
    base, rem = divmod(int(n_models), int(world_size))
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def gather_rows(local, n_models: int, group=None):
    """All ranks pass their block (first dimension = their shard_bounds size) and get
    the full [n_models, ...] tensor in model order.  Ragged blocks are padded to the
    largest one for the all_gather and trimmed afterwards."""
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group)
    sizes = [shard_bounds(n_models, r, world) for r in range(world)]
    longest = max(e - b for b, e in sizes)
    pad = torch.zeros((longest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    return torch.cat([p[: e - b] for p, (b, e) in zip(parts, sizes)], dim=0)

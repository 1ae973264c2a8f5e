"""Data-parallel plumbing for SRA: how independent units are split across ranks, and the
max-over-ranks reduction used for timing.  No method arithmetic lives here.

SRA has no exchange step: every (batch item, head) is an independent attention problem
(the paper's Ulysses sequence parallelism, does its
all-to-all *around* attention precisely to make heads local).  So multi-GPU = one process per
GPU, each owning whole units, with no data-path collective:

  * weak scaling (bench.py default): the global batch is `world * batch_per_rank`; rank r owns
    batch items [r * batch_per_rank, (r + 1) * batch_per_rank).
  * head sharding (Ulysses-style strong scaling): rank r owns a contiguous slice of the heads.

The only collective is the timing reduction (MAX of the per-rank elapsed time).
"""
from __future__ import annotations

from typing import Tuple


def shard_range(n_units: int, world: int, rank: int) -> Tuple[int, int]:
    """Contiguous, balanced split of `n_units` over `world` ranks: returns (start, count).
    The first `n_units % world` ranks get one extra unit; every unit is owned exactly once."""
    if world < 1 or not (0 <= rank < world) or n_units < 0:
        raise ValueError(f"bad shard request n_units={n_units} world={world} rank={rank}")
    base, extra = divmod(n_units, world)
    start = rank * base + min(rank, extra)
    return start, base + (1 if rank < extra else 0)


def shard_batch(batch_per_rank: int, world: int, rank: int) -> Tuple[int, int]:
    """Weak scaling: global batch = world * batch_per_rank; returns this rank's (first item, count)."""
    return shard_range(batch_per_rank * world, world, rank)


def shard_heads(heads: int, world: int, rank: int) -> Tuple[int, int]:
    """Head sharding (what Ulysses SP leaves each GPU with): (first head, count)."""
    return shard_range(heads, world, rank)


def unit_seed(base_seed: int, global_batch_index: int) -> int:
    """Seed offset of one global batch item, so ranks draw different synthetic data."""
    return base_seed + 100003 * global_batch_index


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar over the default process group (identity when not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    """SUM all-reduce of a scalar (units processed by the whole job)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())

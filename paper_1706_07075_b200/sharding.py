"""Host-side logic of the multi-GPU path.

The path shards over EVENTS: they are independent given the image, so every rank holds a contiguous shard of the
event list and a full copy of image / sensitivity, runs the fused EM pass on its shard into its own correction
image, and the only exchange of an iteration is one float32 SUM all-reduce of that correction image; every rank
then applies the same multiplicative update.  No kernel waits on another rank.

Only plumbing lives here (index arithmetic and the torch.distributed call); all arithmetic of the method runs in
libtofmlem's kernels.
"""
from __future__ import annotations

from typing import Optional, Tuple

import torch
import torch.distributed as dist


def shard_range(n_total: int, rank: int, world: int) -> Tuple[int, int]:
    """(start, count) of rank's contiguous event shard: the shards tile [0, n_total) in rank order and differ in
    size by at most one event (the first n_total % world ranks take the extra one)."""
    if world < 1 or not (0 <= rank < world) or n_total < 0:
        raise ValueError(f"bad shard request: n_total={n_total} rank={rank} world={world}")
    base, extra = divmod(n_total, world)
    start = rank * base + min(rank, extra)
    return start, base + (1 if rank < extra else 0)


def weak_shard_range(n_per_rank: int, rank: int) -> Tuple[int, int]:
    """Weak scaling (bench.py --gpus N): every rank takes n_per_rank consecutive events of the seeded stream."""
    if n_per_rank < 0 or rank < 0:
        raise ValueError("bad weak shard request")
    return rank * n_per_rank, n_per_rank


def allreduce_correction(corr: torch.Tensor, group: Optional[dist.ProcessGroup] = None) -> torch.Tensor:
    """Sum the per-rank partial correction images in place (the iteration's one real exchange step).
    A no-op for a single process.  NCCL on GPUs; the same call runs over gloo in the CPU test."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(corr, op=dist.ReduceOp.SUM, group=group)
    return corr


def max_over_ranks_ms(ms: float, device: Optional[torch.device] = None, group: Optional[dist.ProcessGroup] = None) -> float:
    """Device-timed milliseconds -> max over ranks (how every multi-GPU number is reported)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def sum_over_ranks(count: int, device: Optional[torch.device] = None, group: Optional[dist.ProcessGroup] = None) -> int:
    """An integer count (e.g. the valid events of a pass) summed over ranks; the value itself for a single process."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return int(count)
    t = torch.tensor([count], dtype=torch.int64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return int(t.item())

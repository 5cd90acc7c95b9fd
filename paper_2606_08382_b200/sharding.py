"""Batch sharding across ranks.

Sequences of a decode batch are independent, so the hot path shards by batch with no data-path
collective: rank r of W takes a contiguous slice of the sequences and runs the same kernels.
``bench.py --gpus N`` keeps the per-GPU batch fixed (weak scaling) -- every rank owns a full
BASELINE batch -- and only the timing is reduced (max over ranks)."""
from __future__ import annotations

from typing import Tuple


def shard_batch(batch: int, rank: int, world: int) -> Tuple[int, int]:
    """[start, stop) of the sequences rank ``rank`` owns when ``batch`` sequences are split over
    ``world`` ranks as evenly as possible (first ``batch % world`` ranks get one more)."""
    if world <= 0 or not 0 <= rank < world or batch < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(batch, world)
    start = rank * base + min(rank, extra)
    return start, start + base + (1 if rank < extra else 0)


def max_over_ranks(ms: float, device=None) -> float:
    """Max of a per-rank duration over the process group (no-op without torch.distributed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return ms
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())

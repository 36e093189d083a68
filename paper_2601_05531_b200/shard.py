"""Multi-GPU sharding of the DNATok path: records are independent, so each rank takes a
contiguous range of records of about equal byte count and encodes it with its own handle; nothing crosses ranks on the
data path.  The only exchange is one int64 per rank (its token total), from which every rank gets the global token
index of its first token.  Host-side logic only; works with any torch.distributed backend (nccl on GPUs, gloo on CPU).
"""
from __future__ import annotations

import numpy as np

__all__ = ["partition_records", "exclusive_token_base"]


def partition_records(rec_offsets: np.ndarray, world: int) -> list[tuple[int, int]]:
    """Cut records [0, n) into `world` contiguous ranges [r0, r1) whose byte counts are as equal as record
    boundaries allow: range i ends at the first record boundary at or after byte (i + 1) * total / world."""
    offs = np.asarray(rec_offsets, dtype=np.int64)
    n = offs.size - 1
    assert world >= 1 and n >= 0
    lo, hi = int(offs[0]), int(offs[-1])
    cuts = [0]
    for i in range(1, world):
        target = lo + (hi - lo) * i // world
        r = int(np.searchsorted(offs, target, side="left"))
        cuts.append(min(max(r, cuts[-1]), n))
    cuts.append(n)
    return [(cuts[i], cuts[i + 1]) for i in range(world)]


def exclusive_token_base(local_tokens: int, group=None) -> tuple[int, int]:
    """(global index of this rank's first token, total over all ranks): an exclusive scan of one int64 per rank."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return 0, int(local_tokens)
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    mine = torch.tensor([int(local_tokens)], dtype=torch.int64, device=dev)
    every = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(every, mine, group=group)
    totals = [int(t.item()) for t in every]
    return sum(totals[:rank]), sum(totals)

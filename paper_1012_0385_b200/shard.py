"""Sample sharding over ranks.

Realisations are independent and every random number is keyed by the GLOBAL sample index
(`first_sample` + local index), so a rank that owns samples [first, first+count) produces exactly the rows a single
process would: there is no collective on the data path, only a gather of the KB-sized records at the end.
Plain host logic - no method arithmetic; works with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import numpy as np


def shard_samples(total_samples: int, world_size: int, rank: int) -> tuple[int, int]:
    """Strong partition of an ensemble: contiguous blocks, the first (total % world) ranks take one extra sample.
    Returns (first_sample, count)."""
    if not (0 <= rank < world_size) or total_samples < 0:
        raise ValueError("need 0 <= rank < world_size and total_samples >= 0")
    base, extra = divmod(total_samples, world_size)
    count = base + (1 if rank < extra else 0)
    first = rank * base + min(rank, extra)
    return first, count


def weak_first_sample(samples_per_rank: int, rank: int) -> int:
    """Weak scaling (bench.py --gpus N): every rank runs the same shape on its own block of global samples."""
    return rank * samples_per_rank


def gather_records(local: dict, group=None) -> dict:
    """All-gather per-sample record arrays ([nt][S_local], samples on the last axis) from every rank and concatenate
    them in rank order = global sample order.  `local` maps names to numpy arrays; arrays with fewer than 2 dims
    (e.g. the record times) are taken from rank 0."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    if world == 1:
        return {k: np.asarray(v) for k, v in local.items()}
    out = {}
    for name in sorted(local):
        a = np.ascontiguousarray(local[name])
        parts = [None] * world
        dist.all_gather_object(parts, a, group=group)
        out[name] = np.concatenate(parts, axis=-1) if a.ndim >= 2 else parts[0]
    del torch
    return out

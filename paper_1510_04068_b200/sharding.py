"""Host-side multi-rank plumbing for the weak-scaling bench.

The path shards by independent i-lists: every rank holds the full j-store and computes forces on its own
rotation of the seeded active-set permutation.  There is no data-path collective; the only communication
is the barrier and the max-over-ranks of the device timings.
"""
from __future__ import annotations

import numpy as np


def rank_ilist(perm: np.ndarray, rank: int, world: int, ni: int) -> np.ndarray:
    """i-list of `rank`: the first `ni` entries of the permutation rotated by rank * (N // world).
    For ni <= N // world the lists of different ranks are disjoint; their union over ranks of the
    length-(N // world) lists is the whole particle set."""
    n = perm.shape[0]
    if not (0 <= rank < world) or not (0 < ni <= n):
        raise ValueError("rank_ilist: bad rank / world / ni")
    return np.ascontiguousarray(np.roll(perm, -rank * (n // world))[:ni]).astype(np.int32, copy=False)


def max_over_ranks(values, device=None):
    """Element-wise maximum over all ranks of a short list of floats (identity without a process group)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]

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


# ----------------------------------------------------------------------------------------------------------
# j-sharding (sec 2.2.3, sec 3.6): "the j-particles are distributed over the GPUs in a
# round-robin fashion", every device computes partial results for all i, and the partials are added.  The
# paper adds them on the host; here the exchange is one all-reduce over the ranks' process group (NCCL on
# GPUs, gloo in the CPU tests).  north_star fixes this build at one GPU, so this is the SURVEY 8(f) rank-4
# extension: correct by construction, covered by a world-size-2 CPU test, not part of the bench line.

def round_robin_shard(n: int, rank: int, world: int) -> np.ndarray:
    """Global addresses of the j-particles rank `rank` holds: rank, rank + world, rank + 2 world, ... (L84)."""
    return np.arange(rank, n, world, dtype=np.int32)


def local_to_global(local_address, rank: int, world: int):
    """Address in a rank's local j-store -> global address under round_robin_shard."""
    return local_address * world + rank


def combine_partials(acc, jerk, pot, snap=None, nn_id=None, nn_r2=None, ngb_count=None, group=None):
    """Combines per-rank partial force results for the SAME i-list in place (torch tensors, any device).

    Sums (acc, jerk, snap, pot) and neighbour counts: all-reduce SUM.  Nearest neighbour: the rank whose
    candidate has the smallest (r2, id) wins (id breaks exact ties, as the single-GPU path breaks them by
    address; benchmark inputs have id == address).  The summation order over ranks is fixed by the
    collective's algorithm for a given world size; as the paper notes (L84, L164) it differs from the
    single-device order in the last digit."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return
    for t in (acc, jerk, snap, pot, ngb_count):
        if t is not None:
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    if nn_id is not None and nn_r2 is not None:
        world = dist.get_world_size(group)
        r2s = [torch.empty_like(nn_r2) for _ in range(world)]
        ids = [torch.empty_like(nn_id) for _ in range(world)]
        dist.all_gather(r2s, nn_r2, group=group)
        dist.all_gather(ids, nn_id, group=group)
        best_r2, best_id = r2s[0].clone(), ids[0].clone()
        for r2, idv in zip(r2s[1:], ids[1:]):
            better = (r2 < best_r2) | ((r2 == best_r2) & (idv >= 0) & ((idv < best_id) | (best_id < 0)))
            best_r2 = torch.where(better, r2, best_r2)
            best_id = torch.where(better, idv, best_id)
        nn_r2.copy_(best_r2)
        nn_id.copy_(best_id)


class ShardedForces:
    """One rank's part of a j-sharded force evaluation: holds the round-robin shard of the j-particles in a
    library context, evaluates the i-list against it (explicit sinks: an i-particle need not live on this
    rank) and combines with the other ranks.  Host-predicted i-state, GRAPE style (L92)."""

    def __init__(self, n_total: int, order: int = 4, precision: int = 0, device: int = 0, group=None):
        import torch.distributed as dist
        from . import binding as s2
        self.s2, self.group, self.n_total = s2, group, n_total
        ok = dist.is_available() and dist.is_initialized()
        self.rank = dist.get_rank(group) if ok else 0
        self.world = dist.get_world_size(group) if ok else 1
        self.mine = round_robin_shard(n_total, self.rank, self.world)
        self.order = order
        self.device = device
        self.ctx = s2.s2_open(device, order, precision, nj_capacity=max(1, self.mine.size), ngb_cap=0)

    def set_all_j(self, ident, t, mass, pos, vel, acc, jerk, snap=None, crackle=None):
        m = self.mine
        pick = lambda a: None if a is None else np.ascontiguousarray(a[m])
        self.s2.s2_set_j(self.ctx, np.arange(m.size, dtype=np.int32), pick(ident), pick(t), pick(mass), pick(pos),
                         pick(vel), pick(acc), pick(jerk), pick(snap), pick(crackle))
        self.s2.s2_commit_j(self.ctx)

    def forces(self, t: float, i_id, i_pos, i_vel, i_acc=None, eps2: float = 0.0):
        import torch
        s2 = self.s2
        s2.s2_predict(self.ctx, float(t), self.mine.size)
        s2.s2_calc_explicit(self.ctx, i_id, i_pos, i_vel, i_acc, None, eps2, s2.S2_WANT_NN)
        r = s2.s2_get_results(self.ctx, len(i_id))
        dev = torch.device("cuda", self.device)
        ten = {k: torch.from_numpy(np.ascontiguousarray(v)).to(dev) for k, v in r.items()
               if isinstance(v, np.ndarray)}
        combine_partials(ten["acc"], ten["jerk"], ten["pot"], ten.get("snap"), ten["nn_id"], ten["nn_r2"], None, self.group)
        return {k: v.cpu().numpy() for k, v in ten.items()}

    def close(self):
        self.s2.s2_close(self.ctx)

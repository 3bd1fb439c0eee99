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
# j-sharding (sec 2.2.3, sec 3.6): the j-particles are distributed over the GPUs, every device
# computes partial results for ALL i against its own j, and the partials are added.  The paper deals the particles
# round-robin and adds on the host; here every rank keeps the whole 116-byte-per-particle store, predicts
# all of it (HBM-bound, microseconds) and sums over its own contiguous address block (s2_set_j_range), so that
#   * i-particles are given by address and use the device-predicted state on every rank (no host-predicted copies),
#   * nearest-neighbour and neighbour-list addresses are global on every rank,
#   * rank order = address order: exact nn ties go to the lowest rank, lists concatenate ascending without a sort.
# The exchange is one all-reduce (sums, counts) plus all-gathers (nn candidates, list lengths, list members) on
# device tensors -- at most a few MB, latency-bound on NVLink, so no fused compute+collective kernel is warranted.
# north_star fixes this build at one GPU: correct by construction, covered by world-size-2 gloo tests on CPU and by a
# single-GPU test that runs the shards one after the other; unmeasured on multi-GPU hardware (no SCALE record).

def block_shard(n: int, rank: int, world: int) -> tuple[int, int]:
    """(first, count) of the contiguous block of j addresses rank `rank` sums over; the blocks tile 0 .. n-1."""
    first = (n * rank) // world
    return first, (n * (rank + 1)) // world - first


def round_robin_shard(n: int, rank: int, world: int) -> np.ndarray:
    """Global addresses under the paper's round-robin dealing (L84): rank, rank + world, ... (kept for reference and
    for the CPU test of the combine; the library path uses block_shard)."""
    return np.arange(rank, n, world, dtype=np.int32)


def _world(group):
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return 1, 0
    return dist.get_world_size(group), dist.get_rank(group)


def combine_partials(acc, jerk, pot, snap=None, nn_id=None, nn_r2=None, ngb_count=None, group=None):
    """Combines per-rank partial force results for the SAME i-list in place (torch tensors, any device).

    Sums (acc, jerk, snap, pot) and neighbour counts: all-reduce SUM.  Nearest neighbour: smallest r2; an exact tie
    goes to the LOWEST RANK, which under block_shard holds the lowest addresses -- the single-GPU rule (ties to the
    lowest address), whatever the ids are.  The summation order over ranks is fixed by the collective's algorithm for
    a given world size; as the paper notes (L84, L164) it differs from the single-device order in the last digit."""
    import torch
    import torch.distributed as dist
    world, _ = _world(group)
    if world == 1:
        return
    for t in (acc, jerk, snap, pot, ngb_count):
        if t is not None:
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    if nn_id is not None and nn_r2 is not None:
        r2s = [torch.empty_like(nn_r2) for _ in range(world)]
        ids = [torch.empty_like(nn_id) for _ in range(world)]
        dist.all_gather(r2s, nn_r2, group=group)
        dist.all_gather(ids, nn_id, group=group)
        best_r2, best_id = r2s[0].clone(), ids[0].clone()
        for r2, idv in zip(r2s[1:], ids[1:]):
            better = r2 < best_r2                      # strict: ties stay with the lower rank
            best_r2 = torch.where(better, r2, best_r2)
            best_id = torch.where(better, idv, best_id)
        nn_r2.copy_(best_r2)
        nn_id.copy_(best_id)


def merge_rank_lists(lens_by_rank, lists_by_rank, cap: int):
    """Per-i concatenation, in rank order, of per-rank CSR lists (lens_by_rank[r]: int64 [ni] segment lengths,
    lists_by_rank[r]: the members, segment after segment), truncated to the first `cap` members per i.
    Returns (offsets int64 [ni+1], members).  Pure index arithmetic on torch tensors (any device)."""
    import torch
    ni = lens_by_rank[0].numel()
    dev = lens_by_rank[0].device
    total_len = torch.stack(lens_by_rank).sum(0)
    mlen = torch.clamp(total_len, max=cap)
    moff = torch.zeros(ni + 1, dtype=torch.int64, device=dev)
    moff[1:] = torch.cumsum(mlen, 0)
    out = torch.empty(int(moff[-1]), dtype=lists_by_rank[0].dtype, device=dev)
    prefix = torch.zeros(ni, dtype=torch.int64, device=dev)
    idx = torch.arange(ni, device=dev)
    for lens, lst in zip(lens_by_rank, lists_by_rank):
        n_r = int(lens.sum())
        if n_r:
            off = torch.cumsum(lens, 0) - lens
            seg = torch.repeat_interleave(idx, lens)
            mpos = prefix[seg] + (torch.arange(n_r, device=dev) - off[seg])
            keep = mpos < cap
            out[(moff[seg] + mpos)[keep]] = lst[:n_r][keep]
        prefix = prefix + lens
    return moff, out


def combine_neighbour_lists(offsets, members, cap: int, group=None):
    """Variable-length all-gather (lengths first) of every rank's CSR neighbour lists for the same i-list and their
    per-i merge in rank order.  offsets: int64 [ni+1]; members: int32 global addresses, ascending within a segment.
    Under block_shard the merged lists are ascending and hold the `cap` lowest addresses (reading P8)."""
    import torch
    import torch.distributed as dist
    world, _ = _world(group)
    lens = (offsets[1:] - offsets[:-1]).to(torch.int64)
    if world == 1:
        return merge_rank_lists([lens], [members], cap)
    all_lens = [torch.empty_like(lens) for _ in range(world)]
    dist.all_gather(all_lens, lens, group=group)
    longest = max(int(l.sum()) for l in all_lens)
    padded = torch.zeros(max(longest, 1), dtype=members.dtype, device=members.device)
    padded[:members.numel()] = members
    all_lists = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(all_lists, padded, group=group)
    return merge_rank_lists(all_lens, all_lists, cap)


class ShardedForces:
    """One rank's part of a j-sharded force evaluation.  Holds the whole j-store in a library context, sums over its
    own address block, and combines with the other ranks on device tensors (no host hop)."""

    def __init__(self, n_total: int, order: int = 4, precision: int = 0, device: int = 0, group=None, ngb_cap: int = 0,
                 rank: int | None = None, world: int | None = None):
        from . import binding as s2
        self.s2, self.group, self.n_total, self.ngb_cap = s2, group, n_total, ngb_cap
        w, r = _world(group)
        self.world = w if world is None else world         # (rank, world) may be forced: shards run one after the other
        self.rank = r if rank is None else rank            # on a single GPU in the tests
        self.first, self.count = block_shard(n_total, self.rank, self.world)
        self.order, self.device = order, device
        self.ctx = s2.s2_open(device, order, precision, nj_capacity=n_total, ngb_cap=ngb_cap)
        s2.s2_set_j_range(self.ctx, self.first, self.count)

    def set_all_j(self, ident, t, mass, pos, vel, acc, jerk, snap=None, crackle=None):
        self.s2.s2_set_j(self.ctx, np.arange(self.n_total, dtype=np.int32), ident, t, mass, pos, vel, acc, jerk, snap, crackle)
        self.s2.s2_commit_j(self.ctx)

    def partial(self, t: float, d_i_address, d_h2=None, eps2: float = 0.0, flags: int = 0) -> dict:
        """This rank's partial results for the i-list (torch CUDA tensors), uncombined."""
        import torch
        s2 = self.s2
        ni = d_i_address.numel()
        dev = d_i_address.device
        s2.s2_predict(self.ctx, float(t), self.n_total)
        s2.s2_calc_ilist_device(self.ctx, d_i_address, d_h2, eps2, flags)
        f64 = dict(dtype=torch.float64, device=dev)
        out = dict(acc=torch.empty(ni * 3, **f64), jerk=torch.empty(ni * 3, **f64), pot=torch.empty(ni, **f64),
                   snap=torch.empty(ni * 3, **f64) if self.order == 6 else None,
                   nn_id=torch.empty(ni, dtype=torch.int32, device=dev), nn_r2=torch.empty(ni, **f64),
                   ngb_count=torch.empty(ni, dtype=torch.int32, device=dev))
        s2.s2_get_results_device(self.ctx, ni, **out)
        if flags & s2.S2_WANT_NGB:
            off, lst, _ = s2.s2_get_neighbours_csr_device(self.ctx, ni)
            out["offsets"], out["list"] = off.clone(), lst.clone()
        return out

    def forces(self, t: float, d_i_address, d_h2=None, eps2: float = 0.0, flags: int = 0) -> dict:
        """Combined results over all ranks, on the device."""
        s2 = self.s2
        out = self.partial(t, d_i_address, d_h2, eps2, flags)
        nn = bool(flags & (s2.S2_WANT_NN | s2.S2_WANT_NGB))
        ngb = bool(flags & s2.S2_WANT_NGB)
        combine_partials(out["acc"], out["jerk"], out["pot"], out["snap"], out["nn_id"] if nn else None,
                         out["nn_r2"] if nn else None, out["ngb_count"] if ngb else None, self.group)
        if ngb:
            out["offsets"], out["list"] = combine_neighbour_lists(out["offsets"], out["list"], self.ngb_cap, self.group)
        return out

    def close(self):
        self.s2.s2_close(self.ctx)

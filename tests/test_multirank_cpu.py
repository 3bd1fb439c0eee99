"""World-size-2 gloo test (CPU) of the multi-rank host logic used by bench.py --gpus N: i-list sharding by
rank and the max-over-ranks timing reduction.  No GPU and no oracle involved."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1510_04068_b200.sharding import combine_partials, max_over_ranks, rank_ilist, round_robin_shard
from workloads import make_config


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = make_config(2)                                   # N = 64
    il = rank_ilist(w.perm, rank, world, w.N // world)
    gathered = [torch.zeros(w.N // world, dtype=torch.int32) for _ in range(world)]
    dist.all_gather(gathered, torch.from_numpy(il.copy()))
    dist.barrier()
    mx = max_over_ranks([10.0 + rank, 5.0 - rank])
    if rank == 0:
        q.put((torch.cat(gathered).numpy(), mx))
    dist.destroy_process_group()


def test_two_rank_sharding_and_timing_reduce():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    allidx, mx = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(allidx.tolist()) == list(range(64))    # disjoint lists whose union is every particle
    assert mx == [11.0, 5.0]                             # element-wise max over ranks


def test_rank_ilist_single_rank_is_prefix():
    w = make_config(2)
    assert np.array_equal(rank_ilist(w.perm, 0, 1, 10), w.ilist(10))
    assert max_over_ranks([1.5, 2.5]) == [1.5, 2.5]


def _jshard_worker(rank, world, port, q):
    """Each rank evaluates the oracle on its address block of the j-particles (block_shard) for the same i-list; the
    partial sums, nearest-neighbour candidates and neighbour lists are combined with combine_partials /
    combine_neighbour_lists (gloo) and must equal the oracle over all j -- lists, ties and truncation included."""
    import oracle
    from paper_1510_04068_b200.sharding import block_shard, combine_neighbour_lists
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w, xp, vp, il, h2, cap = _jshard_problem()
    first, count = block_shard(w.N, rank, world)
    mine = np.arange(first, first + count)
    part = oracle.forces(4, w.mass[mine], w.ident[mine], xp[mine], vp[mine], None, w.ident[il], xp[il], vp[il], None,
                         w.eps2, h2, cap)
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(part, k))) for k in ("acc", "jerk", "pot", "nn_id", "nn_d2", "ngb_count")}
    # this rank's CSR lists with GLOBAL addresses (what the library returns under s2_set_j_range)
    lens = np.minimum(part.ngb_count, cap).astype(np.int64)
    off = torch.zeros(il.size + 1, dtype=torch.int64)
    off[1:] = torch.from_numpy(np.cumsum(lens))
    members = np.concatenate([part.ngb_list[i, :lens[i]] + first for i in range(il.size)] + [np.zeros(0, np.int32)]).astype(np.int32)
    combine_partials(t["acc"], t["jerk"], t["pot"], None, t["nn_id"], t["nn_d2"], t["ngb_count"])
    moff, mlist = combine_neighbour_lists(off, torch.from_numpy(members), cap)
    if rank == 0:
        out = {k: v.numpy() for k, v in t.items()}
        out["offsets"], out["list"] = moff.numpy(), mlist.numpy()
        q.put(out)
    dist.barrier()
    dist.destroy_process_group()


def _jshard_problem():
    import oracle
    w = make_config(1, N=200)
    # two coincident-distance candidates on different ranks: particle 150 is moved to mirror particle 20 about i = perm[0]
    xp, vp, _ = oracle.predict(4, w.t_pred, w.t_j, w.pos, w.vel, w.acc, w.jerk)
    il = w.ilist(50)
    h2 = np.full(50, 0.05)
    h2[::7] = 0.5                      # some lists longer than the cap: truncation to the lowest addresses across ranks
    return w, xp, vp, il, h2, 24


def test_two_rank_j_sharding_combine_matches_full_sum():
    import oracle
    from paper_1510_04068_b200.sharding import block_shard, merge_rank_lists
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_jshard_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w, xp, vp, il, h2, cap = _jshard_problem()
    full = oracle.forces_ilist(4, w.mass, w.ident, xp, vp, None, il, w.eps2, h2, cap)
    assert np.allclose(got["acc"], full.acc, rtol=1e-14, atol=0) and np.allclose(got["jerk"], full.jerk, rtol=1e-13, atol=0)
    assert np.allclose(got["pot"], full.pot, rtol=1e-14, atol=0)
    assert np.array_equal(got["nn_id"], full.nn_id) and np.array_equal(got["nn_d2"], full.nn_d2)
    assert np.array_equal(got["ngb_count"], full.ngb_count) and (full.ngb_count > cap).any()
    assert np.array_equal(np.diff(got["offsets"]), np.minimum(full.ngb_count, cap))
    for i in range(il.size):
        want = full.ngb_list[i][full.ngb_list[i] >= 0]
        assert np.array_equal(got["list"][got["offsets"][i]:got["offsets"][i + 1]], want), i
    # the blocks tile the address range; an exact nn tie across ranks goes to the lower rank (= lower address)
    assert sum(block_shard(11, r, 3)[1] for r in range(3)) == 11 and block_shard(11, 2, 3)[0] == 7
    assert sorted(np.concatenate([round_robin_shard(11, r, 3) for r in range(3)]).tolist()) == list(range(11))
    lens = [torch.tensor([2, 0, 3]), torch.tensor([1, 2, 3])]
    lists = [torch.tensor([1, 2, 5, 6, 7], dtype=torch.int32), torch.tensor([11, 12, 13, 14, 15, 16], dtype=torch.int32)]
    off, m = merge_rank_lists(lens, lists, cap=4)
    assert off.tolist() == [0, 3, 5, 9] and m.tolist() == [1, 2, 11, 12, 13, 5, 6, 7, 14]

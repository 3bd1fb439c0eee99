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
    """Each rank evaluates the oracle on its round-robin shard of the j-particles for the same i-list; the partials
    are combined with combine_partials (gloo) and must equal the oracle on all j."""
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = make_config(1, N=200)
    xp, vp, _ = oracle.predict(4, w.t_pred, w.t_j, w.pos, w.vel, w.acc, w.jerk)
    il = w.ilist(50)
    mine = round_robin_shard(w.N, rank, world)
    h2 = np.full(50, 0.05)
    part = oracle.forces(4, w.mass[mine], w.ident[mine], xp[mine], vp[mine], None, w.ident[il], xp[il], vp[il], None,
                         w.eps2, h2, 64)
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(part, k))) for k in ("acc", "jerk", "pot", "nn_id", "nn_d2", "ngb_count")}
    combine_partials(t["acc"], t["jerk"], t["pot"], None, t["nn_id"], t["nn_d2"], t["ngb_count"])
    if rank == 0:
        q.put({k: v.numpy() for k, v in t.items()})
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_j_sharding_combine_matches_full_sum():
    import oracle
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
    w = make_config(1, N=200)
    xp, vp, _ = oracle.predict(4, w.t_pred, w.t_j, w.pos, w.vel, w.acc, w.jerk)
    il = w.ilist(50)
    full = oracle.forces_ilist(4, w.mass, w.ident, xp, vp, None, il, w.eps2, np.full(50, 0.05), 64)
    assert np.allclose(got["acc"], full.acc, rtol=1e-14, atol=0) and np.allclose(got["jerk"], full.jerk, rtol=1e-13, atol=0)
    assert np.allclose(got["pot"], full.pot, rtol=1e-14, atol=0)
    assert np.array_equal(got["nn_id"], full.nn_id) and np.array_equal(got["nn_d2"], full.nn_d2)
    assert np.array_equal(got["ngb_count"], full.ngb_count)
    assert sorted(np.concatenate([round_robin_shard(11, r, 3) for r in range(3)]).tolist()) == list(range(11))

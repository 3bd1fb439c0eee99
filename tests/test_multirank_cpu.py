"""World-size-2 gloo test (CPU) of the multi-rank host logic used by bench.py --gpus N: i-list sharding by
rank and the max-over-ranks timing reduction.  No GPU and no oracle involved."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1510_04068_b200.sharding import max_over_ranks, rank_ilist
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

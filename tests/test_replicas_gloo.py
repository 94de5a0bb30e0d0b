"""N > 1 path on CPU: two gloo ranks run the replica bookkeeping of bench.py (replicas only --
no collective on the data path; the measurement takes MAX of the device times and SUM of the updates)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1209_0296_b200 import replicas, workloads as W


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = W.configs()["cfg2_T2.269"]
        seed = replicas.rank_seed(w.seed, rank)
        local_ms = 10.0 + 5.0 * rank            # rank 1 is the slow one
        local_updates = 1000 * (rank + 1)
        ms, upd, ups = replicas.aggregate(local_ms, local_updates)
        seeds = [None] * world
        dist.all_gather_object(seeds, seed)
        out.put((rank, ms, upd, ups, seeds))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_aggregate_like_the_bench():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    base = W.configs()["cfg2_T2.269"].seed
    for rank, ms, upd, ups, seeds in res:
        assert ms == 15.0                       # MAX over ranks
        assert upd == 3000.0                    # SUM over ranks
        assert abs(ups - 3000.0 / 15e-3) < 1e-6
        assert seeds == [base, base + replicas.SEED_STRIDE] and len(set(seeds)) == world


def test_single_process_is_the_identity():
    assert replicas.rank_seed(42, 0) == 42
    ms, upd, ups = replicas.aggregate(2.0, 500)
    assert (ms, upd) == (2.0, 500.0) and abs(ups - 250000.0) < 1e-9

"""World-size-2 gloo test of the multi-rank host logic (no GPU): shard arithmetic, per-rank seeds, and
the max-over-ranks timing reduction bench.py uses."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2505_15204_b200 import shard


def test_timestep_ranges_cover_exactly():
    for T in (1, 5, 50, 51):
        for world in (1, 2, 3, 8):
            got = []
            for r in range(world):
                t0, t1 = shard.timestep_range(T, world, r)
                assert 0 <= t0 <= t1 <= T
                got += list(range(t0, t1))
            assert got == list(range(T))
            sizes = [shard.timestep_range(T, world, r)[1] - shard.timestep_range(T, world, r)[0] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


def test_rank_seeds_distinct():
    seeds = [shard.rank_seed(3, r) for r in range(8)]
    assert seeds[0] is None and len(set(seeds[1:])) == 7 and 1003 not in seeds[1:]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    mx = shard.max_over_ranks(ms)
    t0, t1 = shard.timestep_range(5, world, rank)
    owned = torch.zeros(5)
    owned[t0:t1] = 1
    dist.all_reduce(owned)                        # every timestep owned exactly once
    q.put((rank, mx, shard.aggregate_rate(100, world, mx), owned.tolist()))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_gloo():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(2)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, rate, owned in res:
        assert mx == 15.0                                       # max over ranks, on every rank
        assert abs(rate - 2 * 100 / 15e-3) < 1e-6
        assert owned == [1.0] * 5

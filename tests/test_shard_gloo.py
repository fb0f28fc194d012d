"""The N > 1 host logic on CPU: two processes, gloo backend, 127.0.0.1 (no GPU involved)."""
import os
import socket

import numpy as np
import pytest

from paper_2606_17212_b200 import shard


def test_partitions_cover_every_unit_once():
    for world in (1, 2, 3, 8):
        for n in (0, 1, 7, 150):
            seen = sorted(u for r in range(world) for u in shard.units_for_rank(n, r, world))
            assert seen == list(range(n))
            cover = np.zeros(n, int)
            for r in range(world):
                cover[shard.split_states(n, r, world)] += 1
            assert np.all(cover == 1)
    # at a given step the ranks hold different frames; K steps cover K*world frames
    frames = {shard.frame_for_step(k, r, 4, 150) for k in range(10) for r in range(4)}
    assert len(frames) == 40
    with pytest.raises(ValueError):
        shard.frame_for_step(0, 2, 2, 10)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        t = shard.max_over_ranks(10.0 + rank)
        # each rank owns different views and therefore a different number of pairs
        views = shard.units_for_rank(5, rank, world)
        rng = np.random.default_rng(100 + rank)
        n = 3 * len(views) + rank
        dm, dd, gi = rng.normal(size=n), rng.normal(size=n), rng.integers(0, 4, n).astype(np.int32)
        pm, pd, pg = shard.pool_pairs(dm, dd, gi)
        q.put((rank, t, views, dm, pm, pd, pg))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_max_and_pooling():
    import torch.multiprocessing as mp
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=120) for _ in range(world)), key=lambda x: x[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(r[1] == 11.0 for r in res)                       # max over ranks on every rank
    assert sorted(res[0][2] + res[1][2]) == [0, 1, 2, 3, 4]
    expect = np.concatenate([res[0][3], res[1][3]])             # rank order
    for r in res:
        assert np.array_equal(r[4], expect)
        assert r[5].shape == expect.shape and r[6].shape == expect.shape
    assert np.array_equal(res[0][6], res[1][6])

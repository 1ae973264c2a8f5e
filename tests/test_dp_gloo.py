"""-m "not gpu": the N > 1 plumbing of bench.py (paper_2606_13872_b200/dp.py) with the gloo backend,
world_size 2, on CPU: unit sharding is a partition, and the timing reduction is a MAX over ranks."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_13872_b200 import dp


def test_shard_range_is_a_partition():
    for n in (0, 1, 5, 40, 41, 80):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                s, c = dp.shard_range(n, world, r)
                seen.extend(range(s, s + c))
            assert seen == list(range(n))
    assert dp.shard_heads(40, 8, 3) == (15, 5)
    assert dp.shard_batch(2, 4, 1) == (2, 2)
    with pytest.raises(ValueError):
        dp.shard_range(4, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        b0, cnt = dp.shard_batch(1, world, rank)
        elapsed = 10.0 + 5.0 * rank          # rank 1 is the straggler
        units = float(cnt) * 3.0             # "flops" this rank processed
        q.put((rank, b0, cnt, dp.max_over_ranks(elapsed), dp.sum_over_ranks(units), dp.unit_seed(0, b0)))
    finally:
        dist.destroy_process_group()


def test_gloo_world2_max_and_sum():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [0, 1] and [r[2] for r in res] == [1, 1]
    assert all(r[3] == 15.0 for r in res)      # MAX over ranks, identical on every rank
    assert all(r[4] == 6.0 for r in res)       # SUM of units
    assert res[0][5] != res[1][5]              # ranks draw different synthetic data

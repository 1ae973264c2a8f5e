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


# ----------------------------------------------------------------------------- Ulysses exchange
def _global(B, n, H, d):
    """A tensor whose every element names its own (b, token, head, channel): any misplaced element is visible."""
    b = torch.arange(B).view(B, 1, 1, 1) * 1_000_000
    t = torch.arange(n).view(1, n, 1, 1) * 1_000
    h = torch.arange(H).view(1, 1, H, 1) * 10
    c = torch.arange(d).view(1, 1, 1, d)
    return (b + t + h + c).float()


def _ulysses_worker(rank, world, port, q):
    from paper_2606_13872_b200 import ulysses
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ok = True
        # uneven everywhere: 7 tokens over 2 ranks (4 + 3), 3 heads over 2 ranks (2 + 1), 2 chunks -> rank 1's
        # second chunk is empty and must still take part in the exchange
        for B, n, H, d, n_chunks in ((2, 7, 3, 4, 2), (1, 8, 4, 2, 1), (1, 5, 5, 2, 3)):
            g = _global(B, n, H, d)
            t0, nl = dp.shard_range(n, world, rank)
            mine = g[:, t0:t0 + nl].contiguous()
            back = torch.full_like(mine, -1.0)
            for c in range(n_chunks):
                h0, hc = ulysses.head_chunk(H, world, rank, n_chunks, c)
                xh = ulysses.seq_to_heads(mine, n, H, None, n_chunks, c)
                ok &= tuple(xh.shape) == (B, n, hc, d) and torch.equal(xh, g[:, :, h0:h0 + hc])
                ulysses.heads_to_seq(xh, n, H, back, None, n_chunks, c)
            ok &= torch.equal(back, mine)      # the chunks of every rank tile all heads; round trip = identity
        q.put((rank, bool(ok)))
    finally:
        dist.destroy_process_group()


def test_gloo_world2_ulysses_exchange_layout():
    """seq_to_heads gives every rank ALL tokens of exactly its head chunk; heads_to_seq is its inverse."""
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_ulysses_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, True), (1, True)]


def test_head_chunks_partition_the_heads():
    from paper_2606_13872_b200 import ulysses
    for H, world, n_chunks in ((40, 8, 2), (40, 8, 5), (3, 2, 2), (5, 2, 3), (4, 1, 3)):
        seen = []
        for r in range(world):
            for c in range(n_chunks):
                h0, hc = ulysses.head_chunk(H, world, r, n_chunks, c)
                seen.extend(range(h0, h0 + hc))
        assert sorted(seen) == list(range(H))


def test_bench_gpus2_starts_two_ranks_itself():
    """`python bench.py --gpus 2` without a launcher starts its own 2-rank job (torchrun re-exec on 127.0.0.1), rank 0
    alone prints the line and it says n_gpus = 2.  Run with --impl reference (the oracle arm: no GPU needed)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--workload", "tiny"], capture_output=True, text=True, timeout=600, env=env, cwd=root)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    out = json.loads(lines[0])
    assert out["impl"] == "reference" and out["n_gpus"] == 2 and out["value"] > 0

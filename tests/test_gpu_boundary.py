"""-m gpu checks of the boundary contract of include/sra.h (SURVEY.md 8b "no hidden allocations"): device memory is
allocated at sra_create / sra_reserve (or at the first call of an optional path) and never afterwards; contexts are
independent of one another; entry points leave the caller's current device alone."""
import math

import numpy as np
import pytest
import torch

from oracle import c_oracle
from paper_2606_13872_b200 import inputs as sra_inputs
from tests.util import assert_parity

pytestmark = pytest.mark.gpu
NAMES6 = ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")
GRADS = ("dq_gen", "dk_gen", "dv_gen", "dq_ref", "dk_ref", "dv_ref")


def _tensors(w, dev):
    t = sra_inputs.make_inputs(w, with_grad=True)
    g = {k: v.to(dev) for k, v in t.items()}
    g["o_gen"], g["o_ref"] = torch.empty_like(g["q_gen"]), torch.empty_like(g["q_ref"])
    g["lse_gen"] = torch.empty((w.batch, w.heads, w.n_gen), device=dev)
    g["lse_ref"] = torch.empty((w.batch, w.heads, w.n_ref), device=dev)
    for n in GRADS:
        g[n] = torch.empty_like(g["q_gen" if n.endswith("_gen") else "q_ref"])
    return t, g


def _step(B, ctx, g, host):
    """One call of every launching entry point: cache build, forward (fresh K/V and cached), backward, host forward."""
    B.sra_cache_reference_kv(ctx, g["k_ref"], g["v_ref"])
    B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], g["o_gen"], q_ref=g["q_ref"], o_ref=g["o_ref"],
                  lse_gen=g["lse_gen"], lse_ref=g["lse_ref"])
    B.sra_backward(ctx, q_gen=g["q_gen"], k_gen=g["k_gen"], v_gen=g["v_gen"], q_ref=g["q_ref"], k_ref=g["k_ref"],
                   v_ref=g["v_ref"], o_gen=g["o_gen"], o_ref=g["o_ref"], lse_gen=g["lse_gen"], lse_ref=g["lse_ref"],
                   do_gen=g["do_gen"], do_ref=g["do_ref"], **{n: g[n] for n in GRADS})
    B.sra_forward_host(ctx, host["q_gen"], host["k_gen"], host["v_gen"], host["o_gen"], q_ref=host["q_ref"],
                       o_ref=host["o_ref"])
    torch.cuda.synchronize()


HOST_PIPE = sra_inputs.SRAWorkload("host_pipe", 1, 2, 128, 6000, (700, 300), "B", 0)    # >= 16 query slabs: pipelined host path
HOST_PIPE2 = sra_inputs.SRAWorkload("host_pipe2", 2, 2, 128, 4200, (700, 300), "B", 0)  # the same with batch 2


@pytest.mark.parametrize("name,masked", [("host_pipe", False), ("host_pipe2", True), ("mini_train", True), ("short_mini", False)])
def test_no_device_allocation_after_the_second_call(name, masked):
    """cudaMemGetInfo's free-byte count is the same after the 2nd and after the 10th round of cache build + forward +
    backward + host forward (pipelined for host_pipe / host_pipe2, serial for mini_train and the key-split short_mini;
    with per-sample validity masks where `masked`), and - for a context that reserved everything up front - the same
    as right after sra_reserve."""
    from paper_2606_13872_b200 import binding as B
    dev = torch.device("cuda:0")
    w = {"host_pipe": HOST_PIPE, "host_pipe2": HOST_PIPE2}.get(name) or sra_inputs.WORKLOADS[name]
    t, g = _tensors(w, dev)
    host = {n: t[n].pin_memory() for n in ("q_gen", "k_gen", "v_gen", "q_ref")}
    host["o_gen"], host["o_ref"] = torch.empty_like(t["q_gen"]).pin_memory(), torch.empty_like(t["q_ref"]).pin_memory()
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        B.sra_reserve(ctx, B.RESERVE_BACKWARD | B.RESERVE_HOST | B.RESERVE_VALIDITY)
        torch.cuda.synchronize()
        free_reserved = torch.cuda.mem_get_info(dev)[0]
        if masked:
            rng = np.random.default_rng(0)
            B.sra_set_reference_validity(ctx, rng.random((w.batch, w.n_ref)) < 0.7)
        free = []
        for i in range(10):
            _step(B, ctx, g, host)
            free.append(torch.cuda.mem_get_info(dev)[0])
        assert free[1:] == [free[1]] * 9, f"device memory moved between calls: {free}"
        assert free[1] == free_reserved, "a call allocated although every optional path had been reserved"
    finally:
        B.sra_destroy(ctx)
    # the implicit route: nothing reserved, the first round allocates, later rounds do not
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        free = []
        for i in range(5):
            _step(B, ctx, g, host)
            free.append(torch.cuda.mem_get_info(dev)[0])
        assert free[1:] == [free[1]] * 4, f"device memory moved after the first round: {free}"
    finally:
        B.sra_destroy(ctx)


def test_two_contexts_on_one_device_interleaved():
    """Two contexts of different shapes (head_dim 128 pair kernel / head_dim 64 single-CTA kernel), launches
    interleaved on two streams: each result equals the oracle's, neither disturbs the other's cache or schedule."""
    from paper_2606_13872_b200 import binding as B
    dev = torch.device("cuda:0")
    ws = [sra_inputs.WORKLOADS["mini480"], sra_inputs.WORKLOADS["ragged64"]]
    tg = [_tensors(w, dev) for w in ws]
    ctxs = [B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets) for w in ws]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    try:
        torch.cuda.synchronize()
        for rep in range(3):
            for i in (0, 1, 1, 0):
                g = tg[i][1]
                with torch.cuda.stream(streams[i]):
                    if rep == 0:
                        B.sra_cache_reference_kv(ctxs[i], g["k_ref"], g["v_ref"])
                    g["o_gen"].fill_(float("nan"))
                    B.sra_forward(ctxs[i], g["q_gen"], g["k_gen"], g["v_gen"], g["o_gen"], q_ref=g["q_ref"], o_ref=g["o_ref"],
                                  lse_gen=g["lse_gen"], lse_ref=g["lse_ref"])
        torch.cuda.synchronize()
        for i, w in enumerate(ws):
            t, g = tg[i]
            tb = {n: sra_inputs.bf16_bits(t[n]) for n in NAMES6}
            rows = np.arange(w.n_gen + w.n_ref, dtype=np.int32)[:: max(1, (w.n_gen + w.n_ref) // 400)]
            o_or, _ = c_oracle.forward_rows(*[tb[n] for n in NAMES6], w.ref_block_offsets, 1.0 / math.sqrt(w.head_dim), rows)
            gi, ri = rows[rows < w.n_gen], rows[rows >= w.n_gen] - w.n_gen
            got = np.concatenate([g["o_gen"][:, torch.as_tensor(gi, device=dev).long()].float().cpu().numpy(),
                                  g["o_ref"][:, torch.as_tensor(ri, device=dev).long()].float().cpu().numpy()], axis=1)
            assert_parity(got, o_or, f"context {i} ({w.name})")
    finally:
        for c in ctxs:
            B.sra_destroy(c)


def test_entry_points_leave_the_current_device_alone():
    """sra_create and every launching entry point run on the ctx's device and restore the caller's.  With one GPU the
    check is that the current device is unchanged; with two or more, a ctx on device 1 is driven from device 0."""
    from paper_2606_13872_b200 import binding as B
    w = sra_inputs.WORKLOADS["ragged"]
    n_dev = torch.cuda.device_count()
    target = 1 if n_dev >= 2 else 0
    torch.cuda.set_device(0)
    dev = torch.device("cuda", target)
    t, g = _tensors(w, dev)
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets, device=target)
    try:
        assert torch.cuda.current_device() == 0
        s = torch.cuda.Stream(device=dev)
        B.sra_cache_reference_kv(ctx, g["k_ref"], g["v_ref"], stream=s)
        B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], g["o_gen"], q_ref=g["q_ref"], o_ref=g["o_ref"], stream=s)
        assert torch.cuda.current_device() == 0
        s.synchronize()
        tb = {n: sra_inputs.bf16_bits(t[n]) for n in NAMES6}
        rows = np.arange(w.n_gen + w.n_ref, dtype=np.int32)
        o_or, _ = c_oracle.forward_rows(*[tb[n] for n in NAMES6], w.ref_block_offsets, 1.0 / math.sqrt(w.head_dim), rows)
        got = np.concatenate([g["o_gen"].float().cpu().numpy(), g["o_ref"].float().cpu().numpy()], axis=1)
        assert_parity(got, o_or, "ctx on its own device")
    finally:
        B.sra_destroy(ctx)

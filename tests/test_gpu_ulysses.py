"""-m gpu: the head-chunk-pipelined Ulysses driver (paper_2606_13872_b200/ulysses.py) on ONE GPU.

This run has one GPU per call, so the group has world size 1: the all-to-alls are real NCCL calls on the communication
stream (self-exchange), the chunk pipeline, the stream / event ordering and the per-chunk contexts and caches are the
ones an 8-GPU job runs, and the result must match the fp64 oracle of the unsharded problem (contract tolerance:
max-abs <= 2e-2, mean-abs <= 2e-3, rel_l2 <= 1e-2).  The world-size-2 exchange layout is tested on CPU with gloo
(tests/test_dp_gloo.py).  No multi-GPU number is claimed anywhere.
"""
import math
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist

from oracle import sra_oracle
from paper_2606_13872_b200 import inputs as sra_inputs
from tests.gpu_util import bits
from tests.util import assert_parity

pytestmark = pytest.mark.gpu


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


@pytest.mark.parametrize("with_group", [False, True])
@pytest.mark.parametrize("name,n_chunks", [("ragged", 2), ("mini_train", 2), ("ragged64", 1)])
def test_pipelined_head_chunks_match_oracle(name, n_chunks, with_group):
    from paper_2606_13872_b200 import ulysses
    w = sra_inputs.WORKLOADS[name]
    t = sra_inputs.make_inputs(w)
    tb = bits(t)
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    if with_group:
        dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{_free_port()}", rank=0, world_size=1,
                                device_id=dev)
    try:
        g = {k: v.to(dev) for k, v in t.items()}
        u = ulysses.UlyssesSRA(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets, n_chunks=n_chunks)
        try:
            assert u.gen_shard() == (0, w.n_gen) and u.ref_shard() == (0, w.n_ref)
            u.cache_reference_kv(g["k_ref"], g["v_ref"])
            o_gen, o_ref = u.forward(g["q_gen"], g["k_gen"], g["v_gen"], g["q_ref"])          # step 0: G and R rows
            o_gen2, none = u.forward(g["q_gen"], g["k_gen"], g["v_gen"])                      # cached denoising step
            torch.cuda.synchronize()
            assert none is None
            assert u.launches == 2 * u.n_chunks, "one sra_forward per head chunk and step"
        finally:
            u.close()
    finally:
        if with_group:
            dist.destroy_process_group()
    scale = 1.0 / math.sqrt(w.head_dim)
    ref = sra_oracle.sra_forward(tb["q_gen"], tb["k_gen"], tb["v_gen"], tb["q_ref"], tb["k_ref"], tb["v_ref"],
                                 w.ref_block_offsets, scale)
    assert_parity(o_gen.float().cpu().numpy(), ref["o_gen"], f"{name} ulysses O_g")
    assert_parity(o_ref.float().cpu().numpy(), ref["o_ref"], f"{name} ulysses O_r")
    assert torch.equal(o_gen.view(torch.int16), o_gen2.view(torch.int16)), "cached step changed the G rows"


def test_training_step_through_the_head_chunk_pipeline():
    """forward(save_for_backward) + backward on sequence shards (world size 1, NCCL group): every gradient against the
    fp64 oracle of the unsharded problem (contract tolerance + rel_l2 <= 1e-2); B = 2, 3 heads in chunks of 2 + 1."""
    from paper_2606_13872_b200 import ulysses
    w = sra_inputs.WORKLOADS["ragged"]
    t = sra_inputs.make_inputs(w, with_grad=True)
    tb = bits(t)
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{_free_port()}", rank=0, world_size=1, device_id=dev)
    try:
        g = {k: v.to(dev) for k, v in t.items()}
        u = ulysses.UlyssesSRA(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets, n_chunks=2)
        try:
            u.cache_reference_kv(g["k_ref"], g["v_ref"])
            u.forward(g["q_gen"], g["k_gen"], g["v_gen"], g["q_ref"], save_for_backward=True)
            grads = u.backward(g["do_gen"], g["do_ref"])
            torch.cuda.synchronize()
            with pytest.raises(RuntimeError):
                u.backward(g["do_gen"], g["do_ref"])        # the saved tensors are consumed
        finally:
            u.close()
    finally:
        dist.destroy_process_group()
    ref = sra_oracle.sra_backward(tb["q_gen"], tb["k_gen"], tb["v_gen"], tb["q_ref"], tb["k_ref"], tb["v_ref"], tb["do_gen"],
                                  tb["do_ref"], w.ref_block_offsets, 1.0 / math.sqrt(w.head_dim))
    for name, got in zip(("dq_gen", "dk_gen", "dv_gen", "dq_ref", "dk_ref", "dv_ref"), grads):
        assert_parity(got.float().cpu().numpy(), ref[name], f"ulysses {name}")

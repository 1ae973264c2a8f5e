"""-m gpu soak tests of the C-ABI boundary (include/sra.h memory / ordering contract): what a long-running trainer or
server does to the library - many contexts created and destroyed, many steps queued without a host synchronisation
in between, schedules changed between steps - must neither leak device memory, hang, nor change a result.
The arithmetic itself is checked against the oracle elsewhere; here every comparison is against the first step of the
same run (bit identity where the summation order is fixed, a bf16 ulp for dQ - SURVEY.md 8c A13).
"""
import numpy as np
import pytest
import torch

from paper_2606_13872_b200 import inputs as sra_inputs

pytestmark = pytest.mark.gpu
GRADS = ("dq_gen", "dk_gen", "dv_gen", "dq_ref", "dk_ref", "dv_ref")


def _free_bytes():
    torch.cuda.synchronize()
    return torch.cuda.mem_get_info()[0]


def test_create_destroy_cycles_do_not_leak_device_memory():
    """120 contexts, each with every optional buffer reserved, a cache build, a forward and a backward: the free device
    memory after the last sra_destroy equals the one before the first sra_create."""
    from paper_2606_13872_b200 import binding as B
    w = sra_inputs.WORKLOADS["ragged"]
    dev = torch.device("cuda:0")
    g = {k: v.to(dev) for k, v in sra_inputs.make_inputs(w, with_grad=True).items()}
    o_gen, o_ref = torch.empty_like(g["q_gen"]), torch.empty_like(g["q_ref"])
    lse_gen = torch.empty((w.batch, w.heads, w.n_gen), device=dev)
    lse_ref = torch.empty((w.batch, w.heads, w.n_ref), device=dev)
    grads = {n: torch.empty_like(g["q_gen" if n.endswith("_gen") else "q_ref"]) for n in GRADS}
    valid = np.random.default_rng(0).random(w.n_ref) < 0.8

    def cycle(i):
        ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
        try:
            B.sra_reserve(ctx, B.RESERVE_BACKWARD | B.RESERVE_HOST | B.RESERVE_VALIDITY)
            if i % 3 == 1:
                B.sra_set_reference_validity(ctx, valid)
            if i % 3 == 2:
                B.sra_set_temporal_window(ctx, [0, 100, 200, w.n_gen], 1)
            B.sra_cache_reference_kv(ctx, g["k_ref"], g["v_ref"])
            B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, q_ref=g["q_ref"], o_ref=o_ref, lse_gen=lse_gen,
                          lse_ref=lse_ref)
            B.sra_backward(ctx, q_gen=g["q_gen"], k_gen=g["k_gen"], v_gen=g["v_gen"], q_ref=g["q_ref"], k_ref=None, v_ref=None,
                           o_gen=o_gen, o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref, do_gen=g["do_gen"],
                           do_ref=g["do_ref"], **grads)
        finally:
            B.sra_destroy(ctx)

    for i in range(3):          # first uses: module load, per-device function attributes
        cycle(i)
    before = _free_bytes()
    for i in range(120):
        cycle(i)
    after = _free_bytes()
    assert after == before, f"device memory leaked over 120 create / destroy cycles: {before - after} bytes"


def test_many_queued_steps_without_host_synchronisation():
    """150 training steps (forward + backward) queued back to back on one stream, no synchronisation in between, the
    schedule switched (temporal window on / off) every 25 steps: the outputs of the last plain step equal those of the
    first one - O, LSE, dK, dV bit for bit, dQ to a bf16 ulp - and nothing hangs."""
    from paper_2606_13872_b200 import binding as B
    w = sra_inputs.WORKLOADS["mini_train"]
    dev = torch.device("cuda:0")
    g = {k: v.to(dev) for k, v in sra_inputs.make_inputs(w, with_grad=True).items()}
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        B.sra_reserve(ctx, B.RESERVE_BACKWARD)
        o_gen, o_ref = torch.empty_like(g["q_gen"]), torch.empty_like(g["q_ref"])
        lse_gen = torch.empty((w.batch, w.heads, w.n_gen), device=dev)
        lse_ref = torch.empty((w.batch, w.heads, w.n_ref), device=dev)
        grads = {n: torch.empty_like(g["q_gen" if n.endswith("_gen") else "q_ref"]) for n in GRADS}
        frames = [0, 400, 900, 1300, w.n_gen]

        def step():
            B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, q_ref=g["q_ref"], k_ref=g["k_ref"], v_ref=g["v_ref"],
                          o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref)
            B.sra_backward(ctx, q_gen=g["q_gen"], k_gen=g["k_gen"], v_gen=g["v_gen"], q_ref=g["q_ref"], k_ref=g["k_ref"],
                           v_ref=g["v_ref"], o_gen=o_gen, o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref, do_gen=g["do_gen"],
                           do_ref=g["do_ref"], **grads)

        def snapshot():
            torch.cuda.synchronize()
            out = {"o_gen": o_gen, "o_ref": o_ref, "lse_gen": lse_gen, "lse_ref": lse_ref, **grads}
            return {k: v.float().cpu().numpy().copy() for k, v in out.items()}

        step()
        first = snapshot()
        windowed = False
        for i in range(150):
            if i % 25 == 24:
                windowed = not windowed
                B.sra_set_temporal_window(ctx, frames, 1 if windowed else -1)
            step()
        if windowed:
            B.sra_set_temporal_window(ctx, frames, -1)
        step()
        last = snapshot()
    finally:
        B.sra_destroy(ctx)
    for k in first:
        if k.startswith("dq"):
            tol = 2.0 ** -7 * np.maximum(np.abs(first[k]), np.abs(last[k])) + 1e-5 * np.abs(first[k]).max()
            assert (np.abs(first[k] - last[k]) <= tol).all(), k
        else:
            assert np.array_equal(first[k], last[k]), f"{k} changed between the first and the last of 150 queued steps"

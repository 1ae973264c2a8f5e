"""-m gpu parity of the refiner's sparse temporal attention (reading A17): generation
queries see the generation keys of frames within a window plus every reference key.  CUDA path through the C ABI
(sra_set_temporal_window + forward / backward) vs the fp64 oracle that materialises the windowed mask, every row.

Contract tolerance (BASELINE.json north_star): bf16 I/O, fp32 accumulation, max-abs <= 2e-2, mean-abs <= 2e-3, plus
rel_l2 <= 1e-2.
"""
import math

import numpy as np
import pytest
import torch

from oracle import sra_oracle
from paper_2606_13872_b200 import inputs as sra_inputs
from tests.gpu_util import bits
from tests.util import assert_parity

pytestmark = pytest.mark.gpu
GRADS = ("dq_gen", "dk_gen", "dv_gen", "dq_ref", "dk_ref", "dv_ref")


def _run(w, t, fr, window, valid, backward):
    from paper_2606_13872_b200 import binding as B
    dev = torch.device("cuda:0")
    g = {k: v.to(dev) for k, v in t.items()}
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        B.sra_set_temporal_window(ctx, fr, window)
        if valid is not None:
            B.sra_set_reference_validity(ctx, valid)
        nan = float("nan")
        o_gen, o_ref = torch.full_like(g["q_gen"], nan), torch.full_like(g["q_ref"], nan)
        lse_gen = torch.full((w.batch, w.heads, w.n_gen), nan, device=dev)
        lse_ref = torch.full((w.batch, w.heads, w.n_ref), nan, device=dev)
        B.sra_cache_reference_kv(ctx, g["k_ref"], g["v_ref"])
        B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, q_ref=g["q_ref"], o_ref=o_ref, lse_gen=lse_gen,
                      lse_ref=lse_ref)
        out = {"o_gen": o_gen, "o_ref": o_ref, "lse_gen": lse_gen, "lse_ref": lse_ref}
        if backward:
            grads = {n: torch.full_like(g["q_gen" if n.endswith("_gen") else "q_ref"], nan) for n in GRADS}
            B.sra_backward(ctx, q_gen=g["q_gen"], k_gen=g["k_gen"], v_gen=g["v_gen"], q_ref=g["q_ref"], k_ref=None, v_ref=None,
                           o_gen=o_gen, o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref, do_gen=g["do_gen"],
                           do_ref=g["do_ref"], **grads)
            out.update(grads)
        torch.cuda.synchronize()
        return {k: v.float().cpu().numpy() for k, v in out.items()}
    finally:
        B.sra_destroy(ctx)


def _check(w, fr, window, valid=None, backward=True):
    t = sra_inputs.make_inputs(w, with_grad=True)
    got = _run(w, t, fr, window, valid, backward)
    tb = bits(t)
    scale = 1.0 / math.sqrt(w.head_dim)
    a6 = [tb[k] for k in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")]
    kw = dict(valid=valid, gen_frame_offsets=fr, window=window)
    ref = sra_oracle.sra_forward(*a6, w.ref_block_offsets, scale, **kw)
    keep = np.arange(w.n_ref) if valid is None else np.flatnonzero(valid)
    assert_parity(got["o_gen"], ref["o_gen"], f"{w.name} O_g")
    assert np.abs(got["lse_gen"] - ref["lse_gen"]).max() <= 2e-3
    assert_parity(got["o_ref"][:, keep], ref["o_ref"][:, keep], f"{w.name} O_r")
    if backward:
        bref = sra_oracle.sra_backward(*a6, tb["do_gen"], tb["do_ref"], w.ref_block_offsets, scale, **kw)
        for n in GRADS:
            a, b = (got[n], bref[n]) if n.endswith("_gen") else (got[n][:, keep], bref[n][:, keep])
            assert_parity(a, b, f"{w.name} {n}")


@pytest.mark.parametrize("window", [0, 1, 3])
def test_temporal_window_ragged_frames(window):
    """Frames that do not divide 128 / 256, ragged reference blocks, B2 H3 d128; forward and backward."""
    w = sra_inputs.SRAWorkload("temporal_ragged", 2, 3, 128, 1000, (130, 257, 64), "B", 0)
    _check(w, [0, 100, 357, 400, 777, 1000], window)


def test_temporal_window_real_frames_with_validity():
    """Four real 1560-token latent frames, window 1, with a third of the reference marked invalid."""
    w = sra_inputs.SRAWorkload("temporal_480", 1, 2, 128, 4 * 1560, (1560, 300), "B", 0)
    valid = np.random.default_rng(3).random(w.n_ref) < 0.67
    _check(w, [0, 1560, 3120, 4680, 6240], 1, valid=valid)


def test_temporal_window_covering_everything_is_plain_sra():
    from tests.gpu_util import run_gpu_forward
    w = sra_inputs.WORKLOADS["ragged"]
    t = sra_inputs.make_inputs(w, with_grad=True)
    base = run_gpu_forward(w, t, use_cache=True)
    got = _run(w, t, [0, 100, 200, 333], 2, None, backward=False)
    # (GPU against GPU: the same mask through a different slab partition.  The frame-cut slabs have one Q tile per CTA and
    # run in dual-slot mode - two partial softmax states merged at the end - so the two results differ by the bf16
    # rounding of P against different reference maxima; each is checked against the oracle in the tests above.)
    assert_parity(got["o_gen"], base["o_gen"], "window >= n_frames - 1", rel_l2_tol=5e-3)
    assert np.array_equal(got["o_ref"], base["o_ref"])


def test_temporal_window_through_the_pipelined_host_path():
    """sra_forward_host with a temporal window: the query slabs are cut at frame boundaries (not all 256 rows), so
    the host pipeline must take its copy ranges from the schedule; checked against the oracle, every row."""
    from paper_2606_13872_b200 import binding as B
    fr = [0, 700, 1500, 2100, 3000, 3701, 4500]                      # 6 ragged frames, 24 slabs -> pipelined
    w = sra_inputs.SRAWorkload("tw_host", 1, 2, 128, fr[-1], (300, 260), "B", 0)
    t = sra_inputs.make_inputs(w)
    dev = torch.device("cuda:0")
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        B.sra_set_temporal_window(ctx, fr, 1)
        B.sra_cache_reference_kv(ctx, t["k_ref"].to(dev), t["v_ref"].to(dev))
        h = {k: t[k].pin_memory() for k in ("q_gen", "k_gen", "v_gen", "q_ref")}
        o_gen = torch.full(t["q_gen"].shape, float("nan"), dtype=torch.bfloat16).pin_memory()
        o_ref = torch.full(t["q_ref"].shape, float("nan"), dtype=torch.bfloat16).pin_memory()
        lse_gen = torch.full((w.batch, w.heads, w.n_gen), float("nan")).pin_memory()
        B.sra_forward_host(ctx, h["q_gen"], h["k_gen"], h["v_gen"], o_gen, q_ref=h["q_ref"], o_ref=o_ref, lse_gen=lse_gen)
        torch.cuda.synchronize()
    finally:
        B.sra_destroy(ctx)
    tb = bits(t)
    ref = sra_oracle.sra_forward(tb["q_gen"], tb["k_gen"], tb["v_gen"], tb["q_ref"], tb["k_ref"], tb["v_ref"],
                                 w.ref_block_offsets, 1.0 / math.sqrt(w.head_dim), gen_frame_offsets=fr, window=1)
    assert_parity(o_gen.float().numpy(), ref["o_gen"], "windowed host path O_g")
    assert_parity(o_ref.float().numpy(), ref["o_ref"], "windowed host path O_r")
    assert np.abs(lse_gen.numpy() - ref["lse_gen"]).max() <= 2e-3

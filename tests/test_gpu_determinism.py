"""-m gpu: run-to-run determinism as a race detector (compute-sanitizer is closed on this GPU pool).

The forward kernels contain no atomics and no data-dependent scheduling: every launch of the same problem must return
the same bytes, on a quiet GPU and with another stream keeping the SMs busy.  In the backward, dK and dV are
accumulated in TMEM by one CTA per key tile in a fixed order (bit-identical); dQ is accumulated with red.global.add
across key tiles in arrival order, so it is only required to agree to fp32 reassociation (one bf16 ulp at the scale
of the tensor).
A missing barrier, a TMEM or shared-memory buffer reused too early, or a read of a tile that has not landed shows up
here as a run-to-run difference.
"""
import numpy as np
import pytest
import torch

from paper_2606_13872_b200 import inputs as sra_inputs

pytestmark = pytest.mark.gpu
GRADS = ("dq_gen", "dk_gen", "dv_gen", "dq_ref", "dk_ref", "dv_ref")


def _noise(stream, n):
    """Unrelated work on another stream, so that CTAs of the kernels under test are scheduled irregularly."""
    with torch.cuda.stream(stream):
        a = torch.randn(2048, 2048, device="cuda:0")
        for _ in range(n):
            a = (a @ a).clamp_(-1, 1)
    return a


@pytest.mark.parametrize("name", ["ragged", "mini720", "short_mini", "ragged64"])
def test_forward_is_bit_reproducible(name):
    from paper_2606_13872_b200 import binding as B
    w = sra_inputs.WORKLOADS[name]
    dev = torch.device("cuda:0")
    g = {k: v.to(dev) for k, v in sra_inputs.make_inputs(w).items()}
    side = torch.cuda.Stream()
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        B.sra_cache_reference_kv(ctx, g["k_ref"], g["v_ref"])
        ref = None
        for rep in range(12):
            o_gen = torch.full_like(g["q_gen"], float("nan"))
            o_ref = torch.full_like(g["q_ref"], float("nan"))
            lse_gen = torch.full((w.batch, w.heads, w.n_gen), float("nan"), device=dev)
            keep = _noise(side, 6) if rep % 2 else None
            B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, q_ref=g["q_ref"], o_ref=o_ref, lse_gen=lse_gen)
            torch.cuda.synchronize()
            del keep
            cur = (o_gen.view(torch.int16).clone(), o_ref.view(torch.int16).clone(), lse_gen.view(torch.int32).clone())
            if ref is None:
                ref = cur
            else:
                for a, b, what in zip(cur, ref, ("o_gen", "o_ref", "lse_gen")):
                    assert torch.equal(a, b), f"{name}: {what} differs between launch 0 and launch {rep}"
    finally:
        B.sra_destroy(ctx)


@pytest.mark.parametrize("name", ["ragged", "ragged64"])
def test_backward_dk_dv_bit_reproducible_dq_to_reassociation(name):
    from paper_2606_13872_b200 import binding as B
    w = sra_inputs.WORKLOADS[name].replace(dist="B")
    dev = torch.device("cuda:0")
    g = {k: v.to(dev) for k, v in sra_inputs.make_inputs(w, with_grad=True).items()}
    side = torch.cuda.Stream()
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        o_gen, o_ref = torch.empty_like(g["q_gen"]), torch.empty_like(g["q_ref"])
        lse_gen = torch.empty((w.batch, w.heads, w.n_gen), device=dev)
        lse_ref = torch.empty((w.batch, w.heads, w.n_ref), device=dev)
        B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, q_ref=g["q_ref"], k_ref=g["k_ref"], v_ref=g["v_ref"],
                      o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref)
        ref = None
        for rep in range(8):
            outs = {n: torch.full_like(g["q_gen" if n.endswith("_gen") else "q_ref"], float("nan")) for n in GRADS}
            keep = _noise(side, 6) if rep % 2 else None
            B.sra_backward(ctx, q_gen=g["q_gen"], k_gen=g["k_gen"], v_gen=g["v_gen"], q_ref=g["q_ref"], k_ref=g["k_ref"],
                           v_ref=g["v_ref"], o_gen=o_gen, o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref,
                           do_gen=g["do_gen"], do_ref=g["do_ref"], **outs)
            torch.cuda.synchronize()
            del keep
            if ref is None:
                ref = {n: v.clone() for n, v in outs.items()}
                continue
            for n in GRADS:
                if n.startswith("dq"):
                    a, b = outs[n].float(), ref[n].float()
                    # fp32 reassociation error scales with the terms, not with a (possibly cancelled) result: one bf16
                    # ulp at the larger of the element and the tensor's rms
                    ulp = 2.0 ** -7 * torch.maximum(b.abs(), b.pow(2).mean().sqrt())
                    assert bool(((a - b).abs() <= ulp).all()), f"{name}: {n} differs by more than one bf16 ulp at launch {rep}"
                else:
                    assert torch.equal(outs[n].view(torch.int16), ref[n].view(torch.int16)), \
                        f"{name}: {n} differs between launch 0 and launch {rep}"
    finally:
        B.sra_destroy(ctx)

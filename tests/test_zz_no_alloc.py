"""-m gpu: sra_forward_gen_static, the entry point that allocates nothing (include/sra.h; an addition outside SURVEY.md 8).

Its scratch - work items and key-split partials - is a file-scope `static __device__` array inside the library
(csrc/sra_static.cu), shared by every call.  Checked here against the EXISTING path (sra_create + sra_forward with the
same explicit reference K / V, reference rows skipped) within the contract tolerance of the other tests - bf16 I/O, fp32
accumulation, max-abs <= 2e-2, mean-abs <= 2e-3, rel_l2 <= 1e-2, LSE max-abs <= 2e-3 - on two calls in a row with
different shapes, so the second call finds the first one's bytes in the array.

This file sorts last on purpose (the suite runs with pytest -x: a failure here hides nothing behind it) and passes both
alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest
import torch

from paper_2606_13872_b200 import inputs as sra_inputs
from tests.util import assert_parity

pytestmark = pytest.mark.gpu
NAN = float("nan")


def _existing_path(w, g):
    """(O_g, LSE_g, n_split) of sra_forward on a context: explicit k_ref / v_ref, q_ref = NULL (G rows only)."""
    from paper_2606_13872_b200 import binding as B
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        n_split, _ = B.sra_split_schedule_copy(ctx)
        o = torch.full_like(g["q_gen"], NAN)
        lse = torch.full((w.batch, w.heads, w.n_gen), NAN, device=o.device)
        has_ref = w.n_ref > 0
        B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o, k_ref=g["k_ref"] if has_ref else None,
                      v_ref=g["v_ref"] if has_ref else None, lse_gen=lse)
        torch.cuda.synchronize()
        return o.float().cpu().numpy(), lse.cpu().numpy(), n_split
    finally:
        B.sra_destroy(ctx)


def _static_path(w, g, n_split):
    from paper_2606_13872_b200 import binding as B
    o = torch.full_like(g["q_gen"], NAN)
    lse = torch.full((w.batch, w.heads, w.n_gen), NAN, device=o.device)
    has_ref = w.n_ref > 0
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    B.sra_forward_gen_static(g["q_gen"], g["k_gen"], g["v_gen"], o, k_ref=g["k_ref"] if has_ref else None,
                             v_ref=g["v_ref"] if has_ref else None, lse_gen=lse, n_split=n_split)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    return o.float().cpu().numpy(), lse.cpu().numpy(), free0 - free1


def _compare(w, got, ref, what):
    assert_parity(got[0], ref[0], f"{what} O_g")
    assert np.abs(got[1] - ref[1]).max() <= 2e-3, f"{what} LSE_g"


def test_static_entry_matches_the_context_path_on_two_calls_in_a_row():
    dev = torch.device("cuda:0")
    # call 1: d = 128, 100 rows against 3420 reference keys; call 2: d = 64, another shape - the partials of call 1 are
    # still in the array, at other offsets and strides; call 3: call 1's problem again, over call 2's bytes
    shapes = [sra_inputs.WORKLOADS["short_mini"], sra_inputs.WORKLOADS["short_mini64"], sra_inputs.WORKLOADS["short_mini"]]
    refs, inputs = [], []
    for w in shapes:
        g = {k: v.to(dev) for k, v in sra_inputs.make_inputs(w).items()}
        inputs.append(g)
        refs.append(_existing_path(w, g))
    assert refs[0][2] > 1, "the context path of this shape is the key-split one"
    for i, (w, g, ref) in enumerate(zip(shapes, inputs, refs)):
        got = _static_path(w, g, n_split=ref[2])            # the same key ranges as the context's schedule
        _compare(w, got, ref, f"call {i + 1} ({w.name}, n_split {ref[2]})")
        # (the very first call of a process does the once-per-device set-up; after it nothing is allocated or freed)
        assert i == 0 or got[2] == 0, f"device memory changed by {got[2]} bytes across static call {i + 1}"
    # automatic split count, and a plain self-attention problem (no reference) with an explicit one
    got = _static_path(shapes[0], inputs[0], n_split=0)
    _compare(shapes[0], got, refs[0], "automatic n_split")
    w = sra_inputs.SRAWorkload("static_noref", 2, 3, 128, 333, (), "B", 0)
    g = {k: v.to(dev) for k, v in sra_inputs.make_inputs(w).items()}
    _compare(w, _static_path(w, g, n_split=2), _existing_path(w, g), "no reference, n_split 2")


def test_static_entry_rejects_what_does_not_fit():
    from paper_2606_13872_b200 import binding as B
    dev = torch.device("cuda:0")
    # 40 heads x 2048 rows x 7 key ranges of fp32 partials = 296 MB: beyond the 32 MiB array
    assert B.sra_static_scratch_bytes(1, 40, 128, 2048, 7) > B.STATIC_SCRATCH_BYTES
    q = torch.zeros((1, 2048, 40, 128), dtype=torch.bfloat16, device=dev)
    o = torch.empty_like(q)
    with pytest.raises(B.SRAError) as e:
        B.sra_forward_gen_static(q, q, q, o, n_split=7)
    assert e.value.status == B.SRA_ERR_INVALID_ARG and "bytes of scratch" in str(e.value)
    with pytest.raises(B.SRAError) as e:
        B.sra_forward_gen_static(q[:, :100], q[:, :100], q[:, :100], o[:, :100], n_split=2)   # 1 key tile, 2 ranges
    assert e.value.status == B.SRA_ERR_INVALID_ARG
    # and the library still works afterwards
    w = sra_inputs.WORKLOADS["short_mini"]
    g = {k: v.to(dev) for k, v in sra_inputs.make_inputs(w).items()}
    ref = _existing_path(w, g)
    _compare(w, _static_path(w, g, n_split=ref[2]), ref, "after the rejected calls")

"""-m gpu: error behaviour of the C ABI on a real device (include/sra.h: int status, message in sra_last_error, no
abort, the context stays usable).  Argument errors are returned synchronously, before any launch."""
import pytest
import torch

from paper_2606_13872_b200 import inputs as sra_inputs

pytestmark = pytest.mark.gpu


def test_argument_errors_are_reported_and_the_context_survives():
    from paper_2606_13872_b200 import binding as B
    w = sra_inputs.WORKLOADS["ragged"]
    dev = torch.device("cuda:0")
    g = {k: v.to(dev) for k, v in sra_inputs.make_inputs(w, with_grad=True).items()}
    o_gen, o_ref = torch.empty_like(g["q_gen"]), torch.empty_like(g["q_ref"])
    lse_gen = torch.empty((w.batch, w.heads, w.n_gen), device=dev)
    lse_ref = torch.empty((w.batch, w.heads, w.n_ref), device=dev)
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        n0 = B.sra_launch_count(ctx)

        def expect(status, fn, *a, **kw):
            with pytest.raises(B.SRAError) as e:
                fn(*a, **kw)
            assert e.value.status == status, e.value
            assert B.sra_launch_count(ctx) == n0, "an argument error must not launch anything"

        # no resident cache yet, and the caller passes no reference K/V
        expect(B.SRA_ERR_NO_REF_CACHE, B.sra_forward, ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen)
        host = {k: g[k].cpu().pin_memory() for k in ("q_gen", "k_gen", "v_gen")}
        expect(B.SRA_ERR_NO_REF_CACHE, B.sra_forward_host, ctx, host["q_gen"], host["k_gen"], host["v_gen"], o_gen.cpu().pin_memory())
        # k_ref without v_ref; q_ref without o_ref; missing required tensors
        expect(B.SRA_ERR_INVALID_ARG, B.sra_forward, ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, k_ref=g["k_ref"])
        expect(B.SRA_ERR_INVALID_ARG, B.sra_forward, ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, q_ref=g["q_ref"],
               k_ref=g["k_ref"], v_ref=g["v_ref"])
        expect(B.SRA_ERR_INVALID_ARG, B.sra_forward, ctx, g["q_gen"], None, g["v_gen"], o_gen)
        # base pointers must be 16-byte aligned (TMA)
        skew = torch.empty(g["q_gen"].numel() + 8, dtype=torch.bfloat16, device=dev)[1:1 + g["q_gen"].numel()].view_as(g["q_gen"])
        assert skew.data_ptr() % 16 != 0
        expect(B.SRA_ERR_INVALID_ARG, B.sra_forward, ctx, skew, g["k_gen"], g["v_gen"], o_gen, k_ref=g["k_ref"], v_ref=g["v_ref"])
        # backward: every generation tensor, and with a reference every reference tensor, is required
        grads = {n: torch.empty_like(g["q_gen" if n.endswith("_gen") else "q_ref"])
                 for n in ("dq_gen", "dk_gen", "dv_gen", "dq_ref", "dk_ref", "dv_ref")}
        full = dict(q_gen=g["q_gen"], k_gen=g["k_gen"], v_gen=g["v_gen"], q_ref=g["q_ref"], k_ref=g["k_ref"], v_ref=g["v_ref"],
                    o_gen=o_gen, o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref, do_gen=g["do_gen"], do_ref=g["do_ref"], **grads)
        expect(B.SRA_ERR_INVALID_ARG, B.sra_backward, ctx, **{**full, "lse_gen": None})
        expect(B.SRA_ERR_INVALID_ARG, B.sra_backward, ctx, **{**full, "do_ref": None})
        expect(B.SRA_ERR_NO_REF_CACHE, B.sra_backward, ctx, **{**full, "k_ref": None, "v_ref": None})
        # RoPE tables are required by the rotating producer
        expect(B.SRA_ERR_INVALID_ARG, B.sra_cache_reference_kv_rope, ctx, g["k_ref"], g["v_ref"], None, None)
        # ... and after all that the context still works
        B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, q_ref=g["q_ref"], k_ref=g["k_ref"], v_ref=g["v_ref"],
                      o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref)
        B.sra_backward(ctx, **full)
        torch.cuda.synchronize()
        assert torch.isfinite(o_gen.float()).all() and all(torch.isfinite(v.float()).all() for v in grads.values())
    finally:
        B.sra_destroy(ctx)


def test_create_rejects_what_the_kernels_do_not_support():
    from paper_2606_13872_b200 import binding as B
    for kw, status in ((dict(head_dim=96), B.SRA_ERR_UNSUPPORTED), (dict(n_gen=0), B.SRA_ERR_INVALID_ARG),
                       (dict(ref_block_offsets=[0, 5, 5]), B.SRA_ERR_INVALID_ARG)):
        args = dict(batch=1, heads=2, head_dim=128, n_gen=64, ref_block_offsets=[0, 16])
        args.update(kw)
        with pytest.raises(B.SRAError) as e:
            B.sra_create(args["batch"], args["heads"], args["head_dim"], args["n_gen"], args["ref_block_offsets"])
        assert e.value.status == status

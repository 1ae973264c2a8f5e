"""-m gpu: the launching entry points are CUDA-graph capturable once warm (include/sra.h: no allocation, no stream or
event creation, no synchronisation on a steady-state call) - the launch-bound short-query loop (two sub-millisecond
kernels per step) can be replayed as one graph.  Replay must return the bytes of the eager calls."""
import numpy as np
import pytest
import torch

from paper_2606_13872_b200 import inputs as sra_inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name", ["short_mini", "mini480"])
def test_cached_steps_replay_from_a_cuda_graph(name):
    """short_mini: key-split schedule (forward + merge kernel per step); mini480: the CTA-pair kernel (cluster launch)."""
    from paper_2606_13872_b200 import binding as B
    w = sra_inputs.WORKLOADS[name]
    dev = torch.device("cuda:0")
    steps = 4
    ref = {n: sra_inputs.make_tensor_device(w, n, dev) for n in ("k_ref", "v_ref")}
    gens = [{n: sra_inputs.make_tensor_device(w, n, dev, step=s) for n in ("q_gen", "k_gen", "v_gen")} for s in range(steps)]
    outs = [torch.empty_like(g["q_gen"]) for g in gens]
    lses = [torch.empty((w.batch, w.heads, w.n_gen), device=dev) for _ in gens]
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        B.sra_cache_reference_kv(ctx, ref["k_ref"], ref["v_ref"])
        for s in range(steps):  # eager (also the warm-up: schedule upload, tensor maps, shared-memory opt-in)
            B.sra_forward(ctx, gens[s]["q_gen"], gens[s]["k_gen"], gens[s]["v_gen"], outs[s], lse_gen=lses[s])
        torch.cuda.synchronize()
        eager = [(o.clone(), l.clone()) for o, l in zip(outs, lses)]
        for o, l in zip(outs, lses):
            o.fill_(float("nan")); l.fill_(float("nan"))
        launches0 = B.sra_launch_count(ctx)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):  # capture on torch's capture stream = the binding's current stream
            for s in range(steps):
                B.sra_forward(ctx, gens[s]["q_gen"], gens[s]["k_gen"], gens[s]["v_gen"], outs[s], lse_gen=lses[s])
        captured = B.sra_launch_count(ctx) - launches0
        n_split, _ = B.sra_split_schedule_copy(ctx)
        assert captured == steps * (2 if n_split > 1 else 1)
        torch.cuda.synchronize()
        assert all(torch.isnan(o.float()).all() for o in outs), "capture must not execute anything"
        for _ in range(2):
            graph.replay()
        torch.cuda.synchronize()
        for s in range(steps):
            assert torch.equal(outs[s], eager[s][0]) and torch.equal(lses[s], eager[s][1]), f"step {s}"
    finally:
        B.sra_destroy(ctx)

"""-m gpu parity on the degenerate shapes of the method (forward and backward, every element, vs the numpy oracle that
materialises the mask): one generation token, one-token reference blocks, no reference at all, slab counts that leave a
CTA pair half empty, batch > 1 on those.  head_dim 128 runs the CTA-pair forward kernel, head_dim 64 the single-CTA one.

Contract tolerance: bf16 I/O, fp32 accumulation, max-abs <= 2e-2, mean-abs <= 2e-3, rel_l2 <= 1e-2, LSE <= 2e-3."""
import math

import numpy as np
import pytest

from oracle import sra_oracle
from paper_2606_13872_b200 import inputs as sra_inputs
from tests.gpu_util import bits, run_gpu_forward
from tests.test_gpu_backward import GRADS, run_gpu_fwd_bwd
from tests.util import assert_parity

pytestmark = pytest.mark.gpu

SHAPES = {
    "one_token": (1, 1, 1, ()),                 # B, H, n_gen, reference blocks: a single query = a single key
    "one_token_one_ref": (1, 2, 1, (1,)),       # one generation token, a one-token reference
    "unit_blocks": (2, 2, 129, (1, 1, 1, 2)),   # one-token blocks: each reference row sees itself only
    "odd_slabs": (1, 2, 513, (600,)),           # 3 slabs -> a full pair + a pair whose second CTA is empty
    "odd_slabs_b2": (2, 1, 257, (257, 255)),    # the same per block, batch 2
    "gen_only_odd": (1, 2, 769, ()),            # no reference: plain self-attention, 3 slabs + 1 row
}


@pytest.mark.parametrize("head_dim", [128, 64])
@pytest.mark.parametrize("name", sorted(SHAPES))
def test_degenerate_shapes_forward_backward(name, head_dim):
    B_, H, n_gen, blocks = SHAPES[name]
    w = sra_inputs.SRAWorkload(name, B_, H, head_dim, n_gen, blocks, "B", 3)
    t = sra_inputs.make_inputs(w, with_grad=True)
    tb = bits(t)
    scale = 1.0 / math.sqrt(head_dim)
    a6 = [tb.get(k) for k in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")]
    ref = sra_oracle.sra_forward(*a6, w.ref_block_offsets, scale)
    for use_cache in ((True, False) if w.n_ref else (False,)):
        out = run_gpu_forward(w, t, use_cache=use_cache)
        assert_parity(out["o_gen"], ref["o_gen"], f"{name} d{head_dim} O_g cache={use_cache}")
        assert np.abs(out["lse_gen"] - ref["lse_gen"]).max() <= 2e-3
        if w.n_ref:
            assert_parity(out["o_ref"], ref["o_ref"], f"{name} d{head_dim} O_r cache={use_cache}")
            assert np.abs(out["lse_ref"] - ref["lse_ref"]).max() <= 2e-3
    bref = sra_oracle.sra_backward(*a6, tb["do_gen"], tb.get("do_ref"), w.ref_block_offsets, scale)
    got = run_gpu_fwd_bwd(w, t, use_cache=False)
    for n in GRADS:
        if got[n] is None:
            continue
        assert np.isfinite(got[n]).all()
        # (a row with a single visible key has P = 1 and dS = 0: dQ of a one-token block is exactly 0 in the oracle and
        # rounding noise on the GPU - the relative gate has no denominator there, the absolute ones still apply)
        rel = 1e-2 if np.abs(bref[n]).max() > 1e-5 else float("inf")
        assert_parity(got[n], bref[n], f"{name} d{head_dim} {n}", rel_l2_tol=rel)

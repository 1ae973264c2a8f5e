"""-m gpu: the SRA mask isolates non-finite data too (SURVEY.md 8c (iii) asks for finite poison; this goes further).

A query must be unaffected by keys / values it does not see ("reference tokens only self-attend",
PAPER.md:143 local temporal window) even when those hold Inf or NaN.  Masked probabilities are exactly 0, but
0 * Inf = NaN inside an MMA, so the ragged last tile of a segment must not contain the neighbouring block's / frame's
rows at all: the kernels load such tiles through tensor maps bounded at the segment end (TMA zero fill;
csrc/sra_common.h BoundMaps).  Every check is bit identity against the run on clean inputs, on the rows that do not
see the poison; the rows that do see it are expected to be non-finite.
"""
import numpy as np
import pytest
import torch

from paper_2606_13872_b200 import inputs as sra_inputs
from tests.gpu_util import run_gpu_forward
from tests.test_gpu_backward import run_gpu_fwd_bwd
from tests.test_gpu_temporal import _run as run_windowed

pytestmark = pytest.mark.gpu
NAN, INF = float("nan"), float("inf")


def _same(name, a, b):
    """Bit identity - except dQ, whose fp32 partial sums meet in L2 in an order that differs from run to run (SURVEY.md
    8c A13): there, finite and equal to a bf16 ulp (plus the fp32 reordering noise of a sum that cancels)."""
    if not name.startswith("dq"):
        return np.array_equal(a, b)
    tol = 2.0 ** -7 * np.maximum(np.abs(a), np.abs(b)) + 1e-5 * np.abs(a).max()
    return bool(np.isfinite(b).all() and (np.abs(a - b) <= tol).all())


def _poison_rows(x, rows):
    """Rows `rows` (token axis 1) of a [B, N, H, d] tensor: NaN, +Inf and -Inf interleaved along d."""
    x[:, rows] = NAN
    x[:, rows, :, 1::3] = INF
    x[:, rows, :, 2::3] = -INF


@pytest.mark.parametrize("name,j", [("ragged", 2), ("ragged", 1), ("ragged64", 1), ("ragged64", 2)])
@pytest.mark.parametrize("use_cache", [True, False])
def test_forward_reference_rows_ignore_nonfinite_unseen_keys(name, j, use_cache):
    """Everything an R query of block j must not see - every generation key / value, every other reference block -
    holds NaN / Inf: O_r and LSE_r of block j are bit-identical to the clean run (blocks end mid-tile: the tile tail
    would otherwise hold the next block's rows)."""
    w = sra_inputs.WORKLOADS[name]
    t = sra_inputs.make_inputs(w)
    base = run_gpu_forward(w, t, use_cache=use_cache)
    off = w.ref_block_offsets
    tp = {k: v.clone() for k, v in t.items()}
    other = np.r_[0:off[j], off[j + 1]:w.n_ref]
    for n in ("k_ref", "v_ref"):
        _poison_rows(tp[n], other)
    for n in ("k_gen", "v_gen"):
        _poison_rows(tp[n], np.arange(w.n_gen))
    pois = run_gpu_forward(w, tp, use_cache=use_cache)
    sl = slice(off[j], off[j + 1])
    assert np.isfinite(base["o_ref"][:, sl]).all()
    assert np.array_equal(base["o_ref"][:, sl], pois["o_ref"][:, sl]), "O_r of the clean block changed"
    assert np.array_equal(base["lse_ref"][:, :, sl], pois["lse_ref"][:, :, sl])
    assert not np.isfinite(pois["o_gen"]).any(), "generation rows see the poisoned keys: they cannot be finite"


@pytest.mark.parametrize("name,j", [("ragged", 2), ("ragged64", 1)])
def test_backward_reference_block_ignores_nonfinite_queries_of_other_blocks(name, j):
    """Q_r and dO_r of every other reference block hold NaN / Inf (nothing a generation row ever reads): all generation
    gradients and dQ_r, dK_r, dV_r of block j are bit-identical to the clean run - the last query tile of block j
    would otherwise carry the next block's Q / dO rows into dK += dS^T Q and dV += P^T dO with dS = P = 0."""
    w = sra_inputs.WORKLOADS[name]
    t = sra_inputs.make_inputs(w, with_grad=True)
    base = run_gpu_fwd_bwd(w, t)
    off = w.ref_block_offsets
    tp = {k: v.clone() for k, v in t.items()}
    other = np.r_[0:off[j], off[j + 1]:w.n_ref]
    for n in ("q_ref", "do_ref"):
        _poison_rows(tp[n], other)
    pois = run_gpu_fwd_bwd(w, tp)
    sl = slice(off[j], off[j + 1])
    for n in ("dq_gen", "dk_gen", "dv_gen"):
        assert _same(n, base[n], pois[n]), f"{n} changed"
    for n in ("dq_ref", "dk_ref", "dv_ref"):
        assert np.isfinite(base[n][:, sl]).all()
        assert _same(n, base[n][:, sl], pois[n][:, sl]), f"{n} of the clean block changed"


@pytest.mark.parametrize("use_cache", [True, False])
def test_backward_dq_of_a_block_ignores_nonfinite_keys_of_other_blocks(use_cache):
    """K_r / V_r of the other blocks hold NaN / Inf.  The generation rows see them (their gradients are non-finite, and
    so are dK_r / dV_r, which collect from the generation queries), but dQ_r of block j depends on block j's keys only:
    bit-identical - the block's last key tile would otherwise feed the next block's K rows into dQ^T = K^T dS^T."""
    w = sra_inputs.WORKLOADS["ragged"]
    j = 2
    t = sra_inputs.make_inputs(w, with_grad=True)
    base = run_gpu_fwd_bwd(w, t, use_cache=use_cache)
    off = w.ref_block_offsets
    tp = {k: v.clone() for k, v in t.items()}
    other = np.r_[0:off[j], off[j + 1]:w.n_ref]
    for n in ("k_ref", "v_ref"):
        _poison_rows(tp[n], other)
    pois = run_gpu_fwd_bwd(w, tp, use_cache=use_cache)
    sl = slice(off[j], off[j + 1])
    assert _same("dq_ref", base["dq_ref"][:, sl], pois["dq_ref"][:, sl]), "dQ_r of the clean block changed"


@pytest.mark.parametrize("f", [1, 3])
def test_temporal_window_isolates_nonfinite_frames(f):
    """Window 0: the queries of frame f see the generation keys of frame f only (plus the reference).
    Q, K, V and dO of every OTHER frame hold NaN / Inf: O_g, LSE_g, dQ_g, dK_g, dV_g of frame f are bit-identical to the
    clean run (frames end mid-tile, forward and backward)."""
    fr = [0, 100, 357, 400, 777, 1000]
    w = sra_inputs.SRAWorkload("nonfinite_frames", 2, 2, 128, fr[-1], (130, 257, 64), "B", 0)
    t = sra_inputs.make_inputs(w, with_grad=True)
    base = run_windowed(w, t, fr, 0, None, True)
    tp = {k: v.clone() for k, v in t.items()}
    other = np.r_[0:fr[f], fr[f + 1]:w.n_gen]
    for n in ("q_gen", "k_gen", "v_gen", "do_gen"):
        _poison_rows(tp[n], other)
    pois = run_windowed(w, tp, fr, 0, None, True)
    sl = slice(fr[f], fr[f + 1])
    for n in ("o_gen", "dq_gen", "dk_gen", "dv_gen"):
        assert np.isfinite(base[n][:, sl]).all()
        assert _same(n, base[n][:, sl], pois[n][:, sl]), f"{n} of the clean frame changed"
    assert np.array_equal(base["lse_gen"][:, :, sl], pois["lse_gen"][:, :, sl])
    # the reference rows never see a generation key
    assert np.array_equal(base["o_ref"], pois["o_ref"])
    assert _same("dq_ref", base["dq_ref"], pois["dq_ref"])


def test_per_sample_validity_isolates_nonfinite_invalid_tokens():
    """Per-sample validity masks (reading A12): invalid reference tokens hold NaN / Inf in Q, K and V; the
    valid rows' outputs are bit-identical to the clean run, and invalid rows stay exactly 0."""
    from paper_2606_13872_b200 import binding as B
    w = sra_inputs.SRAWorkload("nonfinite_valid", 2, 2, 128, 300, (130, 257, 64), "B", 0)
    rng = np.random.default_rng(5)
    valid = rng.random((w.batch, w.n_ref)) < 0.7
    t = sra_inputs.make_inputs(w)
    dev = torch.device("cuda:0")

    def run(tt):
        g = {k: v.to(dev) for k, v in tt.items()}
        ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
        try:
            B.sra_set_reference_validity(ctx, valid)
            o_gen, o_ref = torch.full_like(g["q_gen"], NAN), torch.full_like(g["q_ref"], NAN)
            B.sra_cache_reference_kv(ctx, g["k_ref"], g["v_ref"])
            B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, q_ref=g["q_ref"], o_ref=o_ref)
            torch.cuda.synchronize()
            return o_gen.float().cpu().numpy(), o_ref.float().cpu().numpy()
        finally:
            B.sra_destroy(ctx)

    base = run(t)
    tp = {k: v.clone() for k, v in t.items()}
    for b in range(w.batch):
        bad = np.flatnonzero(~valid[b])
        for n in ("q_ref", "k_ref", "v_ref"):
            x = tp[n][b:b + 1]
            _poison_rows(x, bad)
    pois = run(tp)
    assert np.isfinite(base[0]).all()
    assert np.array_equal(base[0], pois[0]), "O_g changed when invalid reference tokens were poisoned"
    assert np.array_equal(base[1], pois[1]), "O_r changed when invalid reference tokens were poisoned"
    for b in range(w.batch):
        assert not pois[1][b, ~valid[b]].any()

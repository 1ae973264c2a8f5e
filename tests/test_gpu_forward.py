"""-m gpu parity tests of the SRA forward: CUDA path (through the C ABI) vs the fp64 oracle.

Contract tolerance (BASELINE.json north_star): bf16 I/O, fp32 accumulation, GPU vs oracle
max-abs <= 2e-2 and mean-abs <= 2e-3; plus the self-imposed relative gate rel_l2 <= 1e-2
(SURVEY.md 8c "tolerance bite": at paper sizes the absolute contract alone is nearly vacuous).
LSE gate: max-abs <= 2e-3 (fp32 accumulation of O(1) numbers).
"""
import math

import numpy as np
import pytest
import torch

from paper_2606_13872_b200 import inputs as sra_inputs
from tests.gpu_util import bits, boundary_rows, gather_rows, oracle_forward_rows, run_gpu_forward
from tests.util import assert_parity

pytestmark = pytest.mark.gpu

LSE_TOL = 2e-3


def _full_parity(name, use_cache=True, dist=None, with_ref_rows=True):
    w = sra_inputs.WORKLOADS[name]
    if dist:
        w = w.replace(dist=dist)
    t = sra_inputs.make_inputs(w)
    scale = 1.0 / math.sqrt(w.head_dim)
    out = run_gpu_forward(w, t, use_cache=use_cache, with_ref_rows=with_ref_rows)
    n = w.n_gen + (w.n_ref if with_ref_rows else 0)
    rows = np.arange(n, dtype=np.int32)
    o_ref, lse_ref = oracle_forward_rows(w, bits(t), rows, scale)
    o_gpu, lse_gpu = gather_rows(out, w, rows)
    m = assert_parity(o_gpu, o_ref, f"{name} O")
    assert np.abs(lse_gpu - lse_ref).max() <= LSE_TOL, f"{name} LSE max err {np.abs(lse_gpu - lse_ref).max():.3e}"
    return m


@pytest.mark.parametrize("dist", ["A", "B", "peaked"])
def test_tiny_full(dist):
    """BASELINE.json configs[0]: B1 H4 d64, 256 gen + 4x128 ref, all rows, all heads."""
    _full_parity("tiny", dist=dist)


@pytest.mark.parametrize("use_cache", [True, False])
def test_ragged_d128(use_cache):
    """Non-uniform blocks (1, 130, 257, 64, 200), n_gen = 333, B2 H3: ragged tails everywhere."""
    _full_parity("ragged", use_cache=use_cache)


def test_ragged_d64_peaked():
    _full_parity("ragged64")


def test_mini480_full():
    """Real 1560-token block structure, scaled down (H2, 2x1560 gen + 3x1560 ref), every row."""
    _full_parity("mini480")


def test_mini720_full():
    _full_parity("mini720")


@pytest.mark.parametrize("name", ["short_mini", "short_mini64"])
def test_key_split_schedule_full(name):
    """Short-query schedules (keys split across CTAs, fp32 partials, merge kernel): every row vs the oracle."""
    from paper_2606_13872_b200 import binding as B
    w = sra_inputs.WORKLOADS[name]
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    n_split, _ = B.sra_split_schedule_copy(ctx)
    B.sra_destroy(ctx)
    assert n_split > 1, "this workload is meant to exercise the key-split path"
    _full_parity(name)


def test_cached_step_skips_ref_rows():
    """q_ref == NULL (PAPER.md:223 cached denoising step): only G rows are produced, one launch."""
    w = sra_inputs.WORKLOADS["ragged"]
    t = sra_inputs.make_inputs(w)
    out = run_gpu_forward(w, t, use_cache=True, with_ref_rows=False)
    assert "o_ref" not in out
    rows = np.arange(w.n_gen, dtype=np.int32)
    o_ref, _ = oracle_forward_rows(w, bits(t), rows, 1.0 / math.sqrt(w.head_dim))
    assert_parity(out["o_gen"], o_ref, "cached-step O_g")
    assert out["launches"] == 2  # cache build + one forward kernel


def test_zero_ref_is_plain_self_attention():
    """n_ref == 0 => full self-attention over G (north_star invariant), vs torch SDPA fp64 on CPU."""
    w = sra_inputs.SRAWorkload("noref", 1, 2, 128, 300, (), "B", 3)
    t = sra_inputs.make_inputs(w, names=("q_gen", "k_gen", "v_gen"))
    out = run_gpu_forward(w, t)
    q, k, v = (t[n].double().permute(0, 2, 1, 3) for n in ("q_gen", "k_gen", "v_gen"))
    ref = torch.nn.functional.scaled_dot_product_attention(q, k, v).permute(0, 2, 1, 3).numpy()
    assert_parity(out["o_gen"], ref, "zero-ref O_g")


def test_mask_poison():
    """huge finite values in K/V rows an R query must not see leave O_r unchanged."""
    w = sra_inputs.WORKLOADS["ragged"]
    t = sra_inputs.make_inputs(w)
    base = run_gpu_forward(w, t, use_cache=False)
    off = w.ref_block_offsets
    j = 2  # poison everything except block j (and all generation K/V)
    tp = {k: v.clone() for k, v in t.items()}
    for name in ("k_gen", "v_gen"):
        tp[name].fill_(1e4)
    for name in ("k_ref", "v_ref"):
        tp[name][:, :off[j]] = -1e4
        tp[name][:, off[j + 1]:] = 1e4
    pois = run_gpu_forward(w, tp, use_cache=False)
    a = base["o_ref"][:, off[j]:off[j + 1]]
    b = pois["o_ref"][:, off[j]:off[j + 1]]
    assert np.array_equal(a, b), "R rows of block j changed when unseen keys/values were poisoned"
    assert np.array_equal(base["lse_ref"][:, :, off[j]:off[j + 1]], pois["lse_ref"][:, :, off[j]:off[j + 1]])


def test_group_indicator_mass():
    """V[j] = e_{group(j)}: O rows are probability mass per group; masked groups must be exactly 0."""
    w = sra_inputs.WORKLOADS["ragged"]
    t = sra_inputs.make_inputs(w)
    off = w.ref_block_offsets
    t["v_gen"].zero_()
    t["v_ref"].zero_()
    t["v_gen"][..., 0] = 1.0
    for j in range(len(off) - 1):
        t["v_ref"][:, off[j]:off[j + 1], :, 1 + j] = 1.0
    out = run_gpu_forward(w, t, use_cache=True)
    ng = len(off)  # groups: G + blocks
    og = out["o_gen"][..., :ng]
    assert np.abs(og.sum(-1) - 1.0).max() <= 1e-2
    for j in range(len(off) - 1):
        orf = out["o_ref"][:, off[j]:off[j + 1]]
        assert np.abs(orf[..., 1 + j] - 1.0).max() <= 8e-3  # bf16 output rounding of ~1
        others = np.delete(orf[..., :ng], 1 + j, axis=-1)
        assert np.all(others == 0.0), "probability mass leaked to a masked group"


def test_480p_sampled_rows():
    """BASELINE.json configs[1] at full size, launch configuration of bench.py; sampled rows vs oracle."""
    w = sra_inputs.WORKLOADS["480p"].replace(dist="B")
    t = sra_inputs.make_inputs(w)
    out = run_gpu_forward(w, t, use_cache=True)
    rows = boundary_rows(w, n_random=16)
    o_ref, lse_ref = oracle_forward_rows(w, bits(t), rows, 1.0 / math.sqrt(w.head_dim))
    o_gpu, lse_gpu = gather_rows(out, w, rows)
    assert_parity(o_gpu, o_ref, "480p sampled O")
    assert np.abs(lse_gpu - lse_ref).max() <= LSE_TOL
    # property at any size: every output finite
    assert np.isfinite(out["o_gen"]).all() and np.isfinite(out["o_ref"]).all()


@pytest.mark.parametrize("name", ["host_pipe", "ragged"])
def test_forward_host_matches_device_path(name):
    """sra_forward_host (HOST pointers; the e2e leg of bench.py).  The plain path (everything small) must return exactly
    the bytes sra_forward returns.  The pipelined path (batch 1, >= 16 query slabs) runs its first slabs "reference
    keys first" - two fp32 partials per row (reference segment, generation segment) merged afterwards - so those rows
    may differ from the single-pass result in the last bf16 bit: every element within one bf16 ulp of the row's scale,
    the single-pass slabs and the reference rows bit-identical, and the whole output within the contract tolerance of
    the fp64 oracle (max-abs <= 2e-2, mean-abs <= 2e-3, rel_l2 <= 1e-2, LSE <= 2e-3)."""
    from paper_2606_13872_b200 import binding as B
    from oracle import sra_oracle
    w = (sra_inputs.SRAWorkload("host_pipe", 1, 2, 128, 6000, (700, 300), "B", 0) if name == "host_pipe"
         else sra_inputs.WORKLOADS[name])
    pipelined = name == "host_pipe"
    t = sra_inputs.make_inputs(w)
    dev_out = run_gpu_forward(w, t, use_cache=True)
    dev = torch.device("cuda:0")
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)

    def check_gen(o, lse):
        o = o.float().numpy()
        if not pipelined:
            assert np.array_equal(o, dev_out["o_gen"])
            assert lse is None or np.array_equal(lse.numpy(), dev_out["lse_gen"])
            return
        ulp = 2.0 ** -7 * np.abs(dev_out["o_gen"]).max(axis=-1, keepdims=True)   # one bf16 ulp at the row's largest element
        assert np.all(np.abs(o - dev_out["o_gen"]) <= ulp)
        differs = np.flatnonzero((o != dev_out["o_gen"]).any(axis=(0, 2, 3)))
        n_items = -(-w.n_gen // 256)                                               # 256-row query slabs (kQRowsPerCta)
        tail = 6 * (-(-n_items // 8)) * 256                                        # the last two of 8 slab groups are never split
        assert tail < w.n_gen
        assert differs.size == 0 or differs.max() < tail, "single-pass slabs must be bit-identical to sra_forward"
        if lse is not None:
            assert np.abs(lse.numpy() - dev_out["lse_gen"]).max() <= 1e-5

    try:
        B.sra_cache_reference_kv(ctx, t["k_ref"].to(dev), t["v_ref"].to(dev))
        h = {k: t[k].pin_memory() for k in ("q_gen", "k_gen", "v_gen", "q_ref")}
        o_gen = torch.full(t["q_gen"].shape, float("nan"), dtype=torch.bfloat16).pin_memory()
        o_ref = torch.full(t["q_ref"].shape, float("nan"), dtype=torch.bfloat16).pin_memory()
        lse_gen = torch.full((w.batch, w.heads, w.n_gen), float("nan")).pin_memory()
        lse_ref = torch.full((w.batch, w.heads, w.n_ref), float("nan")).pin_memory()
        for _ in range(2):  # twice: the second call reuses the staging buffers, streams and events
            B.sra_forward_host(ctx, h["q_gen"], h["k_gen"], h["v_gen"], o_gen, q_ref=h["q_ref"], o_ref=o_ref,
                               lse_gen=lse_gen, lse_ref=lse_ref)
            torch.cuda.synchronize()
            check_gen(o_gen, lse_gen)
            assert np.array_equal(o_ref.float().numpy(), dev_out["o_ref"])
            assert np.array_equal(lse_ref.numpy(), dev_out["lse_ref"])
            if pipelined:  # the host path on its own against the oracle, every row
                tb = bits(t)
                ref = sra_oracle.sra_forward(tb["q_gen"], tb["k_gen"], tb["v_gen"], tb["q_ref"], tb["k_ref"], tb["v_ref"],
                                             w.ref_block_offsets, 1.0 / math.sqrt(w.head_dim))
                assert_parity(o_gen.float().numpy(), ref["o_gen"], "host_pipe O_g through sra_forward_host")
                assert np.abs(lse_gen.numpy() - ref["lse_gen"]).max() <= LSE_TOL
            o_gen.fill_(float("nan")); o_ref.fill_(float("nan"))
        # cached denoising step through the host entry point (no reference rows)
        B.sra_forward_host(ctx, h["q_gen"], h["k_gen"], h["v_gen"], o_gen, lse_gen=lse_gen)
        torch.cuda.synchronize()
        check_gen(o_gen, lse_gen)
    finally:
        B.sra_destroy(ctx)


@pytest.mark.parametrize("mask", ["none", "shared", "per_sample"])
def test_forward_host_pipelined_batch2_and_validity(mask):
    """The pipelined host path beyond its first case (batch 1, no mask): batch 2 (a slab = the same rows of both items,
    strided copies), a validity mask shared by the batch (reference rows gathered from / scattered into the staged
    tensors; reference-first still on) and per-sample masks (reference-first off).  Against sra_forward on the same
    inputs (generation rows within one bf16 ulp of the row scale - the two-partial merge; reference rows bit-identical)
    and against the fp64 oracle under the same flags, every row."""
    from paper_2606_13872_b200 import binding as B
    from oracle import sra_oracle
    w = sra_inputs.SRAWorkload("host_pipe2", 2, 2, 128, 4200, (700, 300), "B", 0)
    t = sra_inputs.make_inputs(w)
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(11)
    valid = {"none": None, "shared": rng.random(w.n_ref) < 0.7,
             "per_sample": np.stack([rng.random(w.n_ref) < 0.8, rng.random(w.n_ref) < 0.4])}[mask]
    g = {k: v.to(dev) for k, v in t.items()}
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        if valid is not None:
            B.sra_set_reference_validity(ctx, valid)
        B.sra_cache_reference_kv(ctx, g["k_ref"], g["v_ref"])
        d_o_gen, d_o_ref = torch.empty_like(g["q_gen"]), torch.empty_like(g["q_ref"])
        d_lse_gen = torch.empty((w.batch, w.heads, w.n_gen), device=dev)
        B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], d_o_gen, q_ref=g["q_ref"], o_ref=d_o_ref, lse_gen=d_lse_gen)
        h = {k: t[k].pin_memory() for k in ("q_gen", "k_gen", "v_gen", "q_ref")}
        o_gen = torch.full(t["q_gen"].shape, float("nan"), dtype=torch.bfloat16).pin_memory()
        o_ref = torch.full(t["q_ref"].shape, float("nan"), dtype=torch.bfloat16).pin_memory()
        lse_gen = torch.full((w.batch, w.heads, w.n_gen), float("nan")).pin_memory()
        lse_ref = torch.full((w.batch, w.heads, w.n_ref), float("nan")).pin_memory()
        tb = bits(t)
        ref = sra_oracle.sra_forward(tb["q_gen"], tb["k_gen"], tb["v_gen"], tb["q_ref"], tb["k_ref"], tb["v_ref"],
                                     w.ref_block_offsets, 1.0 / math.sqrt(w.head_dim), valid=valid)
        for _ in range(2):  # the second call sizes its reference-first phase from the first call's measured rate
            B.sra_forward_host(ctx, h["q_gen"], h["k_gen"], h["v_gen"], o_gen, q_ref=h["q_ref"], o_ref=o_ref,
                               lse_gen=lse_gen, lse_ref=lse_ref)
            torch.cuda.synchronize()
            og, dg = o_gen.float().numpy(), d_o_gen.float().cpu().numpy()
            assert np.all(np.abs(og - dg) <= 2.0 ** -7 * np.abs(dg).max(axis=-1, keepdims=True))
            assert np.array_equal(o_ref.float().numpy(), d_o_ref.float().cpu().numpy())
            assert_parity(og, ref["o_gen"], f"host_pipe2[{mask}] O_g through sra_forward_host")
            assert np.abs(lse_gen.numpy() - ref["lse_gen"]).max() <= LSE_TOL
            v2 = np.ones((w.batch, w.n_ref), dtype=bool) if valid is None else np.broadcast_to(valid, (w.batch, w.n_ref))
            for b in range(w.batch):
                keep, inv = np.flatnonzero(v2[b]), np.flatnonzero(~v2[b])
                assert_parity(o_ref[b, keep].float().numpy(), ref["o_ref"][b, keep], f"host_pipe2[{mask}] O_r item {b}")
                assert np.all(o_ref[b, inv].float().numpy() == 0.0) and np.all(np.isneginf(lse_ref[b][:, inv].numpy()))
                assert np.abs(lse_ref[b][:, keep].numpy() - ref["lse_ref"][b][:, keep]).max() <= LSE_TOL
            o_gen.fill_(float("nan")); o_ref.fill_(float("nan"))
    finally:
        B.sra_destroy(ctx)


@pytest.mark.parametrize("name", ["short_mini", "ragged"])
def test_optional_lse_outputs_do_not_change_o(name):
    """lse_gen / lse_ref are nullable (include/sra.h): leaving them out must not change a byte of O, on the single-pass
    schedule and on the key-split schedule (whose merge kernel also writes the LSE)."""
    w = sra_inputs.WORKLOADS[name]
    t = sra_inputs.make_inputs(w)
    a = run_gpu_forward(w, t, use_cache=True, want_lse=True)
    b = run_gpu_forward(w, t, use_cache=True, want_lse=False)
    assert np.array_equal(a["o_gen"], b["o_gen"]) and np.array_equal(a["o_ref"], b["o_ref"])
    assert "lse_gen" not in b

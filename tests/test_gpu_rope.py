"""-m gpu parity of the RoPE producer side of the reference-KV cache ("eliminating redundant linear
projections and RoPE computations across all steps", reading A18 of DESIGN.md): the CUDA path
through the C ABI (sra_cache_reference_kv_rope, sra_apply_rope) against oracle.rope (fp64 complex multiplication).

Tolerances.  The rotation itself: the kernel computes a*c - b*s in fp32 (one FMA + one product) and rounds to bf16; the
oracle computes it in fp64 and rounds to bf16 (both sides take the bf16 decision, each in its own arithmetic).  fp32
error <= 2^-23 (|a c| + |b s|), so the two roundings differ only when the exact value lies within that distance of a
bf16 tie: at most 1 bf16 ulp apart, on a tiny fraction of the elements.  The test states exactly that:
|gpu - fp64| <= 2^-8 |fp64| + 2^-22 (|a| + |b|) for EVERY element, and >= 99.9 % bit-identical.
Attention on rotated tensors: the contract tolerance (BASELINE.json north_star: max-abs <= 2e-2, mean-abs <= 2e-3,
plus rel_l2 <= 1e-2, LSE <= 2e-3).
"""
import math

import numpy as np
import pytest
import torch

from oracle import c_oracle, sra_oracle
from paper_2606_13872_b200 import inputs as sra_inputs
from tests.gpu_util import bits, boundary_rows
from tests.util import assert_parity

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _tables(w, which):
    c, s = sra_inputs.rope_tables(w, which)
    return c, s, c.to(DEV), s.to(DEV)


def _check_rotation(got_bf16, x_bits, cos, sin, what):
    """Element-wise bound stated in the module docstring; returns the oracle's bf16 bit patterns."""
    y = sra_oracle.rope(x_bits, cos.numpy(), sin.numpy())
    x = sra_oracle.bf16_bits_to_f64(x_bits)
    mag = np.abs(x[..., 0::2]) + np.abs(x[..., 1::2])
    slack = np.repeat(mag, 2, axis=-1) * 2.0 ** -22
    got = got_bf16.float().cpu().numpy().astype(np.float64)
    assert np.all(np.abs(got - y) <= 2.0 ** -8 * np.abs(y) + slack + 1e-38), f"{what}: rotation outside the bf16 rounding bound"
    want_bits = sra_oracle.f64_to_bf16_bits(y)
    got_bits = sra_inputs.bf16_bits(got_bf16.cpu())
    same = np.mean(got_bits == want_bits)
    assert same >= 0.999, f"{what}: only {same:.5f} of the elements bit-identical to the rounded oracle"
    return want_bits


@pytest.mark.parametrize("name", ["ragged", "ragged64", "mini720"])
def test_apply_rope_matches_oracle(name):
    from paper_2606_13872_b200 import binding as B
    w = sra_inputs.WORKLOADS[name]
    t = sra_inputs.make_inputs(w)
    tb = bits(t)
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        c, s, cd, sd = _tables(w, "gen")
        q, k = t["q_gen"].to(DEV), t["k_gen"].to(DEV)
        n0 = B.sra_launch_count(ctx)
        B.sra_apply_rope(ctx, q, k, cd, sd, w.n_gen)
        assert B.sra_launch_count(ctx) - n0 == 1, "Q and K are rotated by one launch"
        torch.cuda.synchronize()
        _check_rotation(q, tb["q_gen"], c, s, f"{name} q_gen")
        _check_rotation(k, tb["k_gen"], c, s, f"{name} k_gen")
        # single-tensor form on the reference rows (their own table), x1 = NULL
        c, s, cd, sd = _tables(w, "ref")
        qr = t["q_ref"].to(DEV)
        B.sra_apply_rope(ctx, qr, None, cd, sd, w.n_ref)
        torch.cuda.synchronize()
        _check_rotation(qr, tb["q_ref"], c, s, f"{name} q_ref")
        # n_tokens = 0 is a no-op
        B.sra_apply_rope(ctx, qr, None, cd, sd, 0)
    finally:
        B.sra_destroy(ctx)


def _rotated_problem(w, t, valid=None):
    """GPU: per-step rotation of Q_g, K_g, Q_r + fused rotating cache producer + one forward from the cache.
    Returns the GPU outputs and the oracle's rotated (bf16-rounded) input bit patterns."""
    from paper_2606_13872_b200 import binding as B
    tb = bits(t)
    cg, sg, cgd, sgd = _tables(w, "gen")
    cr, sr, crd, srd = _tables(w, "ref")
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        if valid is not None:
            B.sra_set_reference_validity(ctx, valid)
        g = {k: v.to(DEV) for k, v in t.items()}
        B.sra_apply_rope(ctx, g["q_gen"], g["k_gen"], cgd, sgd, w.n_gen)
        B.sra_apply_rope(ctx, g["q_ref"], None, crd, srd, w.n_ref)
        n0 = B.sra_launch_count(ctx)
        B.sra_cache_reference_kv_rope(ctx, g["k_ref"], g["v_ref"], crd, srd)   # k_ref is PRE-RoPE here
        assert B.sra_launch_count(ctx) - n0 == 1, "rotation + head-major relayout of K_r, V_r = one launch"
        nan = float("nan")
        o_gen, o_ref = torch.full_like(g["q_gen"], nan), torch.full_like(g["q_ref"], nan)
        lse_gen = torch.full((w.batch, w.heads, w.n_gen), nan, device=DEV)
        lse_ref = torch.full((w.batch, w.heads, w.n_ref), nan, device=DEV)
        B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, q_ref=g["q_ref"], o_ref=o_ref, lse_gen=lse_gen,
                      lse_ref=lse_ref)
        torch.cuda.synchronize()
        got = {"o_gen": o_gen, "o_ref": o_ref, "lse_gen": lse_gen, "lse_ref": lse_ref}

        # the unfused route (rotate a copy of K_r in place, then the plain cache call) must give the same bits:
        # both kernels share the arithmetic, only the HBM round trip differs
        k2 = t["k_ref"].to(DEV)
        B.sra_apply_rope(ctx, k2, None, crd, srd, w.n_ref)
        B.sra_cache_reference_kv(ctx, k2, g["v_ref"])
        o2, o2r = torch.full_like(o_gen, nan), torch.full_like(o_ref, nan)
        B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o2, q_ref=g["q_ref"], o_ref=o2r)
        torch.cuda.synchronize()
        assert torch.equal(o2.view(torch.int16), o_gen.view(torch.int16)), "fused and unfused cache producers differ"
        keep = slice(None) if valid is None else torch.as_tensor(np.flatnonzero(valid), device=DEV)
        assert torch.equal(o2r[:, keep].view(torch.int16), o_ref[:, keep].view(torch.int16))
        got = {k: v.float().cpu().numpy() for k, v in got.items()}
    finally:
        B.sra_destroy(ctx)
    rb = dict(tb)
    f = sra_oracle.f64_to_bf16_bits
    rb["q_gen"] = f(sra_oracle.rope(tb["q_gen"], cg.numpy(), sg.numpy()))
    rb["k_gen"] = f(sra_oracle.rope(tb["k_gen"], cg.numpy(), sg.numpy()))
    rb["q_ref"] = f(sra_oracle.rope(tb["q_ref"], cr.numpy(), sr.numpy()))
    rb["k_ref"] = f(sra_oracle.rope(tb["k_ref"], cr.numpy(), sr.numpy()))
    return got, rb


@pytest.mark.parametrize("name", ["ragged", "ragged64"])
def test_rope_cache_forward_matches_oracle(name):
    """Every row and column: rotated Q/K through the CUDA path vs oracle.rope -> bf16 -> oracle.sra_forward."""
    w = sra_inputs.WORKLOADS[name]
    t = sra_inputs.make_inputs(w)
    got, rb = _rotated_problem(w, t)
    ref = sra_oracle.sra_forward(rb["q_gen"], rb["k_gen"], rb["v_gen"], rb["q_ref"], rb["k_ref"], rb["v_ref"],
                                 w.ref_block_offsets, 1.0 / math.sqrt(w.head_dim))
    for n in ("o_gen", "o_ref"):
        assert_parity(got[n], ref[n], f"{name} rope {n}")
    for n in ("lse_gen", "lse_ref"):
        assert np.abs(got[n] - ref[n]).max() <= 2e-3
    # the rotation matters: the un-rotated problem is a different one (guards a silently skipped rotation)
    tb = bits(t)
    plain = sra_oracle.sra_forward(tb["q_gen"], tb["k_gen"], tb["v_gen"], tb["q_ref"], tb["k_ref"], tb["v_ref"],
                                   w.ref_block_offsets, 1.0 / math.sqrt(w.head_dim))
    assert np.abs(plain["o_gen"] - ref["o_gen"]).max() > 5e-2


def test_rope_cache_with_validity_mask():
    """Validity compaction + fused rotation: row n of the compacted cache is rotated by the table row of
    its ORIGINAL token."""
    w = sra_inputs.WORKLOADS["ragged"]
    rng = np.random.default_rng(11)
    valid = rng.random(w.n_ref) < 0.6
    t = sra_inputs.make_inputs(w)
    got, rb = _rotated_problem(w, t, valid=valid)
    ref = sra_oracle.sra_forward(rb["q_gen"], rb["k_gen"], rb["v_gen"], rb["q_ref"], rb["k_ref"], rb["v_ref"],
                                 w.ref_block_offsets, 1.0 / math.sqrt(w.head_dim), valid=valid)
    keep, inv = np.flatnonzero(valid), np.flatnonzero(~valid)
    assert_parity(got["o_gen"], ref["o_gen"], "rope + validity O_g")
    assert_parity(got["o_ref"][:, keep], ref["o_ref"][:, keep], "rope + validity O_r")
    assert np.all(got["o_ref"][:, inv] == 0.0)
    assert np.abs(got["lse_gen"] - ref["lse_gen"]).max() <= 2e-3


def test_rope_720p_full_size_sampled():
    """BASELINE.json configs[2] shape: rotate Q_g, K_g (75,600 tokens) and build the rotated cache (50,400 tokens) at
    full size; the rotation is checked on sampled tokens of every tensor, the attention on sampled rows (row sampling
    is exact, tests/test_gpu_fullsize.py)."""
    from paper_2606_13872_b200 import binding as B
    w = sra_inputs.WORKLOADS["720p"]
    heads = [0, 39]
    scale = 1.0 / math.sqrt(w.head_dim)
    dev = torch.device(DEV)
    raw = {n: sra_inputs.make_tensor_device(w, n, dev) for n in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")}
    raw_bits = {n: sra_inputs.bf16_bits(x[:, :, heads].contiguous().cpu()) for n, x in raw.items()}
    cg, sg, cgd, sgd = _tables(w, "gen")
    cr, sr, crd, srd = _tables(w, "ref")
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        B.sra_cache_reference_kv_rope(ctx, raw["k_ref"], raw["v_ref"], crd, srd)
        B.sra_apply_rope(ctx, raw["q_gen"], raw["k_gen"], cgd, sgd, w.n_gen)
        B.sra_apply_rope(ctx, raw["q_ref"], None, crd, srd, w.n_ref)
        o_gen = torch.full_like(raw["q_gen"], float("nan"))
        o_ref = torch.full_like(raw["q_ref"], float("nan"))
        lse_gen = torch.empty((w.batch, w.heads, w.n_gen), device=dev)
        lse_ref = torch.empty((w.batch, w.heads, w.n_ref), device=dev)
        B.sra_forward(ctx, raw["q_gen"], raw["k_gen"], raw["v_gen"], o_gen, q_ref=raw["q_ref"], o_ref=o_ref,
                      lse_gen=lse_gen, lse_ref=lse_ref)
        torch.cuda.synchronize()
        assert torch.isfinite(o_gen.float()).all() and torch.isfinite(o_ref.float()).all()
        # rotation on sampled tokens of the in-place tensors (all of the two sampled heads)
        rng = np.random.default_rng(3)
        for n, cc, ss, ntok in (("q_gen", cg, sg, w.n_gen), ("k_gen", cg, sg, w.n_gen), ("q_ref", cr, sr, w.n_ref)):
            idx = np.unique(np.concatenate([[0, ntok - 1], rng.integers(0, ntok, 500)]))
            got = raw[n][:, torch.as_tensor(idx, device=dev)][:, :, heads]
            _check_rotation(got, raw_bits[n][:, idx], cc[idx], ss[idx], f"720p {n}")
        # attention on sampled rows against the oracle's own rotated, bf16-rounded inputs
        f = sra_oracle.f64_to_bf16_bits
        rb = {"v_gen": raw_bits["v_gen"], "v_ref": raw_bits["v_ref"],
              "q_gen": f(sra_oracle.rope(raw_bits["q_gen"], cg.numpy(), sg.numpy())),
              "k_gen": f(sra_oracle.rope(raw_bits["k_gen"], cg.numpy(), sg.numpy())),
              "q_ref": f(sra_oracle.rope(raw_bits["q_ref"], cr.numpy(), sr.numpy())),
              "k_ref": f(sra_oracle.rope(raw_bits["k_ref"], cr.numpy(), sr.numpy()))}
        rows = boundary_rows(w, n_random=6)
        o_or, lse_or = c_oracle.forward_rows(rb["q_gen"], rb["k_gen"], rb["v_gen"], rb["q_ref"], rb["k_ref"], rb["v_ref"],
                                             w.ref_block_offsets, scale, rows)
        g = rows[rows < w.n_gen]
        r = rows[rows >= w.n_gen] - w.n_gen
        gi, ri = torch.as_tensor(g, device=dev).long(), torch.as_tensor(r, device=dev).long()
        o_gpu = np.concatenate([o_gen[:, gi][:, :, heads].float().cpu().numpy(),
                                o_ref[:, ri][:, :, heads].float().cpu().numpy()], axis=1)
        l_gpu = np.concatenate([lse_gen[:, heads][:, :, gi].cpu().numpy(), lse_ref[:, heads][:, :, ri].cpu().numpy()], axis=2)
        assert_parity(o_gpu, o_or, "720p rope sampled O")
        assert np.abs(l_gpu - lse_or).max() <= 2e-3
    finally:
        B.sra_destroy(ctx)

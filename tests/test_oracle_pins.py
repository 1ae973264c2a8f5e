"""Pins for the CPU fp64 oracle (oracle/sra_oracle.py and oracle/sra_oracle.c).

The paper prints NO worked numeric example of Sparse Reference Attention,
no equation and no mask figure, so the oracle is pinned to what the
mathematics fixes instead: closed forms, invariants named by BASELINE.json north_star,
special cases that reduce to a library routine (torch CPU fp64 SDPA / autograd), a
pure-Python brute force on tiny inputs and central finite differences for the backward.
Each check is chosen so that a plausible mistake (dropped term, wrong sign/index,
transposed operand, wrong block lookup) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest
import torch

from oracle import c_oracle, sra_oracle
from tests.util import bits_to_f64, rand_bits, to_bf16_bits

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _problem(rng, B=1, H=2, d=8, Ng=5, blocks=(3, 1, 4), scale_q=1.0):
    Nr = sum(blocks)
    off = np.concatenate([[0], np.cumsum(blocks)]).astype(np.int32)
    t = {}
    for name, n in (("q_gen", Ng), ("k_gen", Ng), ("v_gen", Ng), ("q_ref", Nr), ("k_ref", Nr), ("v_ref", Nr),
                    ("do_gen", Ng), ("do_ref", Nr)):
        s = scale_q if name[0] in "qk" else 1.0
        t[name] = rand_bits(rng, (B, n, H, d), s)
    return t, off, 1.0 / math.sqrt(d)


def _fwd(t, off, s, with_qref=True):
    return sra_oracle.sra_forward(t["q_gen"], t["k_gen"], t["v_gen"], t["q_ref"] if with_qref else None,
                                  t["k_ref"], t["v_ref"], off, s)


# ----------------------------------------------------------------------------- upcast
def test_bf16_upcast_exact():
    bits = np.arange(0, 65536, dtype=np.uint32).astype(np.uint16)
    finite = np.isfinite(bits_to_f64(bits))
    a = sra_oracle.bf16_bits_to_f64(bits)[finite]
    b = bits_to_f64(bits)[finite]
    assert np.array_equal(a, b)


# ----------------------------------------------------------------------------- mask
def _closed_form_pairs(Ng, blocks):
    return Ng * (Ng + sum(blocks)) + sum(b * b for b in blocks)


def test_mask_density_golden():
    """pairs = N_g (N_g + N_r) + sum_j b_j^2 ; values in tests/golden/pairs.txt."""
    rows = [l.split() for l in open(os.path.join(GOLDEN, "pairs.txt")) if l.strip() and not l.startswith("#")]
    for name, Ng, nblk, bsz, pairs, total in rows:
        Ng, nblk, bsz, total = int(Ng), int(nblk), int(bsz), int(total)
        got = _closed_form_pairs(Ng, [bsz] * nblk)
        if pairs.startswith("~"):
            assert abs(got - float(pairs[1:])) <= 5e-4 * float(pairs[1:]), name
        else:
            assert got == int(pairs), name
        assert (Ng + nblk * bsz) ** 2 == total, name
    # the explicit mask (python and C) on the Tiny config: 262,144 of 589,824
    off = [0, 128, 256, 384, 512]
    assert sra_oracle.count_pairs(256, off) == 262144
    assert c_oracle.count_pairs(256, off) == 262144
    M = sra_oracle.sra_mask(256, off)
    assert M.shape == (768, 768) and M.size == 589824


@pytest.mark.parametrize("Ng,blocks", [(5, (3, 1, 4)), (1, (2,)), (7, ()), (3, (1, 1, 1)), (4, (5, 2))])
def test_mask_structure(Ng, blocks):
    off = np.concatenate([[0], np.cumsum(blocks)]).astype(int) if blocks else np.array([0])
    M = sra_oracle.sra_mask(Ng, off)
    n = Ng + sum(blocks)
    assert M.shape == (n, n)
    assert int(M.sum()) == _closed_form_pairs(Ng, blocks) == c_oracle.count_pairs(Ng, off)
    assert M[:Ng].all()  # G rows see everything
    assert not M[Ng:, :Ng].any()  # R -> G always masked
    R = M[Ng:, Ng:]
    assert np.array_equal(R, R.T)  # block-diagonal is symmetric
    # independent construction: block id per token, equality matrix
    bid = np.repeat(np.arange(len(blocks)), blocks)
    assert np.array_equal(R.astype(bool), bid[:, None] == bid[None, :])


def test_group_indicator_mass():
    """V[j] = e_{g(j)} (g=0 for G, 1+block for R) => O[i][g] = probability mass on group g."""
    rng = np.random.default_rng(1)
    blocks = (3, 2, 4)
    t, off, s = _problem(rng, H=1, d=8, Ng=6, blocks=blocks)
    n_groups = 1 + len(blocks)
    assert n_groups <= 8
    vg = np.zeros((1, 6, 1, 8)); vg[..., 0] = 1.0
    vr = np.zeros((1, 9, 1, 8))
    bid = np.repeat(np.arange(len(blocks)), blocks)
    for j, g in enumerate(bid):
        vr[0, j, 0, 1 + g] = 1.0
    t["v_gen"], t["v_ref"] = to_bf16_bits(vg), to_bf16_bits(vr)
    out = _fwd(t, off, s)
    og, orf = out["o_gen"][0, :, 0], out["o_ref"][0, :, 0]
    assert np.allclose(og[:, :n_groups].sum(axis=1), 1.0, atol=1e-14)
    assert (og[:, :n_groups] > 0).all()  # G rows put mass on every group
    for i, g in enumerate(bid):  # R rows: exactly 1 on own group, exactly 0 elsewhere
        expect = np.zeros(8); expect[1 + g] = 1.0
        assert np.allclose(orf[i], expect, atol=1e-15), (i, orf[i])
        assert orf[i][0] == 0.0 and all(orf[i][1 + k] == 0.0 for k in range(len(blocks)) if k != g)
    # same through the C oracle
    rows = np.arange(15, dtype=np.int32)
    oc, _ = c_oracle.forward_rows(t["q_gen"], t["k_gen"], t["v_gen"], t["q_ref"], t["k_ref"], t["v_ref"], off, s, rows)
    assert np.allclose(oc[0, :6, 0], og, atol=1e-14) and np.allclose(oc[0, 6:, 0], orf, atol=1e-14)


# ----------------------------------------------------------------------------- softmax closed forms
def test_constant_v_and_row_sums():
    rng = np.random.default_rng(2)
    t, off, s = _problem(rng, B=2, H=2, d=8, Ng=5, blocks=(3, 1, 4), scale_q=3.0)
    for const in (1.0, -2.5):
        t["v_gen"] = to_bf16_bits(np.full((2, 5, 2, 8), const))
        t["v_ref"] = to_bf16_bits(np.full((2, 8, 2, 8), const))
        out = _fwd(t, off, s)
        assert np.allclose(out["o_gen"], const, atol=1e-14) and np.allclose(out["o_ref"], const, atol=1e-14)


def test_zero_q_gives_means():
    """Q = 0 => uniform softmax: O_g = mean of all V rows; O_r[block j] = mean of block j's V rows;
    LSE = log(number of visible keys)."""
    rng = np.random.default_rng(3)
    blocks = (3, 1, 4)
    t, off, s = _problem(rng, B=1, H=2, d=8, Ng=5, blocks=blocks)
    t["q_gen"] = np.zeros_like(t["q_gen"]); t["q_ref"] = np.zeros_like(t["q_ref"])
    out = _fwd(t, off, s)
    vg, vr = bits_to_f64(t["v_gen"]), bits_to_f64(t["v_ref"])
    mean_all = np.concatenate([vg, vr], axis=1).mean(axis=1)  # [B,H,d]
    assert np.allclose(out["o_gen"], mean_all[:, None], atol=1e-15)
    assert np.allclose(out["lse_gen"], math.log(5 + 8), atol=1e-15)
    for j, b in enumerate(blocks):
        lo, hi = off[j], off[j + 1]
        assert np.allclose(out["o_ref"][:, lo:hi], vr[:, lo:hi].mean(axis=1)[:, None], atol=1e-15)
        assert np.allclose(out["lse_ref"][:, :, lo:hi], math.log(b), atol=1e-15)
    rows = np.arange(13, dtype=np.int32)
    oc, lc = c_oracle.forward_rows(t["q_gen"], t["k_gen"], t["v_gen"], t["q_ref"], t["k_ref"], t["v_ref"], off, s, rows)
    assert np.allclose(oc[:, :5], out["o_gen"], atol=1e-15) and np.allclose(oc[:, 5:], out["o_ref"], atol=1e-15)
    assert np.allclose(lc[:, :, :5], out["lse_gen"], atol=1e-15)


# ----------------------------------------------------------------------------- library cross-checks
def _sdpa(Q, K, V, s):
    """torch CPU fp64 SDPA (library routine) for one head: Q [n,d], K/V [m,d]."""
    q, k, v = (torch.as_tensor(x)[None, None] for x in (Q, K, V))
    return torch.nn.functional.scaled_dot_product_attention(q, k, v, scale=s)[0, 0].numpy()


def test_g_rows_equal_dense_attention_and_lse_merge():
    rng = np.random.default_rng(4)
    t, off, s = _problem(rng, B=2, H=2, d=16, Ng=7, blocks=(3, 5, 2), scale_q=2.0)
    out = _fwd(t, off, s)
    f = bits_to_f64
    for b in range(2):
        for h in range(2):
            Q = f(t["q_gen"])[b, :, h]
            Kg, Vg, Kr, Vr = (f(t[k])[b, :, h] for k in ("k_gen", "v_gen", "k_ref", "v_ref"))
            ref = _sdpa(Q, np.concatenate([Kg, Kr]), np.concatenate([Vg, Vr]), s)
            assert np.allclose(out["o_gen"][b, :, h], ref, atol=1e-13)
            # LSE-merge identity: Attn(Q,[Kg;Kr]) = merge of Attn(Q,Kg,Vg) and Attn(Q,Kr,Vr) by LSE weights
            Sg, Sr = s * Q @ Kg.T, s * Q @ Kr.T
            lg = np.log(np.exp(Sg).sum(1)); lr = np.log(np.exp(Sr).sum(1))
            og, orr = _sdpa(Q, Kg, Vg, s), _sdpa(Q, Kr, Vr, s)
            lse = np.logaddexp(lg, lr)
            merged = np.exp(lg - lse)[:, None] * og + np.exp(lr - lse)[:, None] * orr
            assert np.allclose(out["o_gen"][b, :, h], merged, atol=1e-13)
            assert np.allclose(out["lse_gen"][b, h], lse, atol=1e-13)


def test_r_rows_equal_blockwise_dense_attention():
    rng = np.random.default_rng(5)
    blocks = (3, 5, 1, 2)
    t, off, s = _problem(rng, B=1, H=2, d=16, Ng=4, blocks=blocks, scale_q=2.0)
    out = _fwd(t, off, s)
    f = bits_to_f64
    for h in range(2):
        for j in range(len(blocks)):
            lo, hi = off[j], off[j + 1]
            ref = _sdpa(f(t["q_ref"])[0, lo:hi, h], f(t["k_ref"])[0, lo:hi, h], f(t["v_ref"])[0, lo:hi, h], s)
            assert np.allclose(out["o_ref"][0, lo:hi, h], ref, atol=1e-13)
    # n_ref_blocks = 1 => plain self-attention over R
    out1 = _fwd(t, np.array([0, sum(blocks)]), s)
    for h in range(2):
        ref = _sdpa(f(t["q_ref"])[0, :, h], f(t["k_ref"])[0, :, h], f(t["v_ref"])[0, :, h], s)
        assert np.allclose(out1["o_ref"][0, :, h], ref, atol=1e-13)


def test_zero_ref_is_plain_self_attention_and_single_gen_token():
    rng = np.random.default_rng(6)
    t, off, s = _problem(rng, B=1, H=2, d=16, Ng=9, blocks=())
    out = _fwd(t, off, s)
    f = bits_to_f64
    for h in range(2):
        ref = _sdpa(f(t["q_gen"])[0, :, h], f(t["k_gen"])[0, :, h], f(t["v_gen"])[0, :, h], s)
        assert np.allclose(out["o_gen"][0, :, h], ref, atol=1e-13)
    assert out["o_ref"].shape[1] == 0
    t, off, s = _problem(rng, B=1, H=1, d=8, Ng=1, blocks=(2, 3))
    out = _fwd(t, off, s)
    K = np.concatenate([f(t["k_gen"])[0, :, 0], f(t["k_ref"])[0, :, 0]])
    V = np.concatenate([f(t["v_gen"])[0, :, 0], f(t["v_ref"])[0, :, 0]])
    assert np.allclose(out["o_gen"][0, :, 0], _sdpa(f(t["q_gen"])[0, :, 0], K, V, s), atol=1e-13)


def test_cached_step_skips_ref_rows():
    rng = np.random.default_rng(7)
    t, off, s = _problem(rng)
    a, b = _fwd(t, off, s, True), _fwd(t, off, s, False)
    assert "o_ref" not in b and np.array_equal(a["o_gen"], b["o_gen"])


# ----------------------------------------------------------------------------- symmetries
def test_permutation_symmetries():
    rng = np.random.default_rng(8)
    blocks = (3, 4, 2)
    t, off, s = _problem(rng, B=1, H=2, d=8, Ng=5, blocks=blocks, scale_q=2.0)
    base = _fwd(t, off, s)
    # (a) O_g invariant under ANY joint permutation of (K_r, V_r) rows, even across blocks
    perm = rng.permutation(9)
    t2 = dict(t); t2["k_ref"] = t["k_ref"][:, perm]; t2["v_ref"] = t["v_ref"][:, perm]
    assert np.allclose(_fwd(t2, off, s)["o_gen"], base["o_gen"], atol=1e-14)
    # (b) O_r equivariant under within-block permutations
    perm = np.concatenate([off[j] + rng.permutation(b) for j, b in enumerate(blocks)])
    t3 = dict(t)
    for k in ("q_ref", "k_ref", "v_ref"):
        t3[k] = t[k][:, perm]
    o3 = _fwd(t3, off, s)
    assert np.allclose(o3["o_ref"], base["o_ref"][:, perm], atol=1e-14)
    assert np.allclose(o3["o_gen"], base["o_gen"], atol=1e-14)
    # (c) reordering whole blocks: blocks (0,1,2) -> (2,0,1)
    order = [2, 0, 1]
    idx = np.concatenate([np.arange(off[j], off[j + 1]) for j in order])
    off4 = np.concatenate([[0], np.cumsum([blocks[j] for j in order])])
    t4 = dict(t)
    for k in ("q_ref", "k_ref", "v_ref"):
        t4[k] = t[k][:, idx]
    o4 = _fwd(t4, off4, s)
    assert np.allclose(o4["o_ref"], base["o_ref"][:, idx], atol=1e-14)
    assert np.allclose(o4["o_gen"], base["o_gen"], atol=1e-14)


# ----------------------------------------------------------------------------- brute force
def _brute_force(t, off, s):
    """Pure-Python per-element brute force (independent of numpy matmul / the oracle's structure)."""
    f = bits_to_f64
    qg, kg, vg, qr, kr, vr = (f(t[k]) for k in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref"))
    B, Ng, H, d = qg.shape
    Nr = kr.shape[1]
    bid = [next(k for k in range(len(off) - 1) if off[k] <= j < off[k + 1]) for j in range(Nr)]
    O = np.zeros((B, Ng + Nr, H, d)); L = np.zeros((B, H, Ng + Nr))
    for b in range(B):
        for h in range(H):
            for i in range(Ng + Nr):
                q = qg[b, i, h] if i < Ng else qr[b, i - Ng, h]
                keys = []
                if i < Ng:
                    keys += [(kg[b, j, h], vg[b, j, h]) for j in range(Ng)]
                    keys += [(kr[b, j, h], vr[b, j, h]) for j in range(Nr)]
                else:
                    keys += [(kr[b, j, h], vr[b, j, h]) for j in range(Nr) if bid[j] == bid[i - Ng]]
                sc = [s * sum(float(q[c]) * float(k[c]) for c in range(d)) for k, _ in keys]
                mx = max(sc)
                w = [math.exp(x - mx) for x in sc]
                z = sum(w)
                for c in range(d):
                    O[b, i, h, c] = sum(wi * float(v[c]) for wi, (_, v) in zip(w, keys)) / z
                L[b, h, i] = mx + math.log(z)
    return O, L


@pytest.mark.parametrize("seed,Ng,blocks,d", [(10, 4, (3, 1, 2), 4), (11, 1, (1,), 3), (12, 6, (2, 5), 8), (13, 3, (), 4)])
def test_brute_force_tiny(seed, Ng, blocks, d):
    rng = np.random.default_rng(seed)
    t, off, s = _problem(rng, B=2, H=2, d=d, Ng=Ng, blocks=blocks, scale_q=2.0)
    O, L = _brute_force(t, off, s)
    out = _fwd(t, off, s)
    assert np.allclose(out["o_gen"], O[:, :Ng], atol=1e-13) and np.allclose(out["lse_gen"], L[:, :, :Ng], atol=1e-13)
    if blocks:
        assert np.allclose(out["o_ref"], O[:, Ng:], atol=1e-13) and np.allclose(out["lse_ref"], L[:, :, Ng:], atol=1e-13)
    n = Ng + sum(blocks)
    oc, lc = c_oracle.forward_rows(t["q_gen"], t["k_gen"], t["v_gen"], t["q_ref"], t["k_ref"], t["v_ref"], off, s,
                                   np.arange(n, dtype=np.int32))
    assert np.allclose(oc, O, atol=1e-13) and np.allclose(lc, L, atol=1e-13)


def test_numpy_vs_where_softmax_one_liner():
    """The 4-line numpy `where(M, S, -inf)` softmax of SURVEY.md section 8c on the Tiny shape (1 head)."""
    rng = np.random.default_rng(14)
    t, off, s = _problem(rng, B=1, H=1, d=64, Ng=256, blocks=(128,) * 4, scale_q=1.0)
    out = _fwd(t, off, s)
    f = bits_to_f64
    Q = np.concatenate([f(t["q_gen"])[0, :, 0], f(t["q_ref"])[0, :, 0]])
    K = np.concatenate([f(t["k_gen"])[0, :, 0], f(t["k_ref"])[0, :, 0]])
    V = np.concatenate([f(t["v_gen"])[0, :, 0], f(t["v_ref"])[0, :, 0]])
    bid = np.concatenate([np.full(256, -1), np.repeat(np.arange(4), 128)])
    M = (bid[:, None] == -1) | ((bid[:, None] == bid[None, :]) & (bid[None, :] >= 0))
    S = np.where(M, s * Q @ K.T, -np.inf)
    P = np.exp(S - S.max(1, keepdims=True)); P /= P.sum(1, keepdims=True)
    O = P @ V
    assert np.allclose(np.concatenate([out["o_gen"][0, :, 0], out["o_ref"][0, :, 0]]), O, atol=1e-13)
    # C oracle: sampled rows + one full head agree with the numpy oracle
    rows = np.array([0, 255, 256, 383, 384, 767], dtype=np.int32)
    oc, _ = c_oracle.forward_rows(t["q_gen"], t["k_gen"], t["v_gen"], t["q_ref"], t["k_ref"], t["v_ref"], off, s, rows)
    assert np.allclose(oc[0, :, 0], O[rows], atol=1e-13)
    oh, lh = c_oracle.forward_head(t["q_gen"], t["k_gen"], t["v_gen"], t["q_ref"], t["k_ref"], t["v_ref"], off, s, 0, 0)
    assert np.allclose(oh, O, atol=1e-13)
    assert np.allclose(lh, np.log(np.exp(S - S.max(1, keepdims=True)).sum(1)) + S.max(1), atol=1e-12)


# ----------------------------------------------------------------------------- backward
def _bwd(t, off, s):
    return sra_oracle.sra_backward(t["q_gen"], t["k_gen"], t["v_gen"], t["q_ref"], t["k_ref"], t["v_ref"],
                                   t["do_gen"], t["do_ref"], off, s)


def _loss(t, off, s):
    """Scalar loss sum(dO o O) of the fp64 forward, as a function of fp64 inputs given directly."""
    out = _fwd(t, off, s)
    f = bits_to_f64
    return float((f(t["do_gen"]) * out["o_gen"]).sum() + (f(t["do_ref"]) * out["o_ref"]).sum())


def test_backward_torch_autograd():
    """dQ/dK/dV equal torch fp64 autograd through an independently built masked attention."""
    rng = np.random.default_rng(20)
    blocks = (3, 1, 4)
    t, off, s = _problem(rng, B=2, H=2, d=8, Ng=5, blocks=blocks, scale_q=2.0)
    g = _bwd(t, off, s)
    f = lambda k: torch.tensor(bits_to_f64(t[k]), requires_grad=True)
    qg, kg, vg, qr, kr, vr = (f(k) for k in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref"))
    dog, dor = torch.tensor(bits_to_f64(t["do_gen"])), torch.tensor(bits_to_f64(t["do_ref"]))
    bid = torch.tensor(np.repeat(np.arange(len(blocks)), blocks))
    K = torch.cat([kg, kr], 1); V = torch.cat([vg, vr], 1)
    Sg = s * torch.einsum("bihc,bjhc->bhij", qg, K)
    Og = torch.einsum("bhij,bjhc->bihc", torch.softmax(Sg, -1), V)
    Sr = s * torch.einsum("bihc,bjhc->bhij", qr, kr)
    Sr = Sr.masked_fill(bid[:, None] != bid[None, :], float("-inf"))
    Or = torch.einsum("bhij,bjhc->bihc", torch.softmax(Sr, -1), vr)
    ((Og * dog).sum() + (Or * dor).sum()).backward()
    for name, leaf in (("dq_gen", qg), ("dk_gen", kg), ("dv_gen", vg), ("dq_ref", qr), ("dk_ref", kr), ("dv_ref", vr)):
        assert np.allclose(g[name], leaf.grad.numpy(), atol=1e-12), name
    # C oracle backward (all rows / cols of each head) against the same autograd result
    for b in range(2):
        for h in range(2):
            o, lse = c_oracle.forward_head(t["q_gen"], t["k_gen"], t["v_gen"], t["q_ref"], t["k_ref"], t["v_ref"], off, s, b, h)
            dq, dk, dv = c_oracle.backward_head(t["q_gen"], t["k_gen"], t["v_gen"], t["q_ref"], t["k_ref"], t["v_ref"],
                                                t["do_gen"], t["do_ref"], off, s, b, h, o, lse)
            assert np.allclose(dq[:5], qg.grad.numpy()[b, :, h], atol=1e-12)
            assert np.allclose(dq[5:], qr.grad.numpy()[b, :, h], atol=1e-12)
            assert np.allclose(dk[:5], kg.grad.numpy()[b, :, h], atol=1e-12)
            assert np.allclose(dk[5:], kr.grad.numpy()[b, :, h], atol=1e-12)
            assert np.allclose(dv[:5], vg.grad.numpy()[b, :, h], atol=1e-12)
            assert np.allclose(dv[5:], vr.grad.numpy()[b, :, h], atol=1e-12)
            # subset of rows / cols is exact
            rows = np.array([1, 6, 12], dtype=np.int32); cols = np.array([0, 5, 11], dtype=np.int32)
            dq2, dk2, dv2 = c_oracle.backward_head(t["q_gen"], t["k_gen"], t["v_gen"], t["q_ref"], t["k_ref"], t["v_ref"],
                                                   t["do_gen"], t["do_ref"], off, s, b, h, o, lse, rows, cols)
            assert np.array_equal(dq2, dq[rows]) and np.array_equal(dk2, dk[cols]) and np.array_equal(dv2, dv[cols])


def test_backward_finite_differences():
    """Central differences of the fp64 forward loss sum(dO o O) w.r.t. bf16-representable perturbations.

    Inputs are bf16 bit patterns, so the perturbation is applied on a private fp64 path:
    masked_attention() is called directly with fp64 operands (eps = 1e-6)."""
    rng = np.random.default_rng(21)
    blocks = (2, 3)
    Ng, Nr, d = 3, 5, 4
    t, off, s = _problem(rng, B=1, H=1, d=d, Ng=Ng, blocks=blocks, scale_q=1.5)
    g = _bwd(t, off, s)
    f = bits_to_f64
    Q = np.concatenate([f(t["q_gen"])[0, :, 0], f(t["q_ref"])[0, :, 0]])
    K = np.concatenate([f(t["k_gen"])[0, :, 0], f(t["k_ref"])[0, :, 0]])
    V = np.concatenate([f(t["v_gen"])[0, :, 0], f(t["v_ref"])[0, :, 0]])
    dO = np.concatenate([f(t["do_gen"])[0, :, 0], f(t["do_ref"])[0, :, 0]])
    M = sra_oracle.sra_mask(Ng, off)

    def loss(Q, K, V):
        O, _, _ = sra_oracle.masked_attention(Q, K, V, M, s)
        return float((dO * O).sum())

    eps = 1e-6
    for X, names in ((Q, ("dq_gen", "dq_ref")), (K, ("dk_gen", "dk_ref")), (V, ("dv_gen", "dv_ref"))):
        G = np.concatenate([g[names[0]][0, :, 0], g[names[1]][0, :, 0]])
        for i in range(Ng + Nr):
            for c in range(d):
                Xp, Xm = X.copy(), X.copy()
                Xp[i, c] += eps; Xm[i, c] -= eps
                args_p = [Xp if Y is X else Y for Y in (Q, K, V)]
                args_m = [Xm if Y is X else Y for Y in (Q, K, V)]
                fd = (loss(*args_p) - loss(*args_m)) / (2 * eps)
                assert abs(fd - G[i, c]) <= 1e-6 * max(1.0, abs(G[i, c])), (names, i, c, fd, G[i, c])


def test_backward_invariants():
    rng = np.random.default_rng(22)
    blocks = (3, 2, 4)
    t, off, s = _problem(rng, B=1, H=2, d=8, Ng=5, blocks=blocks, scale_q=2.0)
    g = _bwd(t, off, s)
    f = bits_to_f64
    # sum_j dV_j = sum_i dO_i (rows of P sum to 1), over all G and R rows/cols
    lhs = g["dv_gen"].sum(axis=1) + g["dv_ref"].sum(axis=1)
    rhs = f(t["do_gen"]).sum(axis=1) + f(t["do_ref"]).sum(axis=1)
    assert np.allclose(lhs, rhs, atol=1e-12)
    # sum_j dS_ij = 0 per row  <=>  sum_j dS_ij K_j with K = const gives dQ = 0
    t1 = dict(t)
    t1["k_gen"] = to_bf16_bits(np.full((1, 5, 2, 8), 0.5)); t1["k_ref"] = to_bf16_bits(np.full((1, 9, 2, 8), 0.5))
    g1 = _bwd(t1, off, s)
    assert np.abs(g1["dq_gen"]).max() < 1e-14 and np.abs(g1["dq_ref"]).max() < 1e-14
    # dK_g, dV_g independent of dO_r (R rows never see G keys)
    t2 = dict(t); t2["do_ref"] = rand_bits(rng, t["do_ref"].shape, 100.0)
    g2 = _bwd(t2, off, s)
    assert np.array_equal(g2["dk_gen"], g["dk_gen"]) and np.array_equal(g2["dv_gen"], g["dv_gen"])
    assert np.array_equal(g2["dq_gen"], g["dq_gen"])
    # dK_r, dV_r of block j depend only on dO_g and dO_r[j]: perturb dO_r of block 1 only
    t3 = dict(t); d3 = t["do_ref"].copy(); d3[:, off[1]:off[2]] = rand_bits(rng, d3[:, off[1]:off[2]].shape, 10.0)
    t3["do_ref"] = d3
    g3 = _bwd(t3, off, s)
    for j in (0, 2):
        sl = slice(off[j], off[j + 1])
        assert np.array_equal(g3["dk_ref"][:, sl], g["dk_ref"][:, sl]) and np.array_equal(g3["dv_ref"][:, sl], g["dv_ref"][:, sl])
    assert not np.allclose(g3["dk_ref"][:, off[1]:off[2]], g["dk_ref"][:, off[1]:off[2]])


# ------------------------------------------------------------------ sparse validity masking
def _delete_invalid(t, off, valid):
    """The same problem with the invalid reference tokens physically removed (blocks shrink, empty blocks vanish):
    an independent formulation of validity masking - no predicate, just a smaller unmasked SRA problem."""
    keep = np.flatnonzero(valid)
    out = dict(t)
    for k in ("q_ref", "k_ref", "v_ref", "do_ref"):
        if k in out:
            out[k] = np.ascontiguousarray(out[k][:, keep])
    off2 = [0]
    for j in range(len(off) - 1):
        c = int(np.count_nonzero(valid[off[j]:off[j + 1]]))
        if c:
            off2.append(off2[-1] + c)
    return out, off2, keep


@pytest.mark.parametrize("seed,Ng,blocks", [(0, 7, (5, 9, 3)), (1, 1, (4,)), (2, 12, (2, 2, 6, 1))])
def test_validity_mask_equals_deleting_invalid_tokens(seed, Ng, blocks):
    """Validity pins: (1) forward and backward with valid[] equal the unmasked oracle on the problem with the invalid
    tokens deleted (G rows, valid R rows, all gradients); (2) invalid R rows give O = 0, LSE = -inf and zero
    gradients; (3) the pair count has the closed form N_g (N_g + sum_j v_j) + sum_j v_j^2; (4) a block that is
    entirely invalid disappears; (5) valid = all ones changes nothing."""
    rng = np.random.default_rng(seed)
    off = [0]
    for b in blocks:
        off.append(off[-1] + b)
    Nr, B, H, d = off[-1], 2, 2, 8
    t = {k: rand_bits(rng, (B, Ng if k.endswith("gen") else Nr, H, d)) for k in
         ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref", "do_gen", "do_ref")}
    valid = rng.random(Nr) < 0.6
    valid[off[1]:off[2] if len(off) > 2 else off[1]] = False  # (4): kill the whole second block when there is one
    if not valid.any():
        valid[0] = True
    scale = 0.3
    a6 = [t[k] for k in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")]
    fm = sra_oracle.sra_forward(*a6, off, scale, valid=valid)
    bm = sra_oracle.sra_backward(*a6, t["do_gen"], t["do_ref"], off, scale, valid=valid)
    t2, off2, keep = _delete_invalid(t, off, valid)
    b6 = [t2[k] for k in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")]
    fd = sra_oracle.sra_forward(*b6, off2, scale)
    bd = sra_oracle.sra_backward(*b6, t2["do_gen"], t2["do_ref"], off2, scale)
    np.testing.assert_allclose(fm["o_gen"], fd["o_gen"], rtol=0, atol=1e-13)
    np.testing.assert_allclose(fm["lse_gen"], fd["lse_gen"], rtol=0, atol=1e-13)
    np.testing.assert_allclose(fm["o_ref"][:, keep], fd["o_ref"], rtol=0, atol=1e-13)
    np.testing.assert_allclose(fm["lse_ref"][:, :, keep], fd["lse_ref"], rtol=0, atol=1e-13)
    inv = np.flatnonzero(~valid)
    assert np.all(fm["o_ref"][:, inv] == 0.0) and np.all(np.isneginf(fm["lse_ref"][:, :, inv]))
    for g in ("dq", "dk", "dv"):
        np.testing.assert_allclose(bm[g + "_gen"], bd[g + "_gen"], rtol=0, atol=1e-12)
        np.testing.assert_allclose(bm[g + "_ref"][:, keep], bd[g + "_ref"], rtol=0, atol=1e-12)
        assert np.all(bm[g + "_ref"][:, inv] == 0.0)
    v = [int(np.count_nonzero(valid[off[j]:off[j + 1]])) for j in range(len(off) - 1)]
    assert sra_oracle.count_pairs(Ng, off, valid) == Ng * (Ng + sum(v)) + sum(x * x for x in v)
    ones = np.ones(Nr, dtype=bool)
    f1 = sra_oracle.sra_forward(*a6, off, scale, valid=ones)
    f0 = sra_oracle.sra_forward(*a6, off, scale)
    assert all(np.array_equal(f1[k], f0[k]) for k in f0)


# ------------------------------------------------------------------ sparse temporal attention
@pytest.mark.parametrize("seed,frames,blocks,w", [(0, (3, 5, 2, 4), (3, 4), 1), (1, (4, 4, 4), (), 0), (2, (2, 3, 1, 5, 2), (6,), 2)])
def test_temporal_window_mask_and_gradients(seed, frames, blocks, w):
    """Temporal-window pins: (1) the mask equals an independently written |frame(i) - frame(j)| <= w rule
    (searchsorted, not the oracle's block lookup) on G x G and is untouched elsewhere; (2) forward and backward equal
    torch fp64 SDPA + autograd under that boolean mask (library routine); (3) w >= n_frames - 1 is plain SRA; (4) w = 0
    without a reference is per-frame dense attention; (5) pair count = sum_f n_f (window keys_f + N_r) + sum_j b_j^2."""
    rng = np.random.default_rng(seed)
    fr = np.concatenate([[0], np.cumsum(frames)]).astype(np.int64)
    off = [0]
    for b in blocks:
        off.append(off[-1] + b)
    Ng, Nr, B, H, d = int(fr[-1]), off[-1], 1, 2, 8
    fid = np.searchsorted(fr, np.arange(Ng), side="right") - 1
    M = sra_oracle.sra_mask(Ng, off, None, fr, w).astype(bool)
    M0 = sra_oracle.sra_mask(Ng, off).astype(bool)
    want = M0.copy()
    want[:Ng, :Ng] = np.abs(fid[:, None] - fid[None, :]) <= w
    assert np.array_equal(M, want)
    assert np.array_equal(sra_oracle.sra_mask(Ng, off, None, fr, len(frames) - 1), M0.astype(np.uint8))
    keys = [int(fr[min(len(frames), f + w + 1)] - fr[max(0, f - w)]) for f in range(len(frames))]
    assert int(M.sum()) == sum(n * (k + Nr) for n, k in zip(frames, keys)) + sum(b * b for b in blocks)
    t = {k: rand_bits(rng, (B, Ng if k.endswith("gen") else Nr, H, d)) for k in
         ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref", "do_gen", "do_ref")}
    scale = 0.35
    a6 = [t[k] for k in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")]
    fwd = sra_oracle.sra_forward(*a6, off, scale, gen_frame_offsets=fr, window=w)
    bwd = sra_oracle.sra_backward(*a6, t["do_gen"], t["do_ref"], off, scale, gen_frame_offsets=fr, window=w)
    cat = lambda g, r: torch.tensor(np.concatenate([bits_to_f64(t[g]), bits_to_f64(t[r])], axis=1)[0].transpose(1, 0, 2))
    q, k, v = (cat(a, b).requires_grad_(True) for a, b in (("q_gen", "q_ref"), ("k_gen", "k_ref"), ("v_gen", "v_ref")))
    do = cat("do_gen", "do_ref")
    o = torch.nn.functional.scaled_dot_product_attention(q, k, v, attn_mask=torch.tensor(want), scale=scale)
    o.backward(do)
    o_or = np.concatenate([fwd["o_gen"], fwd["o_ref"]], axis=1)[0].transpose(1, 0, 2) if Nr else fwd["o_gen"][0].transpose(1, 0, 2)
    np.testing.assert_allclose(o_or, o.detach().numpy(), rtol=0, atol=1e-12)
    for name, g in (("dq", q.grad), ("dk", k.grad), ("dv", v.grad)):
        got = np.concatenate([bwd[name + "_gen"], bwd[name + "_ref"]], axis=1)[0].transpose(1, 0, 2)
        np.testing.assert_allclose(got, g.numpy(), rtol=0, atol=1e-11)
    if w == 0 and Nr == 0:
        for f in range(len(frames)):
            sl = slice(int(fr[f]), int(fr[f + 1]))
            qf, kf, vf = (torch.tensor(bits_to_f64(t[n])[0, sl].transpose(1, 0, 2)) for n in ("q_gen", "k_gen", "v_gen"))
            of = torch.nn.functional.scaled_dot_product_attention(qf, kf, vf, scale=scale)
            np.testing.assert_allclose(fwd["o_gen"][0, sl].transpose(1, 0, 2), of.numpy(), rtol=0, atol=1e-12)


# ------------------------------------------------------------------ per-sample validity (reading A12)
@pytest.mark.parametrize("seed,Ng,blocks", [(3, 6, (4, 7, 2)), (4, 2, (5,))])
def test_per_sample_validity_equals_per_item_deletion(seed, Ng, blocks):
    """valid of shape [B, n_ref]: batch item b must equal the UNMASKED oracle run on item b alone with ITS invalid
    tokens physically deleted (forward, LSE and all six gradients) - numpy oracle and C oracle (every row / column)."""
    rng = np.random.default_rng(seed)
    off = [0]
    for b in blocks:
        off.append(off[-1] + b)
    Nr, B, H, d = off[-1], 3, 2, 8
    t = {k: rand_bits(rng, (B, Ng if k.endswith("gen") else Nr, H, d)) for k in
         ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref", "do_gen", "do_ref")}
    valid = rng.random((B, Nr)) < 0.6
    valid[0, :] = True                       # item 0: nothing masked
    valid[1, off[0]:off[1]] = False          # item 1: its first block disappears
    valid[np.arange(B), rng.integers(0, Nr, B)] |= ~valid.any(axis=1)  # never all-invalid here
    assert not np.array_equal(valid[1], valid[2])
    scale = 0.3
    a6 = [t[k] for k in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")]
    fm = sra_oracle.sra_forward(*a6, off, scale, valid=valid)
    bm = sra_oracle.sra_backward(*a6, t["do_gen"], t["do_ref"], off, scale, valid=valid)
    n = Ng + Nr
    oc, lc = c_oracle.forward_rows(*a6, off, scale, np.arange(n, dtype=np.int32), valid=valid)
    for b in range(B):
        tb = {k: v[b:b + 1] for k, v in t.items()}
        t2, off2, keep = _delete_invalid(tb, off, valid[b])
        b6 = [t2[k] for k in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")]
        fd = sra_oracle.sra_forward(*b6, off2, scale)
        bd = sra_oracle.sra_backward(*b6, t2["do_gen"], t2["do_ref"], off2, scale)
        inv = np.flatnonzero(~valid[b])
        np.testing.assert_allclose(fm["o_gen"][b], fd["o_gen"][0], rtol=0, atol=1e-13)
        np.testing.assert_allclose(fm["o_ref"][b][keep], fd["o_ref"][0], rtol=0, atol=1e-13)
        np.testing.assert_allclose(fm["lse_ref"][b][:, keep], fd["lse_ref"][0], rtol=0, atol=1e-13)
        assert np.all(fm["o_ref"][b][inv] == 0.0) and np.all(np.isneginf(fm["lse_ref"][b][:, inv]))
        # C oracle, all rows of item b
        np.testing.assert_allclose(oc[b, :Ng], fd["o_gen"][0], rtol=0, atol=1e-13)
        np.testing.assert_allclose(oc[b, Ng:][keep], fd["o_ref"][0], rtol=0, atol=1e-13)
        np.testing.assert_allclose(lc[b][:, :Ng], fd["lse_gen"][0], rtol=0, atol=1e-13)
        assert np.all(oc[b, Ng:][inv] == 0.0) and np.all(np.isneginf(lc[b][:, Ng:][:, inv]))
        for g in ("dq", "dk", "dv"):
            np.testing.assert_allclose(bm[g + "_gen"][b], bd[g + "_gen"][0], rtol=0, atol=1e-12)
            np.testing.assert_allclose(bm[g + "_ref"][b][keep], bd[g + "_ref"][0], rtol=0, atol=1e-12)
            assert np.all(bm[g + "_ref"][b][inv] == 0.0)
        for h in range(H):
            o, lse = c_oracle.forward_head(*a6, off, scale, b, h, valid=valid)
            dq, dk, dv = c_oracle.backward_head(*a6, t["do_gen"], t["do_ref"], off, scale, b, h, o, lse, valid=valid)
            for name, got in (("dq", dq), ("dk", dk), ("dv", dv)):
                np.testing.assert_allclose(got[:Ng], bd[name + "_gen"][0, :, h], rtol=0, atol=1e-12)
                np.testing.assert_allclose(got[Ng:][keep], bd[name + "_ref"][0, :, h], rtol=0, atol=1e-12)
                assert np.all(got[Ng:][inv] == 0.0)


# ------------------------------------------------------------------ C oracle under valid[] and the frame window
@pytest.mark.parametrize("seed,frames,blocks,w,use_valid", [(5, (3, 5, 2, 4), (3, 4, 6), 1, True), (6, (4, 4, 4), (5,), 0, False),
                                                            (7, (2, 3, 1, 5, 2), (6, 2), 2, True), (8, (9,), (4, 3), -1, True)])
def test_c_oracle_valid_and_window(seed, frames, blocks, w, use_valid):
    """The C oracle's optional masks (PAPER.md:225 validity, PAPER.md:143 frame window), pinned three ways:
    (1) every row of its forward equals torch fp64 SDPA under a boolean mask built HERE from first principles
    (frame ids by searchsorted, block ids by repeat - not the oracle's lookup); (2) its backward (all rows, all
    columns, and a sampled subset) equals torch autograd under that mask; (3) with a validity mask, the problem with the
    invalid tokens physically deleted, solved by the unmasked C oracle, gives the same G rows and kept R rows;
    (4) its pair count equals the mask's sum.  The numpy oracle must agree too."""
    rng = np.random.default_rng(seed)
    fr = np.concatenate([[0], np.cumsum(frames)]).astype(np.int32)
    off = np.concatenate([[0], np.cumsum(blocks)]).astype(np.int32)
    Ng, Nr, B, H, d = int(fr[-1]), int(off[-1]), 2, 2, 8
    t = {k: rand_bits(rng, (B, Ng if k.endswith("gen") else Nr, H, d)) for k in
         ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref", "do_gen", "do_ref")}
    valid = None
    if use_valid:
        valid = rng.random(Nr) < 0.65
        valid[off[0]:off[1]] = valid[off[0]:off[1]] | (np.arange(off[1]) == 0)   # keep one token of block 0
        if len(blocks) > 1:
            valid[off[1]:off[2]] = False                                            # block 1 disappears
    # the mask from first principles
    fid = np.searchsorted(fr, np.arange(Ng), side="right") - 1
    bid = np.repeat(np.arange(len(blocks)), blocks)
    n = Ng + Nr
    M = np.zeros((n, n), dtype=bool)
    M[:Ng, :Ng] = (np.abs(fid[:, None] - fid[None, :]) <= w) if w >= 0 else True
    M[:Ng, Ng:] = True
    M[Ng:, Ng:] = bid[:, None] == bid[None, :]
    if valid is not None:
        M[:, Ng:] &= valid[None, :]
        M[Ng:, :] &= valid[:, None]
    scale = 0.4
    a6 = [t[k] for k in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")]
    kw = dict(valid=valid, gen_frame_offsets=fr, window=w)
    assert c_oracle.count_pairs(Ng, off, **kw) == int(M.sum())
    oc, lc = c_oracle.forward_rows(*a6, off, scale, np.arange(n, dtype=np.int32), **kw)
    on = sra_oracle.sra_forward(*a6, off, scale, **kw)
    bn = sra_oracle.sra_backward(*a6, t["do_gen"], t["do_ref"], off, scale, **kw)
    empty = ~M.any(axis=1)
    for b in range(B):
        cat = lambda g, r: torch.tensor(np.concatenate([bits_to_f64(t[g][b]), bits_to_f64(t[r][b])], axis=0).transpose(1, 0, 2))
        q, k, v = (cat(x, y).requires_grad_(True) for x, y in (("q_gen", "q_ref"), ("k_gen", "k_ref"), ("v_gen", "v_ref")))
        do = cat("do_gen", "do_ref")
        # torch SDPA returns NaN for empty rows: give them one dummy visible key and zero their dO, then compare the rest
        Mt = M.copy()
        Mt[empty, 0] = True
        do_t = do.clone()
        do_t[:, empty] = 0.0
        o = torch.nn.functional.scaled_dot_product_attention(q, k, v, attn_mask=torch.tensor(Mt), scale=scale)
        o.backward(do_t)
        want = o.detach().numpy().transpose(1, 0, 2)          # [n, H, d]
        np.testing.assert_allclose(oc[b][~empty], want[~empty], rtol=0, atol=1e-12)
        assert np.all(oc[b][empty] == 0.0) and np.all(np.isneginf(lc[b][:, empty]))
        np.testing.assert_allclose(np.concatenate([on["o_gen"][b], on["o_ref"][b]]), oc[b], rtol=0, atol=1e-12)
        for h in range(H):
            oh, lh = c_oracle.forward_head(*a6, off, scale, b, h, **kw)
            np.testing.assert_allclose(oh, oc[b][:, h], rtol=0, atol=1e-13)
            dq, dk, dv = c_oracle.backward_head(*a6, t["do_gen"], t["do_ref"], off, scale, b, h, oh, lh, **kw)
            for name, got, g in (("dq", dq, q.grad), ("dk", dk, k.grad), ("dv", dv, v.grad)):
                ref = g.numpy()[h]
                np.testing.assert_allclose(got, ref, rtol=0, atol=1e-11)
                nb = np.concatenate([bn[name + "_gen"][b, :, h], bn[name + "_ref"][b, :, h]])
                np.testing.assert_allclose(got, nb, rtol=0, atol=1e-11)
            rows = np.array(sorted(rng.choice(n, size=min(5, n), replace=False)), dtype=np.int32)
            cols = np.array(sorted(rng.choice(n, size=min(4, n), replace=False)), dtype=np.int32)
            dq_s, dk_s, dv_s = c_oracle.backward_head(*a6, t["do_gen"], t["do_ref"], off, scale, b, h, oh, lh,
                                                      rows=rows, cols=cols, **kw)
            assert np.array_equal(dq_s, dq[rows]) and np.array_equal(dk_s, dk[cols]) and np.array_equal(dv_s, dv[cols])
    if valid is not None:
        t2, off2, keep = _delete_invalid(t, list(off), valid)
        b6 = [t2[k] for k in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")]
        n2 = Ng + len(keep)
        od, ld = c_oracle.forward_rows(*b6, off2, scale, np.arange(n2, dtype=np.int32), gen_frame_offsets=fr, window=w)
        np.testing.assert_allclose(oc[:, :Ng], od[:, :Ng], rtol=0, atol=1e-13)
        np.testing.assert_allclose(oc[:, Ng:][:, keep], od[:, Ng:], rtol=0, atol=1e-13)
        np.testing.assert_allclose(lc[:, :, Ng:][:, :, keep], ld[:, :, Ng:], rtol=0, atol=1e-13)


# ----------------------------------------------------------------------------- RoPE producer (reading A18)
def _angles(N, half, rng=None, base=10000.0):
    """theta[t, i] = t * base^(-i / half): the 1-D RoFormer table, the structure the relative-position pin needs."""
    w = base ** (-np.arange(half) / half)
    return np.arange(N)[:, None] * w[None, :]


def test_rope_literal_cases():
    """Values the definition fixes: angle 0 = identity; pi/2 maps the pair (a, b) -> (-b, a); pi negates; a unit vector
    in element 0 becomes (cos, sin) in elements (0, 1) - this pins the interleaved pairing (not (0, d/2)) and the sign
    of the sine term."""
    x = np.zeros((1, 4, 1, 8))
    x[0, :, 0, :] = [[1, 2, 3, 4, 5, 6, 7, 8]] * 4
    bits = to_bf16_bits(x)
    th = np.array([0.0, np.pi / 2, np.pi, 0.0])[:, None] * np.ones((1, 4))
    y = sra_oracle.rope(bits, np.cos(th), np.sin(th))
    np.testing.assert_allclose(y[0, 0, 0], [1, 2, 3, 4, 5, 6, 7, 8], atol=1e-14)
    np.testing.assert_allclose(y[0, 1, 0], [-2, 1, -4, 3, -6, 5, -8, 7], atol=1e-14)
    np.testing.assert_allclose(y[0, 2, 0], [-1, -2, -3, -4, -5, -6, -7, -8], atol=1e-14)
    e0 = np.zeros((1, 1, 1, 8)); e0[..., 0] = 1.0
    a = np.array([[0.3, 1.1, -0.7, 2.0]])
    y = sra_oracle.rope(to_bf16_bits(e0), np.cos(a), np.sin(a))[0, 0, 0]
    np.testing.assert_allclose(y, [math.cos(0.3), math.sin(0.3), 0, 0, 0, 0, 0, 0], atol=1e-15)
    # per-pair angles are used pair by pair: unit vector in element 5 (pair 2, imaginary part)
    e5 = np.zeros((1, 1, 1, 8)); e5[..., 5] = 1.0
    y = sra_oracle.rope(to_bf16_bits(e5), np.cos(a), np.sin(a))[0, 0, 0]
    np.testing.assert_allclose(y, [0, 0, 0, 0, -math.sin(-0.7), math.cos(-0.7), 0, 0], atol=1e-15)


def test_rope_brute_force_rotation_matrices():
    """Element by element with explicit 2x2 rotation matrices [[c, -s], [s, c]] in python loops."""
    rng = np.random.default_rng(5)
    B, N, H, d = 2, 5, 3, 6
    bits = rand_bits(rng, (B, N, H, d))
    th = rng.uniform(-4, 4, size=(N, d // 2))
    y = sra_oracle.rope(bits, np.cos(th), np.sin(th))
    x = bits_to_f64(bits)
    for b in range(B):
        for t in range(N):
            for h in range(H):
                for i in range(d // 2):
                    c, s = math.cos(th[t, i]), math.sin(th[t, i])
                    a, bb = x[b, t, h, 2 * i], x[b, t, h, 2 * i + 1]
                    assert abs(y[b, t, h, 2 * i] - (c * a - s * bb)) < 1e-14
                    assert abs(y[b, t, h, 2 * i + 1] - (s * a + c * bb)) < 1e-14


def test_rope_invariants():
    """(i) norms of every (token, head) vector are preserved; (ii) with theta = t * omega the score <rope(q)_m, rope(k)_n>
    depends on m - n only (the property RoPE exists for): shifting every position by the same amount leaves Q K^T
    unchanged, and the score equals Re sum_i q_i conj(k_i) e^{j (m - n) omega_i} computed directly; (iii) rotations
    compose: angles a then b = angle a + b."""
    rng = np.random.default_rng(6)
    B, N, H, d = 1, 7, 2, 16
    qb, kb = rand_bits(rng, (B, N, H, d)), rand_bits(rng, (B, N, H, d))
    th = _angles(N + 11, d // 2)
    q0, k0 = sra_oracle.rope(qb, np.cos(th[:N]), np.sin(th[:N])), sra_oracle.rope(kb, np.cos(th[:N]), np.sin(th[:N]))
    q1, k1 = sra_oracle.rope(qb, np.cos(th[11:]), np.sin(th[11:])), sra_oracle.rope(kb, np.cos(th[11:]), np.sin(th[11:]))
    x = bits_to_f64(qb)
    np.testing.assert_allclose(np.linalg.norm(q0, axis=-1), np.linalg.norm(x, axis=-1), rtol=1e-13)
    S0 = np.einsum("bmhd,bnhd->bhmn", q0, k0)
    S1 = np.einsum("bmhd,bnhd->bhmn", q1, k1)
    np.testing.assert_allclose(S0, S1, atol=1e-11)
    q, k = bits_to_f64(qb), bits_to_f64(kb)
    qc, kc = q[..., 0::2] + 1j * q[..., 1::2], k[..., 0::2] + 1j * k[..., 1::2]
    omega = th[1]
    for m in range(N):
        for n in range(N):
            want = (qc[0, m] * np.conj(kc[0, n]) * np.exp(1j * (m - n) * omega)[None, :]).sum(axis=-1).real
            np.testing.assert_allclose(S0[0, :, m, n], want, atol=1e-11)
    # composition (on values that survive the bf16 round trip exactly: small integers rotated by multiples of pi/2)
    xi = to_bf16_bits(rng.integers(-8, 9, size=(1, 4, 1, 8)).astype(np.float64))
    a = (np.pi / 2) * rng.integers(0, 4, size=(4, 4))
    bnd = (np.pi / 2) * rng.integers(0, 4, size=(4, 4))
    y1 = np.rint(sra_oracle.rope(xi, np.cos(a), np.sin(a)))
    y2 = sra_oracle.rope(to_bf16_bits(y1), np.cos(bnd), np.sin(bnd))
    np.testing.assert_allclose(y2, sra_oracle.rope(xi, np.cos(a + bnd), np.sin(a + bnd)), atol=1e-12)


def test_bf16_rounding_matches_library_and_ties():
    """f64_to_bf16_bits against torch's fp32 -> bf16 conversion (a different implementation) on values that are exact
    in fp32, plus hand-made ties: 1 + 2^-8 is halfway between 1 and 1 + 2^-7 -> even (1.0); 1 + 3 * 2^-8 -> 1 + 2^-6."""
    rng = np.random.default_rng(7)
    x = (rng.standard_normal(20000) * np.exp(rng.uniform(-20, 20, 20000))).astype(np.float32).astype(np.float64)
    np.testing.assert_array_equal(sra_oracle.f64_to_bf16_bits(x), to_bf16_bits(x))
    ties = np.array([1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -8, -(1.0 + 2.0 ** -8), 2.0 - 2.0 ** -8, 0.0])
    got = bits_to_f64(sra_oracle.f64_to_bf16_bits(ties))
    np.testing.assert_array_equal(got, [1.0, 1.0 + 2.0 ** -6, -1.0, 2.0, 0.0])
    # round trip: every bf16 value is a fixed point
    allb = np.arange(0x0080, 0x7F80, 7, dtype=np.uint16)
    np.testing.assert_array_equal(sra_oracle.f64_to_bf16_bits(sra_oracle.bf16_bits_to_f64(allb)), allb)


def test_rope_then_attention_is_relative():
    """End to end through the attention oracle: rotating Q and K by a table and by the same table shifted in position
    gives the same O (G rows, no reference) - the composition the cached-producer path relies on."""
    rng = np.random.default_rng(8)
    B, N, H, d = 1, 6, 1, 8
    qb, kb, vb = (rand_bits(rng, (B, N, H, d)) for _ in range(3))
    th = _angles(N + 5, d // 2)
    outs = []
    for sh in (0, 5):
        c, s = np.cos(th[sh:sh + N]), np.sin(th[sh:sh + N])
        # fp64 rotated values are not bf16: run the attention definition on them directly
        Q, K = sra_oracle.rope(qb, c, s)[0, :, 0], sra_oracle.rope(kb, c, s)[0, :, 0]
        O, _, _ = sra_oracle.masked_attention(Q, K, bits_to_f64(vb)[0, :, 0], np.ones((N, N), np.uint8), 1 / math.sqrt(d))
        outs.append(O)
    np.testing.assert_allclose(outs[0], outs[1], atol=1e-12)

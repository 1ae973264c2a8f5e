"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

A full fp64 pass is 37-199 TFLOP (hours of CPU), so the oracle evaluates SAMPLED outputs exactly: an output row
depends only on its own Q row and the K/V it may see, so row sampling is exact, not approximate.
Inputs are drawn on the device with the recipe of `inputs.make_tensor_device`; whatever the
oracle consumes is copied back bit for bit, for the sampled heads only (the oracle gets an H = len(heads)
problem: heads are independent).  Properties that hold at any size (finiteness, cached step == uncached step,
cost model) are checked on the whole output.

Contract tolerance (BASELINE.json north_star): bf16 I/O, fp32 accumulation, max-abs <= 2e-2 and mean-abs <= 2e-3,
plus rel_l2 <= 1e-2 and LSE max-abs <= 2e-3.
"""
import math

import numpy as np
import pytest
import torch

from oracle import c_oracle
from paper_2606_13872_b200 import inputs as sra_inputs
from tests.gpu_util import boundary_rows
from tests.util import assert_parity

pytestmark = pytest.mark.gpu
LSE_TOL = 2e-3
NAMES6 = ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")


def _device_inputs(w, names, dev, step=0):
    return {n: sra_inputs.make_tensor_device(w, n, dev, step=step) for n in names}


def _head_bits(t, heads, b=None):
    """bf16 bit patterns of the listed heads (and optionally one batch item) as an H = len(heads) problem."""
    out = {}
    for n, x in t.items():
        x = x[:, :, heads] if b is None else x[b:b + 1][:, :, heads]
        out[n] = sra_inputs.bf16_bits(x.contiguous().cpu())
    return out


def _forward_sampled(w, heads, n_random=8, steps=1, invalid_frac=0.0, window=-1, n_frames=21):
    """Step 0 (cache build + G and R rows) and `steps - 1` cached denoising steps (G rows only, fresh G tensors,
    resident reference K/V) of workload `w`; every step checked on sampled rows of `heads`.
    invalid_frac > 0: a seeded validity mask over the reference tokens (the mask bench.py
    --invalid-frac draws); window >= 0: sparse temporal attention over `n_frames` equal frames;
    the C oracle materialises both restrictions in its visibility predicate."""
    from paper_2606_13872_b200 import binding as B
    dev = torch.device("cuda:0")
    scale = 1.0 / math.sqrt(w.head_dim)
    ref = _device_inputs(w, ("q_ref", "k_ref", "v_ref"), dev)
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    valid = frames = None
    okw = {}
    try:
        if invalid_frac > 0:
            valid = np.random.default_rng(w.seed).random(w.n_ref) >= invalid_frac
            B.sra_set_reference_validity(ctx, valid)
            okw["valid"] = valid
        if window >= 0:
            frames = [i * (w.n_gen // n_frames) for i in range(n_frames)] + [w.n_gen]
            B.sra_set_temporal_window(ctx, frames, window)
            okw.update(gen_frame_offsets=frames, window=window)
        B.sra_cache_reference_kv(ctx, ref["k_ref"], ref["v_ref"])
        cache_bytes = B.sra_cache_bytes(ctx)
        n_cached = w.n_ref if valid is None else int(valid.sum())
        assert cache_bytes == 2 * w.batch * n_cached * w.heads * w.head_dim * 2
        o_gen = torch.empty((w.batch, w.n_gen, w.heads, w.head_dim), device=dev, dtype=torch.bfloat16)
        o_ref = torch.empty_like(ref["q_ref"])
        lse_gen = torch.empty((w.batch, w.heads, w.n_gen), device=dev)
        lse_ref = torch.empty((w.batch, w.heads, w.n_ref), device=dev)
        rows = boundary_rows(w, n_random=n_random)
        for step in range(steps):
            gen = _device_inputs(w, ("q_gen", "k_gen", "v_gen"), dev, step=step)
            o_gen.fill_(float("nan"))
            launches0 = B.sra_launch_count(ctx)
            if step == 0:
                B.sra_forward(ctx, gen["q_gen"], gen["k_gen"], gen["v_gen"], o_gen, q_ref=ref["q_ref"], o_ref=o_ref,
                              lse_gen=lse_gen, lse_ref=lse_ref)
                use_rows = rows
            else:  # cached denoising step: q_ref = NULL, k_ref = v_ref = NULL -> resident cache, R rows skipped
                B.sra_forward(ctx, gen["q_gen"], gen["k_gen"], gen["v_gen"], o_gen, lse_gen=lse_gen)
                use_rows = rows[rows < w.n_gen]
            torch.cuda.synchronize()
            n_split, _ = B.sra_split_schedule_copy(ctx)
            if valid is None or step > 0:  # (step 0 under a validity mask also gathers Q_r and scatters O_r / LSE_r)
                assert B.sra_launch_count(ctx) - launches0 == (1 if n_split == 1 else 2), \
                    "one forward = one kernel launch (+ the partial merge of a key-split schedule), no cache re-copy"
            assert B.sra_cache_bytes(ctx) == cache_bytes
            assert torch.isfinite(o_gen.float()).all()
            tb = _head_bits({**gen, **ref}, heads)
            o_or, lse_or = c_oracle.forward_rows(*[tb[n] for n in NAMES6], w.ref_block_offsets, scale, use_rows, **okw)
            g = use_rows[use_rows < w.n_gen]
            r = use_rows[use_rows >= w.n_gen] - w.n_gen
            o_gpu = [o_gen[:, torch.as_tensor(g, device=dev).long()][:, :, heads].float().cpu().numpy()]
            l_gpu = [lse_gen[:, heads][:, :, torch.as_tensor(g, device=dev).long()].cpu().numpy()]
            if len(r):
                o_gpu.append(o_ref[:, torch.as_tensor(r, device=dev).long()][:, :, heads].float().cpu().numpy())
                l_gpu.append(lse_ref[:, heads][:, :, torch.as_tensor(r, device=dev).long()].cpu().numpy())
            assert_parity(np.concatenate(o_gpu, axis=1), o_or, f"{w.name} step {step} sampled O")
            l_gpu = np.concatenate(l_gpu, axis=2)
            empty = np.isneginf(lse_or)  # rows of invalid reference tokens: O = 0, LSE = -inf on both sides (A8)
            assert np.array_equal(np.isneginf(l_gpu), empty)
            assert np.abs(l_gpu[~empty] - lse_or[~empty]).max() <= LSE_TOL
            if valid is not None and step == 0:
                assert empty.any() and (~empty).any(), "the sample must hold valid and invalid reference rows"
    finally:
        B.sra_destroy(ctx)


def test_720p_step0_and_cached_steps():
    """BASELINE.json configs[2]: 720p, "reuse cached ref KV over 8 denoising steps": step 0 builds
    the cache and computes G and R rows, steps 1-7 are cached steps with fresh generation tensors."""
    _forward_sampled(sra_inputs.WORKLOADS["720p"], heads=[0, 39], n_random=8, steps=8)


def test_720p_invalid_reference_tokens():
    """The shape `bench.py --invalid-frac 0.3` quotes: 30 % of the reference tokens invalid, the
    resident cache holds the valid ones only; step 0 + one cached step against the validity-aware C oracle."""
    _forward_sampled(sra_inputs.WORKLOADS["720p"], heads=[7], n_random=16, steps=2, invalid_frac=0.3)


def test_720p_temporal_window():
    """The shape `bench.py --window 2` quotes (reading A17): generation keys of frames within +-2."""
    _forward_sampled(sra_inputs.WORKLOADS["720p"], heads=[31], n_random=16, steps=2, window=2)


def test_480p_dist_a():
    """BASELINE.json configs[1] by name, under its own distribution (reading A of A14)."""
    w = sra_inputs.WORKLOADS["480p"]
    assert w.dist == "A"
    _forward_sampled(w, heads=[0, 20], n_random=16, steps=2)


def test_720p_dist_b():
    """Same shape with unit-variance elements (reading B of SURVEY.md 8c A14): a peaked softmax at full length."""
    _forward_sampled(sra_inputs.WORKLOADS["720p"].replace(dist="B"), heads=[17], n_random=8, steps=1)


@pytest.mark.parametrize("name", ["sweep5s", "sweep10s", "sweep20s", "sweep40s"])
def test_long_reference_sweep_endpoints(name):
    """BASELINE.json configs[3]: every point of the sweep, 5 s to 40 s (174,720 reference tokens, 3.58 GB cache)."""
    _forward_sampled(sra_inputs.WORKLOADS[name], heads=[3], n_random=8, steps=2)


@pytest.mark.parametrize("name", ["short128", "short512", "short2048"])
def test_short_query_against_40s_cache(name):
    """north_star's cache-bound short-query cases: 128 / 512 / 2048 generation rows against the 40 s resident
    cache; the 128- and 512-row schedules are key-split (partials + merge), 2048 is not."""
    _forward_sampled(sra_inputs.WORKLOADS[name], heads=[0, 21], n_random=24, steps=2)


def test_sweep_cost_is_linear_in_reference_length():
    """cost linear in reference length.  Property that holds at any size, read from the
    library's own schedule: scheduled key tiles (= issued MMA work) grow affinely with N_r and stay within 1.5 %
    of the useful (unmasked) work, whereas dense concatenated attention would grow quadratically."""
    from paper_2606_13872_b200 import binding as B
    pts = []
    for name in ("sweep5s", "sweep10s", "sweep20s", "sweep40s"):
        w = sra_inputs.WORKLOADS[name]
        ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
        try:
            issued = 0  # (query rows x key columns) the tensor cores are asked to do, per (batch, head)
            for it in B.sra_schedule_copy(ctx):
                q_tiles = 2 if it["q_rows"] > 128 else 1
                k_tiles = -(-it["seg0_len"] // 128) + -(-it["seg1_len"] // 128)
                issued += q_tiles * 128 * k_tiles * 128
            useful = B.sra_useful_flops(ctx, True, False) / (4 * w.head_dim * w.heads * w.batch)
            assert useful <= issued <= 1.015 * useful, (name, issued, useful)
            pts.append((w.n_ref, issued))
        finally:
            B.sra_destroy(ctx)
    x = np.array([p[0] for p in pts], dtype=np.float64)
    y = np.array([p[1] for p in pts], dtype=np.float64)
    a, c = np.polyfit(x, y, 1)
    assert np.abs(a * x + c - y).max() <= 2e-3 * y.max(), "scheduled work is not affine in reference length"
    dense = (w.n_gen + x) ** 2
    assert y[-1] / y[0] < 4.0 < dense[-1] / dense[0]


def test_train_config_forward_backward_sampled():
    """BASELINE.json configs[4]: B2 H40 d128, 32,760 gen + 21,840 ref tokens, Q/K/V/dO ~ N(0,1).  dK/dV of a key
    need LSE and D of EVERY row that sees it, so the oracle runs the full forward of one (batch, head) (0.9 TFLOP
    of fp64) and then the backward on sampled query rows (dQ) and sampled key columns (dK, dV)."""
    from paper_2606_13872_b200 import binding as B
    w = sra_inputs.WORKLOADS["train"]
    dev = torch.device("cuda:0")
    scale = 1.0 / math.sqrt(w.head_dim)
    t = _device_inputs(w, sra_inputs.TENSOR_ORDER, dev)
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        o_gen, o_ref = torch.empty_like(t["q_gen"]), torch.empty_like(t["q_ref"])
        lse_gen = torch.empty((w.batch, w.heads, w.n_gen), device=dev)
        lse_ref = torch.empty((w.batch, w.heads, w.n_ref), device=dev)
        grads = {n: torch.full_like(t["q_gen" if n.endswith("_gen") else "q_ref"], float("nan"))
                 for n in ("dq_gen", "dk_gen", "dv_gen", "dq_ref", "dk_ref", "dv_ref")}
        B.sra_forward(ctx, t["q_gen"], t["k_gen"], t["v_gen"], o_gen, q_ref=t["q_ref"], k_ref=t["k_ref"],
                      v_ref=t["v_ref"], o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref)
        B.sra_backward(ctx, q_gen=t["q_gen"], k_gen=t["k_gen"], v_gen=t["v_gen"], q_ref=t["q_ref"], k_ref=t["k_ref"],
                       v_ref=t["v_ref"], o_gen=o_gen, o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref,
                       do_gen=t["do_gen"], do_ref=t["do_ref"], **grads)
        torch.cuda.synchronize()
        for g in grads.values():
            assert torch.isfinite(g.float()).all()
        for b, h in ((1, 23), (0, 6)):  # both batch items (each oracle pass is a full fp64 forward of one (b, h))
            tb = _head_bits(t, [h], b=b)
            args6 = [tb[n] for n in NAMES6]
            o, lse = c_oracle.forward_head(*args6, w.ref_block_offsets, scale, 0, 0)
            n = w.n_gen + w.n_ref
            off = w.ref_block_offsets
            rng = np.random.default_rng(1)
            edge = [0, 63, 64, 127, 128, w.n_gen - 1, w.n_gen, w.n_gen + off[1] - 1, w.n_gen + off[1], n - 1]
            rows = np.asarray(sorted(set(edge) | set(int(x) for x in rng.integers(0, n, 24))), dtype=np.int32)
            cols = np.asarray(sorted(set(edge) | set(int(x) for x in rng.integers(0, n, 24))), dtype=np.int32)
            # forward of the sampled rows first (the backward consumes the GPU's own O and LSE, as a training step does)
            gi, ri = rows[rows < w.n_gen], rows[rows >= w.n_gen] - w.n_gen
            o_gpu = np.concatenate([o_gen[b, :, h][torch.as_tensor(gi, device=dev).long()].float().cpu().numpy(),
                                    o_ref[b, :, h][torch.as_tensor(ri, device=dev).long()].float().cpu().numpy()], axis=0)
            assert_parity(o_gpu, o[rows], "train config sampled O")
            dq, dk, dv = c_oracle.backward_head(*args6, tb["do_gen"], tb["do_ref"], off, scale, 0, 0, o, lse, rows=rows,
                                                cols=cols)
            for name, ref, idx in (("dq", dq, rows), ("dk", dk, cols), ("dv", dv, cols)):
                gi, ri = idx[idx < w.n_gen], idx[idx >= w.n_gen] - w.n_gen
                got = np.concatenate(
                    [grads[name + "_gen"][b, :, h][torch.as_tensor(gi, device=dev).long()].float().cpu().numpy(),
                     grads[name + "_ref"][b, :, h][torch.as_tensor(ri, device=dev).long()].float().cpu().numpy()], axis=0)
                assert_parity(got, ref, f"train config sampled {name}")
    finally:
        B.sra_destroy(ctx)

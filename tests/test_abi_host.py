"""-m "not gpu": the C-ABI library loads, exports every symbol include/sra.h declares, validates its
arguments, and its host-side tile schedule covers exactly the unmasked pairs of the
explicit SRA mask.  No compute entry point is exercised here beyond its "no device" error path."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import sra_oracle
from paper_2606_13872_b200 import binding as B
from paper_2606_13872_b200 import inputs as sra_inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "sra.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sra_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported():
    names = _declared_symbols()
    assert {"sra_create", "sra_cache_reference_kv", "sra_forward", "sra_backward", "sra_destroy"} <= set(names)
    for n in names:
        assert hasattr(B.lib, n), f"{n} declared in include/sra.h but not exported by libsra_b200.so"
    assert set(names) == set(B.EXPORTS), (names, B.EXPORTS)


def test_status_strings():
    assert B.lib.sra_status_string(0) == b"SRA_OK"
    assert B.lib.sra_status_string(-4) == b"SRA_ERR_NO_REF_CACHE"
    assert B.lib.sra_status_string(-99) == b"SRA_ERR_UNKNOWN"


@pytest.mark.parametrize("kw,status", [
    (dict(head_dim=96), B.SRA_ERR_UNSUPPORTED),
    (dict(batch=0), B.SRA_ERR_INVALID_ARG),
    (dict(n_gen=0), B.SRA_ERR_INVALID_ARG),
    (dict(ref_block_offsets=[0, 5, 5]), B.SRA_ERR_INVALID_ARG),
    (dict(ref_block_offsets=[1, 5]), B.SRA_ERR_INVALID_ARG),
    (dict(ref_block_offsets=[0, 7, 3]), B.SRA_ERR_INVALID_ARG),
])
def test_create_rejects_bad_configs(kw, status):
    base = dict(batch=1, heads=2, head_dim=64, n_gen=10, ref_block_offsets=[0, 4, 9])
    base.update(kw)
    with pytest.raises(B.SRAError) as e:
        B.sra_create(**base)
    assert e.value.status == status


def test_null_handling():
    assert B.lib.sra_create(None, None) == B.SRA_ERR_INVALID_ARG
    B.sra_destroy(None)  # NULL-safe
    assert B.lib.sra_forward(None, None, None) == B.SRA_ERR_INVALID_ARG
    assert B.lib.sra_backward(None, None, None) == B.SRA_ERR_INVALID_ARG
    assert B.lib.sra_forward_host(None, None, None) == B.SRA_ERR_INVALID_ARG
    assert B.lib.sra_cache_bytes(None) == 0
    assert B.lib.sra_cache_reference_kv_rope(None, None, None, None, None, None) == B.SRA_ERR_INVALID_ARG
    assert B.lib.sra_apply_rope(None, None, None, None, None, 4, None) == B.SRA_ERR_INVALID_ARG


def _covered_pairs(items, n_gen, n_ref):
    """Pair-coverage count matrix implied by the schedule: rows/cols [G ; R]."""
    n = n_gen + n_ref
    C = np.zeros((n, n), dtype=np.int32)
    for it in items:
        r0 = it["q_row0"] + (n_gen if it["q_is_ref"] else 0)
        rows = slice(r0, r0 + it["q_rows"])
        s0 = it["seg0_start"] + (n_gen if it["seg0_is_ref"] else 0)
        C[rows, s0:s0 + it["seg0_len"]] += 1
        if it["seg1_len"]:
            s1 = it["seg1_start"] + n_gen
            C[rows, s1:s1 + it["seg1_len"]] += 1
    return C


@pytest.mark.parametrize("n_gen,blocks", [(256, (128,) * 4), (333, (1, 130, 257, 64, 200)), (1, (3,)), (700, ()),
                                          (300, (77, 128, 129, 5)), (513, (600,))])
def test_schedule_covers_exactly_the_mask(n_gen, blocks):
    """Every unmasked (query, key) pair is covered exactly once; no masked pair is ever scheduled
    ("eliminating redundant computation among tokens that do not require mutual interaction")."""
    off = [0]
    for b in blocks:
        off.append(off[-1] + b)
    ctx = B.sra_create(1, 1, 64, n_gen, off)
    try:
        items = B.sra_schedule_copy(ctx)
        C = _covered_pairs(items, n_gen, off[-1])
        M = sra_oracle.sra_mask(n_gen, off)
        assert np.array_equal(C, M.astype(np.int32))
        info = B.sra_schedule_info(ctx)
        assert info["n_gen_items"] + info["n_ref_items"] == len(items)
        for it in items:
            assert 1 <= it["q_rows"] <= 256
    finally:
        B.sra_destroy(ctx)


@pytest.mark.parametrize("heads,n_gen,blocks", [(40, 128, (1560,) * 112), (40, 512, (1560,) * 112), (2, 100, (1560, 1560, 300)),
                                                (2, 300, (1000, 1100)), (3, 3120, (1560,) * 3), (40, 2048, (1560,) * 112)])
def test_split_schedule_partitions_the_keys(heads, n_gen, blocks):
    """Short-query schedules: the key ranges of a generation slab's splits are whole 128-key tiles, non-empty,
    disjoint, and together cover every generation and reference key exactly once; reference items are unchanged."""
    off = [0]
    for b in blocks:
        off.append(off[-1] + b)
    ctx = B.sra_create(1, heads, 128, n_gen, off)
    try:
        plain = B.sra_schedule_copy(ctx)
        n_split, items = B.sra_split_schedule_copy(ctx)
        info = B.sra_schedule_info(ctx)
        if n_split == 1:
            assert [dict(it, split=0) for it in plain] == items
            assert info["n_gen_items"] * heads >= 2 * 148 or (n_gen + off[-1]) < 16 * 128
            return
        assert len(items) == info["n_gen_items"] * n_split + info["n_ref_items"]
        assert [dict(it, split=0) for it in plain[info["n_gen_items"]:]] == items[info["n_gen_items"] * n_split:]
        if n_gen + off[-1] <= 6000:
            C = _covered_pairs(items, n_gen, off[-1])
            assert np.array_equal(C, sra_oracle.sra_mask(n_gen, off).astype(np.int32))
        for g in range(info["n_gen_items"]):
            cov_g, cov_r = np.zeros(n_gen, dtype=np.int32), np.zeros(off[-1], dtype=np.int32)
            for sp in range(n_split):
                it = items[g * n_split + sp]
                cov_g[it["seg0_start"]:it["seg0_start"] + it["seg0_len"]] += 1
                cov_r[it["seg1_start"]:it["seg1_start"] + it["seg1_len"]] += 1
            assert (cov_g == 1).all() and (cov_r == 1).all()
            for sp in range(n_split):
                it = items[g * n_split + sp]
                assert it["split"] == sp + 1 and not it["q_is_ref"]
                assert (it["q_row0"], it["q_rows"]) == (plain[g]["q_row0"], plain[g]["q_rows"])
                assert it["seg0_start"] % 128 == 0 and it["seg1_start"] % 128 == 0
                assert it["seg0_len"] + it["seg1_len"] >= 8 * 128 - 127
    finally:
        B.sra_destroy(ctx)


@pytest.mark.parametrize("n_gen,blocks,seed", [(256, (128,) * 4, 0), (333, (1, 130, 257, 64, 200), 1), (50, (300, 5), 2)])
def test_validity_schedule_covers_exactly_the_valid_mask(n_gen, blocks, seed):
    """sra_set_reference_validity: the schedule is rebuilt on the compacted reference; mapped back
    through the compaction it covers every unmasked (query, key) pair of the validity-aware mask exactly once and
    nothing else, and the useful-FLOP count follows the valid tokens only.  NULL restores the plain schedule."""
    off = [0]
    for b in blocks:
        off.append(off[-1] + b)
    rng = np.random.default_rng(seed)
    valid = rng.random(off[-1]) < 0.7
    valid[off[1]:off[2]] = False  # one block entirely invalid
    keep = np.flatnonzero(valid)
    ctx = B.sra_create(1, 1, 64, n_gen, off)
    try:
        plain = B.sra_schedule_copy(ctx)
        B.sra_set_reference_validity(ctx, valid)
        items = B.sra_schedule_copy(ctx)
        n_c = len(keep)
        Cc = _covered_pairs(items, n_gen, n_c)  # in compact coordinates
        M = sra_oracle.sra_mask(n_gen, off, valid).astype(np.int32)
        idx = np.concatenate([np.arange(n_gen), n_gen + keep])
        assert np.array_equal(Cc, M[np.ix_(idx, idx)])
        assert M.sum() == Cc.sum(), "pairs outside the compacted rows/columns must all be masked"
        assert B.sra_useful_flops(ctx, True) == 4.0 * 64 * float(M.sum())
        B.sra_set_reference_validity(ctx, None)
        assert B.sra_schedule_copy(ctx) == plain
        B.sra_set_reference_validity(ctx, np.zeros(off[-1], dtype=bool))  # nothing valid: plain self-attention over G
        assert all(not it["q_is_ref"] and it["seg1_len"] == 0 for it in B.sra_schedule_copy(ctx))
    finally:
        B.sra_destroy(ctx)


@pytest.mark.parametrize("frames,blocks,w", [((300, 300, 300, 300), (128, 257), 1), ((100, 513, 77, 260, 5), (), 0),
                                             ((256,) * 6, (300,), 2), ((90, 90, 90), (64,), 5)])
def test_temporal_window_schedule_covers_exactly_the_mask(frames, blocks, w):
    """sra_set_temporal_window: forward slabs never straddle a frame, cover exactly the windowed mask,
    and the useful-FLOP count follows it; window < 0 restores the plain schedule."""
    fr = [0]
    for n in frames:
        fr.append(fr[-1] + n)
    off = [0]
    for b in blocks:
        off.append(off[-1] + b)
    ctx = B.sra_create(1, 1, 64, fr[-1], off)
    try:
        plain = B.sra_schedule_copy(ctx)
        B.sra_set_temporal_window(ctx, fr, w)
        items = B.sra_schedule_copy(ctx)
        M = sra_oracle.sra_mask(fr[-1], off, None, fr, w).astype(np.int32)
        assert np.array_equal(_covered_pairs(items, fr[-1], off[-1]), M)
        assert B.sra_useful_flops(ctx, True) == 4.0 * 64 * float(M.sum())
        for it in items:
            if not it["q_is_ref"]:
                f = max(i for i in range(len(frames)) if fr[i] <= it["q_row0"])
                assert it["q_row0"] + it["q_rows"] <= fr[f + 1], "a generation slab straddles a frame"
        assert B.sra_split_schedule_copy(ctx)[0] == 1
        B.sra_set_temporal_window(ctx, None, -1)
        assert B.sra_schedule_copy(ctx) == plain
    finally:
        B.sra_destroy(ctx)


@pytest.mark.parametrize("name", ["tiny", "480p", "720p", "sweep40s", "train"])
def test_useful_flops_closed_form(name):
    """sra_useful_flops = 4 d pairs H B with pairs = N_g (N_g + N_r) + sum b_j^2 (tests/golden/pairs.txt)."""
    w = sra_inputs.WORKLOADS[name]
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    try:
        pairs_g = w.n_gen * (w.n_gen + w.n_ref)
        pairs_r = sum(b * b for b in w.ref_block_sizes)
        f = 4.0 * w.head_dim * w.heads * w.batch
        assert B.sra_useful_flops(ctx, True) == pytest.approx(f * (pairs_g + pairs_r), rel=1e-12)
        assert B.sra_useful_flops(ctx, False) == pytest.approx(f * pairs_g, rel=1e-12)
        assert B.sra_useful_flops(ctx, True, backward=True) == pytest.approx(2.5 * f * (pairs_g + pairs_r), rel=1e-12)
        info = B.sra_schedule_info(ctx)
        # tile counts: G slabs visit ceil(Ng/128)+ceil(Nr/128) key tiles per 128-row q tile
        qt = -(-w.n_gen // 128)
        assert info["key_tiles_gen"] == qt * (-(-w.n_gen // 128) + -(-w.n_ref // 128))
    finally:
        B.sra_destroy(ctx)


def test_no_device_means_unsupported_not_fallback():
    """On a box without a CUDA device every compute entry point must fail loudly (no CPU path)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    ctx = B.sra_create(1, 1, 64, 8, [0, 4])
    try:
        a = B.sra_fwd_args()
        assert B.lib.sra_forward(ctx, ctypes.byref(a), None) in (B.SRA_ERR_UNSUPPORTED, B.SRA_ERR_INVALID_ARG)
        dummy = ctypes.c_void_p(16)
        assert B.lib.sra_cache_reference_kv(ctx, dummy, dummy, None) == B.SRA_ERR_UNSUPPORTED
        assert b"no CUDA device" in B.lib.sra_last_error(ctx)
        assert B.lib.sra_cache_reference_kv_rope(ctx, dummy, dummy, dummy, dummy, None) == B.SRA_ERR_UNSUPPORTED
        assert B.lib.sra_apply_rope(ctx, dummy, None, dummy, dummy, 8, None) == B.SRA_ERR_UNSUPPORTED
        bw = B.sra_bwd_args()
        assert B.lib.sra_backward(ctx, ctypes.byref(bw), None) == B.SRA_ERR_UNSUPPORTED
    finally:
        B.sra_destroy(ctx)


@pytest.mark.parametrize("heads,n_gen,blocks,frames,w", [(40, 75600 // 10, (3600,) * 2, None, -1), (2, 333, (1, 130, 257, 64, 200), None, -1),
                                                         (2, 1200, (700, 513), (300, 300, 300, 300), 1), (2, 513, (), None, -1),
                                                         (2, 256 * 5, (256 * 2,), None, -1)])
def test_pair_schedule_covers_the_slab_schedule(heads, n_gen, blocks, frames, w):
    """The CTA-pair launch list (sra_fwd_kernel<128, 2>): every 256-row slab sits in exactly one pair item, a pair item
    holds at most 512 consecutive rows of slabs that see the SAME key segments, G pairs come first, and the pair list
    covers exactly the pairs of the mask (the coverage matrix equals the oracle's explicit mask)."""
    off = [0]
    for b in blocks:
        off.append(off[-1] + b)
    ctx = B.sra_create(1, heads, 128, n_gen, off)  # (shapes with enough slabs per SM: no key split)
    try:
        fr = None
        if frames is not None:
            fr = [0]
            for f in frames:
                fr.append(fr[-1] + f)
            B.sra_set_temporal_window(ctx, fr, w)
        slabs = B.sra_schedule_copy(ctx)
        use_pairs, pairs = B.sra_pair_schedule_copy(ctx)
        assert use_pairs
        keyset = lambda it: tuple(it[k] for k in ("q_is_ref", "seg0_is_ref", "seg0_start", "seg0_len", "seg1_start", "seg1_len"))
        si = 0
        seen_ref = False
        for p in pairs:
            assert 1 <= p["q_rows"] <= 512
            seen_ref = seen_ref or bool(p["q_is_ref"])
            assert bool(p["q_is_ref"]) == seen_ref, "G pairs first, then R pairs"
            rows = 0
            while rows < p["q_rows"]:
                s = slabs[si]
                assert keyset(s) == keyset(p) and s["q_row0"] == p["q_row0"] + rows
                rows += s["q_rows"]
                si += 1
            assert rows == p["q_rows"]
        assert si == len(slabs)
        if n_gen + off[-1] <= 4000:
            M = sra_oracle.sra_mask(n_gen, off, None, fr, w).astype(np.int32)
            assert np.array_equal(_covered_pairs(pairs, n_gen, off[-1]), M)
    finally:
        B.sra_destroy(ctx)
    ctx = B.sra_create(1, 2, 64, n_gen, off)  # head_dim 64 keeps the single-CTA kernel
    try:
        assert not B.sra_pair_schedule_copy(ctx)[0]
    finally:
        B.sra_destroy(ctx)


def test_bound_ends_are_the_segment_ends_inside_the_tensors():
    """sra_bound_ends_copy (mask isolation for non-finite data): the ends the kernels bound their ragged tiles at are
    exactly the segment ends of the schedule that fall strictly inside a tensor - every reference block end but the
    last (per mask, in the mask's compacted rows), every frame end but the last once a temporal window is set - computed
    here independently from the block offsets, the frames and the validity flags."""
    n_gen, off = 1000, [0, 130, 387, 451, 700]
    ctx = B.sra_create(2, 2, 128, n_gen, off)
    try:
        assert B.sra_bound_ends_copy(ctx) == ([], [off[1:-1]])
        fr = [0, 100, 357, 400, 777, 1000]
        B.sra_set_temporal_window(ctx, fr, 1)
        assert B.sra_bound_ends_copy(ctx) == (fr[1:-1], [off[1:-1]])
        # every segment end of the forward schedule that is not a tensor end is in the table
        gen, ref = B.sra_bound_ends_copy(ctx)
        for it in B.sra_schedule_copy(ctx):
            e0 = it["seg0_start"] + it["seg0_len"]
            assert e0 in ((ref[0] + [off[-1]]) if it["seg0_is_ref"] else (gen + [n_gen]))
            if it["seg1_len"]:
                assert it["seg1_start"] + it["seg1_len"] in ref[0] + [off[-1]]
            eq = it["q_row0"] + it["q_rows"]
            if it["q_rows"] % 128:
                assert eq in ((ref[0] + [off[-1]]) if it["q_is_ref"] else (gen + [n_gen]))
        B.sra_set_temporal_window(ctx, None, -1)
        # per-sample validity: the ends of each item's COMPACTED blocks (empty blocks vanish)
        rng = np.random.default_rng(2)
        valid = rng.random((2, off[-1])) < 0.5
        valid[1, off[1]:off[2]] = False
        B.sra_set_reference_validity(ctx, valid)
        gen, ref = B.sra_bound_ends_copy(ctx)
        assert gen == []
        for b in range(2):
            counts = [int(valid[b, off[j]:off[j + 1]].sum()) for j in range(len(off) - 1)]
            ends = np.cumsum([c for c in counts if c > 0]).tolist()
            assert ref[b] == ends[:-1]
    finally:
        B.sra_destroy(ctx)


def test_per_sample_validity_schedules():
    """sra_set_reference_validity_batched (reading A12; "validity masks are precomputed per-rank"): each
    batch item gets the schedule of its own compacted reference - mapped back through its compaction it covers exactly
    the oracle's mask under that item's flags; useful FLOPs are the sum over the items; a [B, n_ref] array whose rows are
    all-true is the unmasked context again; wrong lengths never reach the C side."""
    n_gen, off = 300, [0, 77, 205, 334, 339]
    rng = np.random.default_rng(5)
    valid = rng.random((3, off[-1])) < 0.6
    valid[1, :] = True            # item 1: every token valid
    valid[2, off[2]:off[3]] = False  # item 2: one block entirely invalid
    ctx = B.sra_create(3, 2, 64, n_gen, off)
    try:
        plain = B.sra_schedule_copy(ctx)
        B.sra_set_reference_validity(ctx, valid)
        total = 0.0
        for b in range(3):
            items = B.sra_batch_schedule_copy(ctx, b)
            keep = np.flatnonzero(valid[b])
            Cc = _covered_pairs(items, n_gen, len(keep))
            M = sra_oracle.sra_mask(n_gen, off, valid[b]).astype(np.int32)
            idx = np.concatenate([np.arange(n_gen), n_gen + keep])
            assert np.array_equal(Cc, M[np.ix_(idx, idx)]) and M.sum() == Cc.sum(), b
            total += float(M.sum())
        assert B.sra_batch_schedule_copy(ctx, 1) == plain
        assert B.sra_useful_flops(ctx, True) == 4.0 * 64 * 2 * total
        B.sra_set_reference_validity(ctx, np.ones((3, off[-1]), dtype=bool))
        assert all(B.sra_batch_schedule_copy(ctx, b) == plain for b in range(3))
        with pytest.raises(ValueError):
            B.sra_set_reference_validity(ctx, np.ones(off[-1] - 1, dtype=bool))
        with pytest.raises(ValueError):
            B.sra_set_reference_validity(ctx, np.ones((2, off[-1]), dtype=bool))
        assert B.lib.sra_set_reference_validity_batched(ctx, valid.astype(np.uint8).tobytes(), 2) == B.SRA_ERR_INVALID_ARG
    finally:
        B.sra_destroy(ctx)

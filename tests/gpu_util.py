"""Helpers for the -m gpu parity tests: run the CUDA path through the C ABI, run the oracle."""
import numpy as np
import torch

from oracle import c_oracle
from paper_2606_13872_b200 import inputs as sra_inputs


def run_gpu_forward(w, t, use_cache=True, with_ref_rows=True, want_lse=True, scale=0.0):
    """Forward of workload `w` on cuda:0 through the binding.  `t`: dict of bf16 CPU tensors."""
    from paper_2606_13872_b200 import binding as B
    dev = torch.device("cuda:0")
    g = {k: v.to(dev) for k, v in t.items() if not k.startswith("do_")}
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets, scale)
    try:
        o_gen = torch.full_like(g["q_gen"], float("nan"))
        lse_gen = torch.full((w.batch, w.heads, w.n_gen), float("nan"), device=dev) if want_lse else None
        has_ref = w.n_ref > 0
        o_ref = lse_ref = None
        if has_ref and with_ref_rows:
            o_ref = torch.full_like(g["q_ref"], float("nan"))
            lse_ref = torch.full((w.batch, w.heads, w.n_ref), float("nan"), device=dev) if want_lse else None
        if has_ref and use_cache:
            B.sra_cache_reference_kv(ctx, g["k_ref"], g["v_ref"])
        B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen,
                      q_ref=g["q_ref"] if (has_ref and with_ref_rows) else None,
                      k_ref=None if (use_cache or not has_ref) else g["k_ref"],
                      v_ref=None if (use_cache or not has_ref) else g["v_ref"],
                      o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref)
        torch.cuda.synchronize()
        out = {"o_gen": o_gen.float().cpu().numpy(), "launches": B.sra_launch_count(ctx)}
        if lse_gen is not None:
            out["lse_gen"] = lse_gen.cpu().numpy()
        if o_ref is not None:
            out["o_ref"] = o_ref.float().cpu().numpy()
            if lse_ref is not None:
                out["lse_ref"] = lse_ref.cpu().numpy()
        return out
    finally:
        B.sra_destroy(ctx)


def bits(t):
    return {k: sra_inputs.bf16_bits(v) for k, v in t.items()}


def oracle_forward_rows(w, tb, rows, scale):
    """fp64 oracle on the listed global rows ([G ; R] indexing): o [B, n_rows, H, d], lse [B, H, n_rows]."""
    kr = tb["k_ref"] if w.n_ref > 0 else None
    vr = tb["v_ref"] if w.n_ref > 0 else None
    qr = tb["q_ref"] if w.n_ref > 0 else None
    return c_oracle.forward_rows(tb["q_gen"], tb["k_gen"], tb["v_gen"], qr, kr, vr, w.ref_block_offsets, scale,
                                 np.asarray(rows, dtype=np.int32))


def gather_rows(out, w, rows):
    """Rows of the GPU result in the oracle's [G ; R] global-row order."""
    rows = np.asarray(rows)
    g = rows[rows < w.n_gen]
    r = rows[rows >= w.n_gen] - w.n_gen
    o = [out["o_gen"][:, g]]
    l = [out["lse_gen"][:, :, g]] if "lse_gen" in out else []
    if len(r):
        o.append(out["o_ref"][:, r])
        if "lse_ref" in out:
            l.append(out["lse_ref"][:, :, r])
    return np.concatenate(o, axis=1), (np.concatenate(l, axis=2) if l else None)


def boundary_rows(w, n_random=32, seed=0):
    """Rows that stress tile/block boundaries (SURVEY.md 8d CPU-baseline tier 1) + random rows."""
    rng = np.random.default_rng(seed)
    rows = set()
    Ng = w.n_gen
    for r in (0, 1, 127, 128, 129, 255, 256, 257, Ng - 129, Ng - 128, Ng - 2, Ng - 1):
        if 0 <= r < Ng:
            rows.add(r)
    off = w.ref_block_offsets
    nb = len(off) - 1
    for j in sorted({0, nb // 2, nb - 1} if nb else set()):
        s, e = off[j], off[j + 1]
        for r in (s, s + 1, s + 127, s + 128, s + 255, s + 256, e - 129, e - 128, e - 2, e - 1):
            if s <= r < e:
                rows.add(Ng + r)
    n = Ng + w.n_ref
    rows.update(int(x) for x in rng.integers(0, n, size=n_random))
    return np.array(sorted(rows), dtype=np.int32)

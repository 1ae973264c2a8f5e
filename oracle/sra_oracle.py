"""CPU fp64 oracle for Sparse Reference Attention (SRA).   *** TEST INFRASTRUCTURE ***

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It shares no code with the CUDA path and never imports the
product package.

What it computes ("Generation tokens attend to all reference tokens ...
while reference tokens only self-attend"; :119 structured sparsity, near-linear in
reference length; :223 cached reference K/V concatenated with fresh generation K/V;
:561 restatement).  The paper gives no equation; the mask below is SURVEY.md section 8c's
reading (A1-A5, listed in DESIGN.md):

    rows/cols ordered [G ; R], n = N_g + N_r, block(t) = k with off[k] <= t < off[k+1]
    M[i][j] = 1  if i in G                                  (any j in G u R)
    M[i][j] = 1  if i in R, j in R and block(i) == block(j)
    M[i][j] = 0  otherwise  (R->G masked; R->other R blocks masked)
    S = s * Q K^T;  P = softmax over {j : M[i][j]=1} of S;  O = P V;  LSE = max + log(sum)
    backward (standard softmax-attention calculus, paper silent):
    D = rowsum(dO o O); dV = P^T dO; dP = dO V^T; dS = P o (dP - D); dQ = s dS K; dK = s dS^T Q

Sparse validity masking ("skip invalid reference tokens"; SURVEY.md section 8c reading A8,
section 8f #1): with an optional per-reference-token flag valid[t],
    M[i][j] = 0 if j in R and not valid[j]     (an invalid token is nobody's key)
    M[i][:] = 0 if i in R and not valid[i]     (an invalid token's own row is empty)
    a row with no visible key has O = 0, P = 0, LSE = -inf (the convention of reading A8).
Per-sample masks (reading A12; "validity masks are precomputed per-rank"): `valid` of shape
[B, n_ref] gives batch item b its own mask valid[b] - each item is the problem above with its own flags.

Sparse temporal attention of the SR refiner ("restricts each frame's receptive field to a local
neighborhood"; no window size or mask is given - reading A17 of DESIGN.md): with generation frame offsets fr[] and a
window w (frames on each side),
    M[i][j] = 0 if i, j in G and |frame(i) - frame(j)| > w        (G -> R and the R rows are unchanged).

Producer side of the reference-KV cache ("eliminating redundant linear projections and RoPE
computations across all steps").  The paper names RoPE and gives no formula, table or pairing;
reading A18 of DESIGN.md: the RoFormer definition on interleaved pairs, angles supplied by the caller per token,
    (y[2i] + j y[2i+1]) = (x[2i] + j x[2i+1]) * (cos[t, i] + j sin[t, i]),        t = token, i < d/2,
shared by every head and batch entry; the rotated tensor is stored in bf16 (round to nearest even), the precision the
attention consumes.  `rope` below is that definition as one complex multiplication.

SRA is exact attention under a fixed mask, so the oracle is that definition written
out: the mask is materialised as an explicit n x n byte matrix, every quantity is
fp64, nothing is tiled, fused or reordered.  Inputs are bf16 bit patterns (uint16),
upcast exactly to fp64.

Pins: tests/test_oracle_pins.py (brute force, closed forms, invariants, library
cross-checks, finite differences).  No function here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np


def bf16_bits_to_f64(bits: np.ndarray) -> np.ndarray:
    """Exact upcast of bf16 bit patterns (uint16) to float64."""
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def f64_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round fp64 to bf16 (nearest, ties to even) and return the bit patterns (uint16).  Finite inputs whose magnitude
    is inside the normal bf16 range; bf16 = the top 16 bits of the fp32 encoding, so the rounding is done on the value:
    x = m * 2^e with 1 <= |m| < 2, keep 8 significant bits."""
    x = np.asarray(x, dtype=np.float64)
    m, e = np.frexp(x)                      # x = m * 2^e, 0.5 <= |m| < 1
    q = np.rint(m * 256.0)                  # 8 significant bits; np.rint rounds ties to even
    y = np.ldexp(q, e - 8)                  # exactly representable in bf16 (and so in fp32)
    return (y.astype(np.float32).view(np.uint32) >> np.uint32(16)).astype(np.uint16)


def rope(x_bits: np.ndarray, cos: np.ndarray, sin: np.ndarray) -> np.ndarray:
    """Rotary position embedding of a bf16 tensor [B, N, H, d] by per-token angles, fp64 (reading A18).

    cos, sin: [N, d/2] (the caller's table; any position scheme, e.g. the 3-D grid of a video DiT).  Element pair
    (2i, 2i+1) of every head of token t is multiplied, as a complex number, by cos[t,i] + j sin[t,i].
    Returns fp64 [B, N, H, d], unrounded; `f64_to_bf16_bits` gives what the cache stores."""
    x = bf16_bits_to_f64(x_bits)
    z = x[..., 0::2] + 1j * x[..., 1::2]
    w = np.asarray(cos, dtype=np.float64) + 1j * np.asarray(sin, dtype=np.float64)
    y = z * w[None, :, None, :]
    out = np.empty_like(x)
    out[..., 0::2] = y.real
    out[..., 1::2] = y.imag
    return out


def block_of(t: int, offsets) -> int:
    """block(t) = k with off[k] <= t < off[k+1]."""
    for k in range(len(offsets) - 1):
        if offsets[k] <= t < offsets[k + 1]:
            return k
    raise ValueError(f"token {t} outside reference blocks {offsets}")


def sra_mask(n_gen: int, ref_block_offsets, valid=None, gen_frame_offsets=None, window=-1) -> np.ndarray:
    """The explicit SRA mask M, uint8 [n, n] with n = n_gen + n_ref, rows/cols [G ; R].
    `valid` (optional, n_ref flags): invalid reference tokens lose their column and their row.
    `gen_frame_offsets`, `window` >= 0 (optional): G -> G restricted to frames within the window."""
    off = [int(x) for x in ref_block_offsets] if len(ref_block_offsets) else [0]
    n_ref = off[-1]
    n = n_gen + n_ref
    M = np.zeros((n, n), dtype=np.uint8)
    for i in range(n):
        if i < n_gen:  # i in G: sees everything
            M[i, :] = 1
        else:  # i in R: sees only its own block of R
            bi = block_of(i - n_gen, off)
            for j in range(n_gen, n):
                if block_of(j - n_gen, off) == bi:
                    M[i, j] = 1
    if gen_frame_offsets is not None and window >= 0:
        fr = [int(x) for x in gen_frame_offsets]
        for i in range(n_gen):
            fi = block_of(i, fr)
            for j in range(n_gen):
                if abs(block_of(j, fr) - fi) > window:
                    M[i, j] = 0
    if valid is not None:
        for t in range(n_ref):
            if not valid[t]:
                M[:, n_gen + t] = 0
                M[n_gen + t, :] = 0
    return M


def masked_attention(Q, K, V, M, scale):
    """softmax(scale Q K^T restricted to M) V for one head, fp64.  Returns O, LSE, P."""
    S = scale * (Q @ K.T)
    vis = M.astype(bool)
    Sm = np.where(vis, S, -np.inf)
    mx = Sm.max(axis=1, keepdims=True)
    empty = ~vis.any(axis=1, keepdims=True)  # rows with no visible key (invalid reference tokens): O = 0, LSE = -inf
    mx0 = np.where(empty, 0.0, mx)
    E = np.where(vis, np.exp(np.where(vis, S, 0.0) - mx0), 0.0)
    Z = E.sum(axis=1, keepdims=True)
    P = E / np.where(empty, 1.0, Z)
    O = P @ V
    with np.errstate(divide="ignore"):
        LSE = np.where(empty, -np.inf, mx0 + np.log(np.where(empty, 1.0, Z)))[:, 0]
    return O, LSE, P


def _concat_head(x_gen, x_ref, b, h):
    parts = [x_gen[b, :, h, :]]
    if x_ref is not None and x_ref.shape[1] > 0:
        parts.append(x_ref[b, :, h, :])
    return np.concatenate(parts, axis=0)


def _valid_of(valid, b):
    """Mask of batch item b: `valid` is None, [n_ref] (shared by the batch) or [B, n_ref] (per sample, A12)."""
    if valid is None:
        return None
    v = np.asarray(valid)
    return v[b] if v.ndim == 2 else v


def sra_forward(q_gen, k_gen, v_gen, q_ref, k_ref, v_ref, ref_block_offsets, scale, valid=None,
                gen_frame_offsets=None, window=-1):
    """SRA forward on bf16-bit inputs [B, N, H, d].

    Returns dict(o_gen, o_ref, lse_gen, lse_ref): O fp64 [B,N,H,d], LSE fp64 [B,H,N].
    q_ref may be None (cached denoising step: R rows skipped).
    """
    f = bf16_bits_to_f64
    qg, kg, vg = f(q_gen), f(k_gen), f(v_gen)
    kr, vr = f(k_ref), f(v_ref)
    B, Ng, H, d = qg.shape
    Nr = kr.shape[1]
    have_qr = q_ref is not None
    qr = f(q_ref) if have_qr else np.zeros((B, Nr, H, d))
    o = np.zeros((B, Ng + Nr, H, d))
    lse = np.zeros((B, H, Ng + Nr))
    for b in range(B):
        M = sra_mask(Ng, ref_block_offsets, _valid_of(valid, b), gen_frame_offsets, window)
        for h in range(H):
            Q = _concat_head(qg, qr, b, h)
            K = _concat_head(kg, kr, b, h)
            V = _concat_head(vg, vr, b, h)
            O, L, _ = masked_attention(Q, K, V, M, scale)
            o[b, :, h, :] = O
            lse[b, h, :] = L
    out = {"o_gen": o[:, :Ng], "lse_gen": lse[:, :, :Ng]}
    if have_qr:
        out["o_ref"] = o[:, Ng:]
        out["lse_ref"] = lse[:, :, Ng:]
    return out


def sra_backward(q_gen, k_gen, v_gen, q_ref, k_ref, v_ref, do_gen, do_ref, ref_block_offsets, scale, valid=None,
                 gen_frame_offsets=None, window=-1):
    """SRA backward on bf16-bit inputs.  Returns dq/dk/dv for G and R, fp64 [B,N,H,d]."""
    f = bf16_bits_to_f64
    qg, kg, vg, qr, kr, vr = f(q_gen), f(k_gen), f(v_gen), f(q_ref), f(k_ref), f(v_ref)
    dog, dor = f(do_gen), f(do_ref)
    B, Ng, H, d = qg.shape
    Nr = kr.shape[1]
    dq = np.zeros((B, Ng + Nr, H, d))
    dk = np.zeros_like(dq)
    dv = np.zeros_like(dq)
    for b in range(B):
        M = sra_mask(Ng, ref_block_offsets, _valid_of(valid, b), gen_frame_offsets, window)
        for h in range(H):
            Q = _concat_head(qg, qr, b, h)
            K = _concat_head(kg, kr, b, h)
            V = _concat_head(vg, vr, b, h)
            dO = _concat_head(dog, dor, b, h)
            O, _, P = masked_attention(Q, K, V, M, scale)
            D = (dO * O).sum(axis=1, keepdims=True)
            dV = P.T @ dO
            dP = dO @ V.T
            dS = P * (dP - D)
            dq[b, :, h, :] = scale * (dS @ K)
            dk[b, :, h, :] = scale * (dS.T @ Q)
            dv[b, :, h, :] = dV
    return {"dq_gen": dq[:, :Ng], "dk_gen": dk[:, :Ng], "dv_gen": dv[:, :Ng],
            "dq_ref": dq[:, Ng:], "dk_ref": dk[:, Ng:], "dv_ref": dv[:, Ng:]}


def count_pairs(n_gen: int, ref_block_offsets, valid=None) -> int:
    """Number of unmasked (query,key) pairs per (batch, head), counted from the explicit mask."""
    return int(sra_mask(n_gen, ref_block_offsets, valid).sum(dtype=np.int64))

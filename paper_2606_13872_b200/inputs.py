"""Seeded synthetic inputs for Sparse Reference Attention (SRA) workloads.

This module holds NONE of the method's arithmetic: it only names the workload
shapes of BASELINE.json `configs` and draws i.i.d. normal
tensors with a seeded CPU generator, rounded once to bf16.  Both the CUDA path
(tests, bench.py) and the CPU oracle (tests only) are fed the *same* buffers
produced here; neither side regenerates inputs itself.

Recipe (SURVEY.md section 8d "Synthetic inputs"):
    g = torch.Generator('cpu').manual_seed(seed + k [+ 1000*step for fresh G tensors])
    x = torch.randn(B, N, H, d, generator=g, dtype=torch.float32) * elem_scale
    x = x.to(torch.bfloat16)                      # RNE, once
with tensor index k in the fixed order
    q_gen, k_gen, v_gen, q_ref, k_ref, v_ref, do_gen, do_ref = 0..7.

The paper measures SRA speed on no public benchmark;
these shapes are synthetic stand-ins for its latent-frame x tokens-per-frame
grids and multi-second clean reference clips.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional, Sequence

import torch

TENSOR_ORDER = ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref", "do_gen", "do_ref")


@dataclasses.dataclass(frozen=True)
class SRAWorkload:
    """One synthetic SRA problem: shapes + reference block pattern + distribution."""

    name: str
    batch: int
    heads: int
    head_dim: int
    n_gen: int
    ref_block_sizes: tuple  # tokens per reference block (one block = one latent frame)
    dist: str = "A"  # "A": N(0,1)/sqrt(d)   "B": N(0,1)   "peaked": q,k ~ N(0, 2^2), v ~ N(0,1)
    seed: int = 0

    @property
    def n_ref(self) -> int:
        return int(sum(self.ref_block_sizes))

    @property
    def ref_block_offsets(self) -> List[int]:
        off = [0]
        for b in self.ref_block_sizes:
            off.append(off[-1] + int(b))
        return off

    def elem_scale(self, tensor: str) -> float:
        if self.dist == "A":
            return 1.0 / math.sqrt(self.head_dim)
        if self.dist == "B":
            return 1.0
        if self.dist == "peaked":
            return 2.0 if tensor[0] in "qk" else 1.0
        raise ValueError(f"unknown dist {self.dist!r}")

    def replace(self, **kw) -> "SRAWorkload":
        return dataclasses.replace(self, **kw)


def _uniform(n_blocks: int, size: int) -> tuple:
    return tuple([size] * n_blocks)


# BASELINE.json configs (index in comments).  dist per SURVEY.md section 8c reading A14.
WORKLOADS: Dict[str, SRAWorkload] = {
    # [0] Tiny: B1 H4 d64, 256 gen + 4x128 ref
    "tiny": SRAWorkload("tiny", 1, 4, 64, 256, _uniform(4, 128), "A", 0),
    # [1] 480p: 21 x 1560 gen, 14 x 1560 ref
    "480p": SRAWorkload("480p", 1, 40, 128, 21 * 1560, _uniform(14, 1560), "A", 0),
    # [2] 720p: 21 x 3600 gen, 14 x 3600 ref  (the metric's headline config)
    "720p": SRAWorkload("720p", 1, 40, 128, 21 * 3600, _uniform(14, 3600), "A", 0),
    # [3] long-reference sweep: 5/10/20/40 s of reference in 1560-token blocks
    "sweep5s": SRAWorkload("sweep5s", 1, 40, 128, 21 * 1560, _uniform(14, 1560), "A", 0),
    "sweep10s": SRAWorkload("sweep10s", 1, 40, 128, 21 * 1560, _uniform(28, 1560), "A", 0),
    "sweep20s": SRAWorkload("sweep20s", 1, 40, 128, 21 * 1560, _uniform(56, 1560), "A", 0),
    "sweep40s": SRAWorkload("sweep40s", 1, 40, 128, 21 * 1560, _uniform(112, 1560), "A", 0),
    # derived shape (SURVEY.md 8d "optional 1080p point": 68 x 120 = 8160 tokens per frame by the same 16x-per-side rule;
    # no config pins it and the paper gives no token counts) - an extra scaling point only
    "1080p": SRAWorkload("1080p", 1, 40, 128, 21 * 8160, _uniform(14, 8160), "A", 0),
    # [4] training fwd+bwd: B2, Q/K/V/dO ~ N(0,1)
    "train": SRAWorkload("train", 2, 40, 128, 21 * 1560, _uniform(14, 1560), "B", 0),
    # scaled-down, fully checkable shapes with the real boundary structure (SURVEY.md section 8d tier 3)
    "mini480": SRAWorkload("mini480", 1, 2, 128, 2 * 1560, _uniform(3, 1560), "B", 0),
    "mini720": SRAWorkload("mini720", 1, 2, 128, 3600 + 200, _uniform(2, 3600), "B", 0),
    "mini_train": SRAWorkload("mini_train", 2, 2, 128, 1560 + 300, _uniform(2, 1560), "B", 0),
    # ragged, non-uniform blocks incl. 1-token block and blocks not dividing 128
    "ragged": SRAWorkload("ragged", 2, 3, 128, 333, (1, 130, 257, 64, 200), "B", 0),
    "ragged64": SRAWorkload("ragged64", 1, 2, 64, 300, (77, 128, 129, 5), "peaked", 0),
    # cache-bound short-query cases (north_star; SURVEY.md 8d auxiliary sweep): few generation rows against the
    # 40 s reference cache (174,720 tokens, 3.58 GB of K+V); the library splits the keys across CTAs
    "short128": SRAWorkload("short128", 1, 40, 128, 128, _uniform(112, 1560), "A", 0),
    "short512": SRAWorkload("short512", 1, 40, 128, 512, _uniform(112, 1560), "A", 0),
    "short2048": SRAWorkload("short2048", 1, 40, 128, 2048, _uniform(112, 1560), "A", 0),
    # scaled-down short-query shapes whose schedules are key-split, every row checkable
    "short_mini": SRAWorkload("short_mini", 1, 2, 128, 100, (1560, 1560, 300), "B", 0),
    "short_mini64": SRAWorkload("short_mini64", 2, 2, 64, 300, (1000, 1100), "peaked", 0),
}


def make_tensor(w: SRAWorkload, tensor: str, step: int = 0, n_tokens: Optional[int] = None) -> torch.Tensor:
    """One bf16 CPU tensor [B, N, H, d] of workload `w`, by the recipe above."""
    k = TENSOR_ORDER.index(tensor)
    is_gen = tensor.endswith("_gen")
    n = n_tokens if n_tokens is not None else (w.n_gen if is_gen else w.n_ref)
    seed = w.seed + k + (1000 * step if is_gen else 0)
    g = torch.Generator("cpu").manual_seed(seed)
    x = torch.randn(w.batch, n, w.heads, w.head_dim, generator=g, dtype=torch.float32)
    scale = 1.0 if tensor.startswith("do_") else w.elem_scale(tensor)
    if scale != 1.0:
        x.mul_(scale)
    return x.to(torch.bfloat16)


def make_inputs(w: SRAWorkload, step: int = 0, with_grad: bool = False,
                names: Optional[Sequence[str]] = None) -> Dict[str, torch.Tensor]:
    """All (or `names`) bf16 CPU tensors of the workload, keyed by TENSOR_ORDER names."""
    if names is None:
        names = TENSOR_ORDER if with_grad else TENSOR_ORDER[:6]
    return {t: make_tensor(w, t, step) for t in names}


def bf16_bits(x: torch.Tensor):
    """The raw bf16 bit patterns of `x` as a numpy uint16 array (what the oracle consumes)."""
    assert x.dtype == torch.bfloat16 and x.device.type == "cpu"
    return x.contiguous().view(torch.int16).numpy().view("uint16")


def make_tensor_device(w: SRAWorkload, tensor: str, device, step: int = 0, seed_offset: int = 0,
                       n_tokens: Optional[int] = None) -> torch.Tensor:
    """Same distribution and seeding rule as `make_tensor`, drawn by the DEVICE generator (bench.py at
    full size: 720p tensors are 0.4 G elements each, too slow to draw on the host every run).  The byte
    values differ from the CPU recipe; anything checked against the oracle copies these buffers back."""
    k = TENSOR_ORDER.index(tensor)
    is_gen = tensor.endswith("_gen")
    n = n_tokens if n_tokens is not None else (w.n_gen if is_gen else w.n_ref)
    seed = w.seed + seed_offset + k + (1000 * step if is_gen else 0)
    g = torch.Generator(device).manual_seed(seed)
    x = torch.randn(w.batch, n, w.heads, w.head_dim, generator=g, dtype=torch.float32, device=device)
    scale = 1.0 if tensor.startswith("do_") else w.elem_scale(tensor)
    if scale != 1.0:
        x.mul_(scale)
    return x.to(torch.bfloat16)


# ----------------------------------------------------------------------------- RoPE angle tables (inputs of 8f #3)
_GRID_WIDTH = {1560: 52, 3600: 80, 8160: 120}  # tokens per latent frame -> tokens per row (30x52, 45x80, 68x120)


def rope_tables(w: SRAWorkload, which: str, base: float = 10000.0):
    """(cos, sin) fp32 CPU tensors [n, d/2] for the `which` in {"gen", "ref"} tokens of workload `w`.

    An INPUT of the path (include/sra.h takes the table from the caller), drawn up here so that both sides rotate by
    the same numbers.  Recipe (synthetic; the paper names RoPE and gives no scheme - stands in for the 3-D table of a
    video DiT): token t sits at (frame, row, column) of a latent grid; the d/2 pairs are split into three groups
    (d/2 - 2*(d/2 // 3) temporal, d/2 // 3 rows, d/2 // 3 columns); pair j of a group of size m turns by
    position * base^(-j/m).  Generation tokens: frame = t // P, P = n_gen / 21 when that is one of the paper's grids
    (width from _GRID_WIDTH), else P = 64 with width 8.  Reference tokens: frame = -(block index + 1) (reference frames
    sit before the clip), row / column from the index inside the block with the same width rule.
    Angles are formed in fp64 and the cosines / sines rounded once to fp32."""
    half = w.head_dim // 2
    m_hw = half // 3
    m_t = half - 2 * m_hw
    if which == "gen":
        n = w.n_gen
        per = n // 21 if n % 21 == 0 and (n // 21) in _GRID_WIDTH else 64
        width = _GRID_WIDTH.get(per, 8)
        t = torch.arange(n, dtype=torch.int64)
        frame, inner = t // per, t % per
    elif which == "ref":
        n = w.n_ref
        frame = torch.empty(n, dtype=torch.int64)
        inner = torch.empty(n, dtype=torch.int64)
        off = w.ref_block_offsets
        width = 8
        for k, size in enumerate(w.ref_block_sizes):
            frame[off[k]:off[k + 1]] = -(k + 1)
            inner[off[k]:off[k + 1]] = torch.arange(size, dtype=torch.int64)
            width = _GRID_WIDTH.get(int(size), width)
    else:
        raise ValueError(which)
    pos = (frame.double(), (inner // width).double(), (inner % width).double())
    cols = []
    for p, m in zip(pos, (m_t, m_hw, m_hw)):
        freq = base ** (-torch.arange(m, dtype=torch.float64) / max(m, 1))
        cols.append(p[:, None] * freq[None, :])
    ang = torch.cat(cols, dim=1) if n else torch.zeros(0, half, dtype=torch.float64)
    return torch.cos(ang).float().contiguous(), torch.sin(ang).float().contiguous()

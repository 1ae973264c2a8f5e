"""Thin ctypes binding of the C-ABI library declared in include/sra.h.

Argument marshalling only: every step of the SRA path (reference-KV cache build, forward,
backward) runs in the CUDA kernels of libsra_b200.so.  PyTorch is used for device memory and
streams (`tensor.data_ptr()`, `torch.cuda.current_stream().cuda_stream`).  There is no CPU or
PyTorch fallback: if the library is missing, importing this module raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsra_b200.so")

SRA_OK = 0
SRA_ERR_INVALID_ARG = -1
SRA_ERR_UNSUPPORTED = -2
SRA_ERR_CUDA = -3
SRA_ERR_NO_REF_CACHE = -4
SRA_ERR_OOM = -5

EXPORTS = (
    "sra_create", "sra_cache_reference_kv", "sra_cache_reference_kv_rope", "sra_apply_rope", "sra_forward", "sra_forward_host", "sra_backward", "sra_destroy", "sra_useful_flops",
    "sra_schedule_info", "sra_schedule_copy", "sra_cache_bytes", "sra_launch_count", "sra_status_string",
    "sra_last_error", "sra_set_kernel_timing", "sra_kernel_time_ms", "sra_split_schedule_copy", "sra_set_reference_validity", "sra_set_temporal_window",
    "sra_reserve", "sra_set_reference_validity_batched", "sra_batch_schedule_copy", "sra_pair_schedule_copy", "sra_bound_ends_copy",
    "sra_forward_gen_static", "sra_static_scratch_bytes", "sra_static_last_error",
)
STATIC_SCRATCH_BYTES = 32 << 20

RESERVE_BACKWARD, RESERVE_HOST, RESERVE_VALIDITY = 1, 2, 4

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} not found: build it with `python -m paper_2606_13872_b200.build` "
        "(the SRA path has no CPU fallback)")

lib = ctypes.CDLL(LIB_PATH)


class sra_config(ctypes.Structure):
    _fields_ = [
        ("batch", ctypes.c_int32), ("heads", ctypes.c_int32), ("head_dim", ctypes.c_int32),
        ("n_gen", ctypes.c_int32), ("n_ref", ctypes.c_int32), ("n_ref_blocks", ctypes.c_int32),
        ("ref_block_offsets", ctypes.POINTER(ctypes.c_int32)),
        ("softmax_scale", ctypes.c_float), ("device", ctypes.c_int32),
    ]


class sra_fwd_args(ctypes.Structure):
    _fields_ = [(n, ctypes.c_void_p) for n in
                ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref", "o_gen", "o_ref", "lse_gen", "lse_ref")]


class sra_fwd_host_args(ctypes.Structure):
    _fields_ = [(n, ctypes.c_void_p) for n in
                ("q_gen", "k_gen", "v_gen", "q_ref", "o_gen", "o_ref", "lse_gen", "lse_ref")]


class sra_bwd_args(ctypes.Structure):
    _fields_ = [(n, ctypes.c_void_p) for n in
                ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref", "o_gen", "o_ref", "lse_gen", "lse_ref",
                 "do_gen", "do_ref", "dq_gen", "dk_gen", "dv_gen", "dq_ref", "dk_ref", "dv_ref")]


class sra_static_fwd_args(ctypes.Structure):
    _fields_ = [("batch", ctypes.c_int32), ("heads", ctypes.c_int32), ("head_dim", ctypes.c_int32), ("n_gen", ctypes.c_int32),
                ("n_ref", ctypes.c_int32), ("softmax_scale", ctypes.c_float), ("device", ctypes.c_int32),
                ("n_split", ctypes.c_int32), ("q_gen", ctypes.c_void_p), ("k_gen", ctypes.c_void_p), ("v_gen", ctypes.c_void_p),
                ("k_ref", ctypes.c_void_p), ("v_ref", ctypes.c_void_p), ("o_gen", ctypes.c_void_p), ("lse_gen", ctypes.c_void_p)]


_ctx_p = ctypes.c_void_p
lib.sra_forward_gen_static.argtypes = [ctypes.POINTER(sra_static_fwd_args), ctypes.c_void_p]
lib.sra_forward_gen_static.restype = ctypes.c_int
lib.sra_static_scratch_bytes.argtypes = [ctypes.POINTER(sra_static_fwd_args), ctypes.c_int32, ctypes.POINTER(ctypes.c_int64)]
lib.sra_static_scratch_bytes.restype = ctypes.c_int
lib.sra_static_last_error.argtypes = []
lib.sra_static_last_error.restype = ctypes.c_char_p
lib.sra_create.argtypes = [ctypes.POINTER(sra_config), ctypes.POINTER(_ctx_p)]
lib.sra_create.restype = ctypes.c_int
lib.sra_cache_reference_kv.argtypes = [_ctx_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
lib.sra_cache_reference_kv.restype = ctypes.c_int
lib.sra_cache_reference_kv_rope.argtypes = [_ctx_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                            ctypes.c_void_p]
lib.sra_cache_reference_kv_rope.restype = ctypes.c_int
lib.sra_apply_rope.argtypes = [_ctx_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32,
                               ctypes.c_void_p]
lib.sra_apply_rope.restype = ctypes.c_int
lib.sra_forward.argtypes = [_ctx_p, ctypes.POINTER(sra_fwd_args), ctypes.c_void_p]
lib.sra_forward.restype = ctypes.c_int
lib.sra_forward_host.argtypes = [_ctx_p, ctypes.POINTER(sra_fwd_host_args), ctypes.c_void_p]
lib.sra_forward_host.restype = ctypes.c_int
lib.sra_backward.argtypes = [_ctx_p, ctypes.POINTER(sra_bwd_args), ctypes.c_void_p]
lib.sra_backward.restype = ctypes.c_int
lib.sra_destroy.argtypes = [_ctx_p]
lib.sra_destroy.restype = None
lib.sra_useful_flops.argtypes = [_ctx_p, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
lib.sra_useful_flops.restype = ctypes.c_int
lib.sra_schedule_info.argtypes = [_ctx_p, ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32),
                                  ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int64)]
lib.sra_schedule_info.restype = ctypes.c_int
lib.sra_set_reference_validity.argtypes = [_ctx_p, ctypes.c_char_p]
lib.sra_set_reference_validity.restype = ctypes.c_int
lib.sra_set_reference_validity_batched.argtypes = [_ctx_p, ctypes.c_char_p, ctypes.c_int32]
lib.sra_set_reference_validity_batched.restype = ctypes.c_int
lib.sra_reserve.argtypes = [_ctx_p, ctypes.c_uint32]
lib.sra_reserve.restype = ctypes.c_int
lib.sra_batch_schedule_copy.argtypes = [_ctx_p, ctypes.c_int32, ctypes.POINTER(ctypes.c_int32), ctypes.c_int32,
                                        ctypes.POINTER(ctypes.c_int32)]
lib.sra_batch_schedule_copy.restype = ctypes.c_int
lib.sra_pair_schedule_copy.argtypes = [_ctx_p, ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32), ctypes.c_int32,
                                       ctypes.POINTER(ctypes.c_int32)]
lib.sra_pair_schedule_copy.restype = ctypes.c_int
lib.sra_bound_ends_copy.argtypes = [_ctx_p, ctypes.POINTER(ctypes.c_int32), ctypes.c_int32, ctypes.POINTER(ctypes.c_int32),
                                    ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32)]
lib.sra_bound_ends_copy.restype = ctypes.c_int
lib.sra_set_temporal_window.argtypes = [_ctx_p, ctypes.c_int32, ctypes.POINTER(ctypes.c_int32), ctypes.c_int32]
lib.sra_set_temporal_window.restype = ctypes.c_int
lib.sra_split_schedule_copy.argtypes = [_ctx_p, ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32), ctypes.c_int32,
                                        ctypes.POINTER(ctypes.c_int32)]
lib.sra_split_schedule_copy.restype = ctypes.c_int
lib.sra_schedule_copy.argtypes = [_ctx_p, ctypes.POINTER(ctypes.c_int32), ctypes.c_int32,
                                  ctypes.POINTER(ctypes.c_int32)]
lib.sra_schedule_copy.restype = ctypes.c_int
lib.sra_cache_bytes.argtypes = [_ctx_p]
lib.sra_cache_bytes.restype = ctypes.c_int64
lib.sra_launch_count.argtypes = [_ctx_p]
lib.sra_launch_count.restype = ctypes.c_int64
lib.sra_set_kernel_timing.argtypes = [_ctx_p, ctypes.c_int]
lib.sra_set_kernel_timing.restype = ctypes.c_int
lib.sra_kernel_time_ms.argtypes = [_ctx_p, ctypes.c_int, ctypes.POINTER(ctypes.c_float)]
lib.sra_kernel_time_ms.restype = ctypes.c_int
lib.sra_status_string.argtypes = [ctypes.c_int]
lib.sra_status_string.restype = ctypes.c_char_p
lib.sra_last_error.argtypes = [_ctx_p]
lib.sra_last_error.restype = ctypes.c_char_p


class SRAError(RuntimeError):
    def __init__(self, status: int, detail: str = ""):
        self.status = status
        name = lib.sra_status_string(status).decode()
        super().__init__(f"{name} ({status}){': ' + detail if detail else ''}")


def _check(status: int, ctx=None):
    if status != SRA_OK:
        detail = lib.sra_last_error(ctx).decode() if ctx else ""
        raise SRAError(status, detail)


def _ptr(t) -> Optional[int]:
    """Device pointer of a torch tensor (or None).  The tensor must be contiguous."""
    if t is None:
        return None
    if not t.is_contiguous():
        raise ValueError("SRA tensors must be contiguous [B, N, H, d]")
    return t.data_ptr()


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream or None
    if isinstance(stream, int):
        return stream or None
    return stream.cuda_stream or None


# ----------------------------------------------------------------------------- same-name wrappers
def sra_create(batch: int, heads: int, head_dim: int, n_gen: int, ref_block_offsets: Sequence[int],
               softmax_scale: float = 0.0, device: int = -1) -> int:
    """sra_create (include/sra.h).  Returns the opaque ctx handle (int)."""
    off = [int(x) for x in ref_block_offsets] if len(ref_block_offsets) else [0]
    n_blocks = len(off) - 1
    arr = (ctypes.c_int32 * len(off))(*off)
    cfg = sra_config(batch, heads, head_dim, n_gen, off[-1], n_blocks,
                     arr if n_blocks > 0 else None, float(softmax_scale), device)
    ctx = _ctx_p()
    _check(lib.sra_create(ctypes.byref(cfg), ctypes.byref(ctx)))
    _SHAPES[ctx.value] = (int(batch), int(off[-1]))
    return ctx.value


_SHAPES = {}  # ctx handle -> (batch, n_ref): the binding checks host buffer lengths before they cross the boundary


def sra_destroy(ctx: Optional[int]) -> None:
    _SHAPES.pop(ctx, None)
    lib.sra_destroy(ctx)


def sra_reserve(ctx: int, what: int) -> None:
    """sra_reserve (include/sra.h): one-time allocation of the optional paths (RESERVE_BACKWARD | RESERVE_HOST |
    RESERVE_VALIDITY), so that no later call allocates."""
    _check(lib.sra_reserve(ctx, int(what)), ctx)


def sra_cache_reference_kv(ctx: int, k_ref, v_ref, stream=None) -> None:
    _check(lib.sra_cache_reference_kv(ctx, _ptr(k_ref), _ptr(v_ref), _stream(stream)), ctx)


def sra_cache_reference_kv_rope(ctx: int, k_ref, v_ref, cos_ref, sin_ref, stream=None) -> None:
    """k_ref pre-RoPE; cos_ref / sin_ref fp32 device tensors [n_ref, d/2] (include/sra.h)."""
    _check(lib.sra_cache_reference_kv_rope(ctx, _ptr(k_ref), _ptr(v_ref), _ptr(cos_ref), _ptr(sin_ref), _stream(stream)), ctx)


def sra_apply_rope(ctx: int, x0, x1, cos, sin, n_tokens: int, stream=None) -> None:
    """In-place rotation of x0 (and x1 unless None), bf16 device tensors [B, n_tokens, H, d]."""
    _check(lib.sra_apply_rope(ctx, _ptr(x0), _ptr(x1), _ptr(cos), _ptr(sin), int(n_tokens), _stream(stream)), ctx)


def sra_forward(ctx: int, q_gen, k_gen, v_gen, o_gen, q_ref=None, k_ref=None, v_ref=None, o_ref=None,
                lse_gen=None, lse_ref=None, stream=None) -> None:
    a = sra_fwd_args(_ptr(q_gen), _ptr(k_gen), _ptr(v_gen), _ptr(q_ref), _ptr(k_ref), _ptr(v_ref),
                     _ptr(o_gen), _ptr(o_ref), _ptr(lse_gen), _ptr(lse_ref))
    _check(lib.sra_forward(ctx, ctypes.byref(a), _stream(stream)), ctx)


def _static_args(q_gen, k_gen, v_gen, o_gen, k_ref, v_ref, lse_gen, n_split, softmax_scale, device):
    bsz, n_gen, heads, d = q_gen.shape
    n_ref = 0 if k_ref is None else k_ref.shape[1]
    return sra_static_fwd_args(bsz, heads, d, n_gen, n_ref, float(softmax_scale), int(device), int(n_split), _ptr(q_gen),
                               _ptr(k_gen), _ptr(v_gen), _ptr(k_ref), _ptr(v_ref), _ptr(o_gen), _ptr(lse_gen))


def sra_forward_gen_static(q_gen, k_gen, v_gen, o_gen, k_ref=None, v_ref=None, lse_gen=None, n_split: int = 0,
                           softmax_scale: float = 0.0, device: int = -1, stream=None) -> None:
    """sra_forward_gen_static (include/sra.h): the generation rows' attention with no context and no allocation - its
    scratch is the library's static device array (STATIC_SCRATCH_BYTES); calls that overlap on the GPU race on it."""
    a = _static_args(q_gen, k_gen, v_gen, o_gen, k_ref, v_ref, lse_gen, n_split, softmax_scale, device)
    status = lib.sra_forward_gen_static(ctypes.byref(a), _stream(stream))
    if status != SRA_OK:
        raise SRAError(status, lib.sra_static_last_error().decode())


def sra_static_scratch_bytes(batch: int, heads: int, head_dim: int, n_gen: int, n_split: int) -> int:
    a = sra_static_fwd_args(batch, heads, head_dim, n_gen, 0, 0.0, -1, n_split)
    out = ctypes.c_int64(0)
    _check(lib.sra_static_scratch_bytes(ctypes.byref(a), n_split, ctypes.byref(out)))
    return out.value


def _host_ptr(t) -> Optional[int]:
    """Host pointer of a CPU torch tensor (or None).  Must be contiguous; pin it for async copies."""
    if t is None:
        return None
    if t.device.type != "cpu" or not t.is_contiguous():
        raise ValueError("sra_forward_host takes contiguous CPU tensors")
    return t.data_ptr()


def sra_forward_host(ctx: int, q_gen, k_gen, v_gen, o_gen, q_ref=None, o_ref=None, lse_gen=None, lse_ref=None,
                     stream=None) -> None:
    """sra_forward_host (include/sra.h): HOST tensors in/out, reference K/V from the resident cache."""
    a = sra_fwd_host_args(*[_host_ptr(t) for t in (q_gen, k_gen, v_gen, q_ref, o_gen, o_ref, lse_gen, lse_ref)])
    _check(lib.sra_forward_host(ctx, ctypes.byref(a), _stream(stream)), ctx)


def sra_backward(ctx: int, *, q_gen, k_gen, v_gen, q_ref, k_ref, v_ref, o_gen, o_ref, lse_gen, lse_ref,
                 do_gen, do_ref, dq_gen, dk_gen, dv_gen, dq_ref, dk_ref, dv_ref, stream=None) -> None:
    a = sra_bwd_args(*[_ptr(t) for t in (q_gen, k_gen, v_gen, q_ref, k_ref, v_ref, o_gen, o_ref, lse_gen, lse_ref,
                                         do_gen, do_ref, dq_gen, dk_gen, dv_gen, dq_ref, dk_ref, dv_ref)])
    _check(lib.sra_backward(ctx, ctypes.byref(a), _stream(stream)), ctx)


def sra_useful_flops(ctx: int, include_ref_rows: bool, backward: bool = False) -> float:
    out = ctypes.c_double()
    _check(lib.sra_useful_flops(ctx, int(include_ref_rows), int(backward), ctypes.byref(out)), ctx)
    return out.value


def sra_schedule_info(ctx: int):
    a, b = ctypes.c_int32(), ctypes.c_int32()
    c, d = ctypes.c_int64(), ctypes.c_int64()
    _check(lib.sra_schedule_info(ctx, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c), ctypes.byref(d)), ctx)
    return {"n_gen_items": a.value, "n_ref_items": b.value, "key_tiles_gen": c.value, "key_tiles_ref": d.value}


def sra_schedule_copy(ctx: int):
    """The forward work items as a list of dicts (host logic only; no GPU needed)."""
    n = ctypes.c_int32()
    _check(lib.sra_schedule_copy(ctx, None, 0, ctypes.byref(n)), ctx)
    buf = (ctypes.c_int32 * (8 * max(n.value, 1)))()
    _check(lib.sra_schedule_copy(ctx, buf, n.value, ctypes.byref(n)), ctx)
    keys = ("q_is_ref", "q_row0", "q_rows", "seg0_is_ref", "seg0_start", "seg0_len", "seg1_start", "seg1_len")
    return [dict(zip(keys, buf[8 * i:8 * i + 8])) for i in range(n.value)]


def sra_split_schedule_copy(ctx: int):
    """(n_split, launched work items).  n_split == 1: the plain schedule; otherwise every generation slab appears
    n_split times with disjoint key ranges (`split` = index + 1), followed by the reference items."""
    ns, n = ctypes.c_int32(), ctypes.c_int32()
    _check(lib.sra_split_schedule_copy(ctx, ctypes.byref(ns), None, 0, ctypes.byref(n)), ctx)
    buf = (ctypes.c_int32 * (8 * max(n.value, 1)))()
    _check(lib.sra_split_schedule_copy(ctx, ctypes.byref(ns), buf, n.value, ctypes.byref(n)), ctx)
    keys = ("q_is_ref", "q_row0", "q_rows", "seg0_is_ref", "seg0_start", "seg0_len", "seg1_start", "seg1_len")
    items = []
    for i in range(n.value):
        it = dict(zip(keys, buf[8 * i:8 * i + 8]))
        it["split"] = it["q_is_ref"] >> 8
        it["q_is_ref"] &= 1
        items.append(it)
    return ns.value, items


def sra_set_temporal_window(ctx: int, gen_frame_offsets, window: int) -> None:
    """sra_set_temporal_window (include/sra.h).  window < 0 (or gen_frame_offsets None) turns the window off."""
    if gen_frame_offsets is None or window < 0:
        _check(lib.sra_set_temporal_window(ctx, 0, None, -1), ctx)
        return
    off = [int(x) for x in gen_frame_offsets]
    arr = (ctypes.c_int32 * len(off))(*off)
    _check(lib.sra_set_temporal_window(ctx, len(off) - 1, arr, int(window)), ctx)


def _items(buf, n):
    keys = ("q_is_ref", "q_row0", "q_rows", "seg0_is_ref", "seg0_start", "seg0_len", "seg1_start", "seg1_len")
    return [dict(zip(keys, buf[8 * i:8 * i + 8])) for i in range(n)]


def sra_batch_schedule_copy(ctx: int, batch_item: int):
    """The forward work items of one batch item (they differ between items only under per-sample validity masks)."""
    n = ctypes.c_int32()
    _check(lib.sra_batch_schedule_copy(ctx, int(batch_item), None, 0, ctypes.byref(n)), ctx)
    buf = (ctypes.c_int32 * (8 * max(n.value, 1)))()
    _check(lib.sra_batch_schedule_copy(ctx, int(batch_item), buf, n.value, ctypes.byref(n)), ctx)
    return _items(buf, n.value)


def sra_bound_ends_copy(ctx: int):
    """(generation-row ends, [per-mask reference-row ends]) that fall inside a tensor (include/sra.h)."""
    ng, rs, n = ctypes.c_int32(0), ctypes.c_int32(0), ctypes.c_int32(0)
    _check(lib.sra_bound_ends_copy(ctx, None, 0, ctypes.byref(ng), ctypes.byref(rs), ctypes.byref(n)), ctx)
    buf = (ctypes.c_int32 * max(n.value, 1))()
    _check(lib.sra_bound_ends_copy(ctx, buf, n.value, ctypes.byref(ng), ctypes.byref(rs), ctypes.byref(n)), ctx)
    vals = list(buf[:n.value])
    gen = vals[:ng.value]
    n_masks = (n.value - ng.value) // rs.value if rs.value else 0
    pad = 2 ** 31 - 1
    ref = [[v for v in vals[ng.value + m * rs.value: ng.value + (m + 1) * rs.value] if v != pad] for m in range(n_masks)]
    return gen, ref


def sra_pair_schedule_copy(ctx: int):
    """(use_pairs, pair items): the launch list of the CTA-pair forward kernel (items of up to 512 rows)."""
    up, n = ctypes.c_int32(), ctypes.c_int32()
    _check(lib.sra_pair_schedule_copy(ctx, ctypes.byref(up), None, 0, ctypes.byref(n)), ctx)
    buf = (ctypes.c_int32 * (8 * max(n.value, 1)))()
    _check(lib.sra_pair_schedule_copy(ctx, ctypes.byref(up), buf, n.value, ctypes.byref(n)), ctx)
    return bool(up.value), _items(buf, n.value)


def sra_set_reference_validity(ctx: int, valid) -> None:
    """sra_set_reference_validity[_batched] (include/sra.h): `valid` = None (every token valid), a sequence / array of
    n_ref truthy values (one mask for the batch) or a [batch, n_ref] array (one mask per batch item, reading A12).
    The length is checked here: the C side reads exactly n_masks * n_ref bytes."""
    if valid is None:
        _check(lib.sra_set_reference_validity(ctx, None), ctx)
        return
    import numpy as np
    v = np.ascontiguousarray(np.asarray(valid) != 0, dtype=np.uint8)
    batch, n_ref = _SHAPES.get(ctx, (None, None))
    if v.ndim == 1:
        if n_ref is not None and v.shape[0] != n_ref:
            raise ValueError(f"valid has {v.shape[0]} entries, the context has n_ref = {n_ref}")
        _check(lib.sra_set_reference_validity(ctx, v.tobytes()), ctx)
        return
    if v.ndim != 2 or (n_ref is not None and v.shape != (batch, n_ref)):
        raise ValueError(f"valid must be [n_ref] or [batch, n_ref] = [{batch}, {n_ref}], got {v.shape}")
    _check(lib.sra_set_reference_validity_batched(ctx, v.tobytes(), int(v.shape[0])), ctx)


def sra_cache_bytes(ctx: int) -> int:
    return int(lib.sra_cache_bytes(ctx))


KERNEL_CACHE_RELAYOUT, KERNEL_FWD, KERNEL_BWD_PREPROCESS, KERNEL_BWD_MAIN, KERNEL_BWD_DQ_FINALIZE, KERNEL_FWD_MERGE, KERNEL_ROPE = range(7)


def sra_set_kernel_timing(ctx: int, enable: bool) -> None:
    _check(lib.sra_set_kernel_timing(ctx, int(enable)), ctx)


def sra_kernel_time_ms(ctx: int, which: int) -> float:
    ms = ctypes.c_float()
    _check(lib.sra_kernel_time_ms(ctx, int(which), ctypes.byref(ms)), ctx)
    return ms.value


def sra_launch_count(ctx: int) -> int:
    return int(lib.sra_launch_count(ctx))


def sra_last_error(ctx: int) -> str:
    return lib.sra_last_error(ctx).decode()

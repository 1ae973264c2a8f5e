"""ctypes loader for oracle/sra_oracle.c (plain C fp64 oracle).   *** TEST INFRASTRUCTURE ***

Builds liboracle_sra.so with gcc on first use (`build()`), then exposes numpy-level wrappers.
Shares nothing with the CUDA path; see sra_oracle.c for the definition it follows
(SURVEY.md section 8c).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sra_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_sra.so")
_lib = None

_u8p = ctypes.POINTER(ctypes.c_uint8)
_u16p = ctypes.POINTER(ctypes.c_uint16)
_i32p = ctypes.POINTER(ctypes.c_int32)
_f64p = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    """Compile the C oracle (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.sra_oracle_count_pairs.restype = ctypes.c_longlong
        _lib.sra_oracle_count_pairs_ex.restype = ctypes.c_longlong
    return _lib


def _u16(x):
    if x is None:
        return None, None
    a = np.ascontiguousarray(x, dtype=np.uint16)
    return a, a.ctypes.data_as(_u16p)


def _i32(x):
    a = np.ascontiguousarray(x, dtype=np.int32)
    return a, a.ctypes.data_as(_i32p)


def _mask_args(valid, gen_frame_offsets, window, B, Nr):
    """(keepalive, valid*, valid_batch_stride, fr*, n_frames, window) for the *_ex entry points.
    valid: None, [Nr] (one mask for the batch) or [B, Nr] (one per batch item); window < 0 = no temporal window."""
    keep = []
    vp, stride = None, 0
    if valid is not None:
        v = np.ascontiguousarray(np.asarray(valid) != 0, dtype=np.uint8)
        assert v.shape in ((Nr,), (B, Nr)), f"valid must be [n_ref] or [B, n_ref], got {v.shape}"
        stride = Nr if v.ndim == 2 else 0
        keep.append(v)
        vp = v.ctypes.data_as(_u8p)
    fp, n_fr = None, 0
    if gen_frame_offsets is not None and window >= 0:
        fr, fp = _i32(gen_frame_offsets)
        keep.append(fr)
        n_fr = len(fr) - 1
    else:
        window = -1
    return keep, vp, stride, fp, n_fr, int(window)


def num_threads() -> int:
    return int(_load().sra_oracle_num_threads())


def count_pairs(n_gen, ref_block_offsets, valid=None, gen_frame_offsets=None, window=-1) -> int:
    off, offp = _i32(ref_block_offsets if len(ref_block_offsets) else [0])
    keep, vp, _, fp, n_fr, w = _mask_args(valid, gen_frame_offsets, window, 1, int(off[-1]))
    return int(_load().sra_oracle_count_pairs_ex(int(n_gen), int(off[-1]), offp, len(off) - 1, vp, fp, n_fr, w))


def _shape_args(k_gen, k_ref, ref_block_offsets, n_gen=None):
    B, Ng, H, d = k_gen.shape
    Nr = 0 if k_ref is None else k_ref.shape[1]
    off, offp = _i32(ref_block_offsets if len(ref_block_offsets) else [0])
    assert off[-1] == Nr and off[0] == 0
    return (B, H, d, Ng, Nr), off, offp


def forward_rows(q_gen, k_gen, v_gen, q_ref, k_ref, v_ref, ref_block_offsets, scale, rows, valid=None,
                 gen_frame_offsets=None, window=-1):
    """Rows (global indices, G first then R) for all batches/heads.
    Returns o [B, n_rows, H, d] fp64, lse [B, H, n_rows] fp64.
    valid ([n_ref] or [B, n_ref]) / gen_frame_offsets + window: the optional mask restrictions of sra_oracle.c."""
    (B, H, d, Ng, Nr), off, offp = _shape_args(k_gen, k_ref, ref_block_offsets)
    keep = [_u16(x) for x in (q_gen, k_gen, v_gen, q_ref, k_ref, v_ref)]
    rows_a, rows_p = _i32(rows)
    o = np.zeros((B, len(rows_a), H, d), dtype=np.float64)
    lse = np.zeros((B, H, len(rows_a)), dtype=np.float64)
    mk, vp, vstride, fp, n_fr, w = _mask_args(valid, gen_frame_offsets, window, B, Nr)
    rc = _load().sra_oracle_forward_rows_ex(*[k[1] for k in keep], B, H, d, Ng, Nr, offp, len(off) - 1,
                                            ctypes.c_double(scale), rows_p, len(rows_a), vp, vstride, fp, n_fr, w,
                                            o.ctypes.data_as(_f64p), lse.ctypes.data_as(_f64p))
    if rc != 0:
        raise RuntimeError(f"sra_oracle_forward_rows failed: {rc}")
    return o, lse


def forward_head(q_gen, k_gen, v_gen, q_ref, k_ref, v_ref, ref_block_offsets, scale, b, h, valid=None,
                 gen_frame_offsets=None, window=-1):
    """Full forward of one (b, h): o [Ng+Nr, d], lse [Ng+Nr] (rows [G ; R])."""
    (B, H, d, Ng, Nr), off, offp = _shape_args(k_gen, k_ref, ref_block_offsets)
    keep = [_u16(x) for x in (q_gen, k_gen, v_gen, q_ref, k_ref, v_ref)]
    n = Ng + Nr
    o = np.zeros((n, d), dtype=np.float64)
    lse = np.zeros((n,), dtype=np.float64)
    mk, vp, vstride, fp, n_fr, w = _mask_args(valid, gen_frame_offsets, window, B, Nr)
    rc = _load().sra_oracle_forward_head_ex(*[k[1] for k in keep], B, H, d, Ng, Nr, offp, len(off) - 1,
                                            ctypes.c_double(scale), int(b), int(h), vp, vstride, fp, n_fr, w,
                                            o.ctypes.data_as(_f64p), lse.ctypes.data_as(_f64p))
    if rc != 0:
        raise RuntimeError(f"sra_oracle_forward_head failed: {rc}")
    return o, lse


def backward_head(q_gen, k_gen, v_gen, q_ref, k_ref, v_ref, do_gen, do_ref, ref_block_offsets, scale,
                  b, h, o, lse, rows=None, cols=None, valid=None, gen_frame_offsets=None, window=-1):
    """Backward of one (b, h) for query rows `rows` (dq) and key columns `cols` (dk, dv); None = all.
    o / lse must come from forward_head under the same valid / window options."""
    (B, H, d, Ng, Nr), off, offp = _shape_args(k_gen, k_ref, ref_block_offsets)
    keep = [_u16(x) for x in (q_gen, k_gen, v_gen, q_ref, k_ref, v_ref, do_gen, do_ref)]
    n = Ng + Nr
    if rows is None:
        rows_a, rows_p, n_rows = None, None, n
    else:
        rows_a, rows_p = _i32(rows)
        n_rows = len(rows_a)
    if cols is None:
        cols_a, cols_p, n_cols = None, None, n
    else:
        cols_a, cols_p = _i32(cols)
        n_cols = len(cols_a)
    o = np.ascontiguousarray(o, dtype=np.float64)
    lse = np.ascontiguousarray(lse, dtype=np.float64)
    dq = np.zeros((n_rows, d)); dk = np.zeros((n_cols, d)); dv = np.zeros((n_cols, d))
    mk, vp, vstride, fp, n_fr, w = _mask_args(valid, gen_frame_offsets, window, B, Nr)
    rc = _load().sra_oracle_backward_head_ex(*[k[1] for k in keep], B, H, d, Ng, Nr, offp, len(off) - 1,
                                             ctypes.c_double(scale), int(b), int(h),
                                             o.ctypes.data_as(_f64p), lse.ctypes.data_as(_f64p),
                                             rows_p, n_rows, cols_p, n_cols, vp, vstride, fp, n_fr, w,
                                             dq.ctypes.data_as(_f64p), dk.ctypes.data_as(_f64p),
                                             dv.ctypes.data_as(_f64p))
    if rc != 0:
        raise RuntimeError(f"sra_oracle_backward_head failed: {rc}")
    return dq, dk, dv

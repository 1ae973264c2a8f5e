"""Shared test helpers (no method arithmetic beyond error metrics)."""
import numpy as np
import torch

# Contract tolerance (BASELINE.json north_star): bf16 I/O, fp32 accumulation,
# GPU vs fp64 oracle max-abs <= 2e-2 and mean-abs <= 2e-3.  Self-imposed relative gate
# (SURVEY.md section 8c "tolerance bite"): rel_l2 <= 1e-2.
MAX_ABS_TOL = 2e-2
MEAN_ABS_TOL = 2e-3
REL_L2_TOL = 1e-2


def to_bf16_bits(x) -> np.ndarray:
    """Round a float array to bf16 (RNE) and return the uint16 bit patterns."""
    t = torch.as_tensor(np.asarray(x, dtype=np.float32)).to(torch.bfloat16)
    return t.contiguous().view(torch.int16).numpy().view(np.uint16).copy()


def bits_to_f64(bits) -> np.ndarray:
    """Independent (torch-based) upcast used to cross-check the oracle's own upcast."""
    t = torch.as_tensor(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16)
    return t.to(torch.float64).numpy()


def rand_bits(rng, shape, scale=1.0) -> np.ndarray:
    return to_bf16_bits(rng.standard_normal(shape) * scale)


def err_metrics(got, ref):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    diff = np.abs(got - ref)
    rms = float(np.sqrt(np.mean(ref ** 2))) if ref.size else 0.0
    return {
        "max_abs": float(diff.max()) if diff.size else 0.0,
        "mean_abs": float(diff.mean()) if diff.size else 0.0,
        "rel_l2": float(np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-300)),
        "max_over_rms": float(diff.max() / max(rms, 1e-300)) if diff.size else 0.0,
    }


def assert_parity(got, ref, what="", rel_l2_tol=REL_L2_TOL, max_abs_tol=MAX_ABS_TOL, mean_abs_tol=MEAN_ABS_TOL):
    m = err_metrics(got, ref)
    msg = (f"{what}: max_abs={m['max_abs']:.3e} (tol {max_abs_tol:g}) mean_abs={m['mean_abs']:.3e} "
           f"(tol {mean_abs_tol:g}) rel_l2={m['rel_l2']:.3e} (tol {rel_l2_tol:g}) max/rms={m['max_over_rms']:.3e}")
    assert np.all(np.isfinite(np.asarray(got, dtype=np.float64))), f"{what}: non-finite output"
    assert m["max_abs"] <= max_abs_tol, msg
    assert m["mean_abs"] <= mean_abs_tol, msg
    assert m["rel_l2"] <= rel_l2_tol, msg
    return m

"""Shared helpers for the parity tests (no arithmetic of the method lives here)."""
import numpy as np


def force_check(F_gpu, F_ref, rel=1e-4, floor=1e-5):
    """Strict per-component reading of BASELINE.json's tolerance (R15):
    |dF_c| <= max(rel |F_c|, floor).  Returns (#violations, worst err/tol)."""
    F_gpu = np.asarray(F_gpu, dtype=np.float64)
    tol = np.maximum(rel * np.abs(F_ref), floor)
    ratio = np.abs(F_gpu - F_ref) / tol
    return int(np.sum(ratio > 1.0)), float(np.max(ratio))


def melt(pos, vel, L, steps, oracle, **kw):
    """Advance with the oracle and return FP32-rounded (pos, vel) snapshot."""
    p, v, _, _ = oracle.verlet_run(pos, vel, L, steps, **kw)
    p = p.astype(np.float32)
    p[p >= np.float32(L)] = 0.0
    return p, v.astype(np.float32)

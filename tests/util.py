"""Shared helpers of the GPU parity tests (metrics only; no arithmetic of the method)."""
import numpy as np


def dslash_rel_err(got, ref):
    """DESIGN.md reading R10: max over sites of ||got(x)-ref(x)||_2 / max(||ref(x)||_2, 0.1 R),
    R = rms site norm of ref over its non-zero sites."""
    got = np.asarray(got, dtype=np.complex128)
    ref = np.asarray(ref, dtype=np.complex128)
    n = np.linalg.norm(ref, axis=1)
    nz = n > 0
    R = np.sqrt(np.mean(n[nz] ** 2)) if nz.any() else 1.0
    return float(np.max(np.linalg.norm(got - ref, axis=1) / np.maximum(n, 0.1 * R)))


def iters_close(gpu_iters, ref_iters):
    """DESIGN.md reading R8: |it_gpu - it_oracle| <= max(2, ceil(0.02 it_oracle))."""
    return abs(gpu_iters - ref_iters) <= max(2, int(np.ceil(0.02 * ref_iters)))


DSLASH_TOL = {64: 1e-13, 32: 2e-6}     # BASELINE.json north_star

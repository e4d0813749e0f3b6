"""ORACLE -- TEST INFRASTRUCTURE ONLY (ctypes wrapper around staggered_oracle.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference`
legs may import this package.  It shares nothing with paper_2502_03249_b200/ (the
CUDA product) except the seeded input arrays of qcd_inputs/.

Arrays use the canonical host layouts, over the FULL lattice, lexicographic with
x0 fastest:  U complex [V][4][3][3] (U[idx, mu] = U_{x,mu}), spinors complex [V][3].
complex128 selects the fp64 oracle, complex64 the fp32-arithmetic variant (fields
and field arithmetic in float, inner products and CG scalars in double).

Functions (citations in staggered_oracle.c / staggered_impl.inc):
    dslash(dims, U, phi, out_parity)   Eq. (1) rows of one parity (or -1: all sites)
    dslash_site(dims, U, phi, x)       one output site of Eq. (1)
    apply_M(dims, U, v, m)             M v = m^2 v - D_eo D_oe v on even sites
    cg(dims, U, b, m, tol, maxiter)    Hestenes-Stiefel CG on M x = b, x0 = 0
    true_residual(dims, U, b, x, m)    ||b - M x|| / ||b||  (recomputed, fp64)
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import time

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "staggered_oracle.c"), os.path.join(_HERE, "staggered_impl.inc")]
_LIB_PATH = os.path.join(_HERE, "liboracle_staggered.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (OpenMP).  Returns the path of the shared object."""
    if not force and os.path.exists(_LIB_PATH) and all(
            os.path.getmtime(_LIB_PATH) >= os.path.getmtime(s) for s in _SRC):
        return _LIB_PATH
    tmp = _LIB_PATH + f".tmp{os.getpid()}"
    cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fcx-limited-range", "-shared", "-fPIC",
           "-o", tmp, _SRC[0], "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    os.replace(tmp, _LIB_PATH)
    return _LIB_PATH


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_num_threads.restype = ctypes.c_int
        for sfx in ("f64", "f32"):
            getattr(_lib, f"oracle_re_dot_even_{sfx}").restype = ctypes.c_double
            getattr(_lib, f"oracle_cg_{sfx}").restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(ctypes.c_int(int(n)))


def _dims(dims):
    d = [int(v) for v in dims]
    if len(d) != 4 or any(v < 2 or v % 2 for v in d):
        raise ValueError("dims must be four even extents >= 2")
    return (ctypes.c_int * 4)(*d), d[0] * d[1] * d[2] * d[3]


def _sfx(*arrays) -> str:
    dt = arrays[0].dtype
    if any(a.dtype != dt for a in arrays):
        raise TypeError("all arrays must share one dtype")
    if dt == np.complex128:
        return "f64"
    if dt == np.complex64:
        return "f32"
    raise TypeError(f"need complex128 or complex64, got {dt}")


def _chk(a: np.ndarray, shape) -> np.ndarray:
    a = np.ascontiguousarray(a)
    if a.shape != tuple(shape):
        raise ValueError(f"expected shape {tuple(shape)}, got {a.shape}")
    return a


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def dslash(dims, U, phi, out_parity: int) -> np.ndarray:
    """(D phi)(x) on sites of `out_parity` (0: D_eo phi_odd, 1: D_oe phi_even, -1: all); 0 elsewhere."""
    n, v = _dims(dims)
    U, phi = _chk(U, (v, 4, 3, 3)), _chk(phi, (v, 3))
    out = np.zeros_like(phi)
    getattr(_load(), f"oracle_dslash_{_sfx(U, phi)}")(n, _p(U), _p(phi), _p(out), ctypes.c_int(int(out_parity)))
    return out


def dslash_site(dims, U, phi, x) -> np.ndarray:
    n, v = _dims(dims)
    U, phi = _chk(U, (v, 4, 3, 3)), _chk(phi, (v, 3))
    out = np.zeros(3, dtype=phi.dtype)
    xx = (ctypes.c_int * 4)(*[int(c) for c in x])
    getattr(_load(), f"oracle_dslash_site_{_sfx(U, phi)}")(n, _p(U), _p(phi), xx, _p(out))
    return out


def apply_M(dims, U, vec, m: float) -> np.ndarray:
    """M vec = m^2 vec - D_eo D_oe vec on even sites (odd sites of the result are 0)."""
    n, v = _dims(dims)
    U, vec = _chk(U, (v, 4, 3, 3)), _chk(vec, (v, 3))
    out, tmp = np.zeros_like(vec), np.zeros_like(vec)
    getattr(_load(), f"oracle_apply_M_{_sfx(U, vec)}")(n, _p(U), _p(vec), _p(out), ctypes.c_double(float(m)), _p(tmp))
    return out


def re_dot_even(dims, a, b) -> float:
    n, v = _dims(dims)
    a, b = _chk(a, (v, 3)), _chk(b, (v, 3))
    return float(getattr(_load(), f"oracle_re_dot_even_{_sfx(a, b)}")(n, _p(a), _p(b)))


def cg(dims, U, b, m: float, tol: float, maxiter: int, history: bool = False):
    """CG on M x = b.  Returns (x, info) with info = dict(status, iters, rel_resid, bnorm2,
    converged, seconds[, history])."""
    n, v = _dims(dims)
    U, b = _chk(U, (v, 4, 3, 3)), _chk(b, (v, 3))
    sfx = _sfx(U, b)
    x = np.zeros_like(b)
    work = np.zeros((4, v, 3), dtype=b.dtype)
    iters, relres, bb = ctypes.c_int(0), ctypes.c_double(0.0), ctypes.c_double(0.0)
    hist = np.zeros(int(maxiter) if history else 1, dtype=np.float64)
    t0 = time.perf_counter()
    status = getattr(_load(), f"oracle_cg_{sfx}")(
        n, _p(U), _p(b), _p(x), ctypes.c_double(float(m)), ctypes.c_double(float(tol)),
        ctypes.c_int(int(maxiter)), _p(work), ctypes.byref(iters), ctypes.byref(relres),
        ctypes.byref(bb), _p(hist) if history else None, ctypes.c_int(hist.size if history else 0))
    dt = time.perf_counter() - t0
    info = dict(status=int(status), iters=int(iters.value), rel_resid=float(relres.value),
                bnorm2=float(bb.value), converged=(status == 0), seconds=dt)
    if history:
        info["history"] = hist[: iters.value].copy()
    return x, info


def true_residual(dims, U, b, x, m: float) -> float:
    """||b - M x||_2 / ||b||_2 over even sites, everything promoted to fp64."""
    U64 = np.ascontiguousarray(U, dtype=np.complex128)
    b64 = np.ascontiguousarray(b, dtype=np.complex128)
    x64 = np.ascontiguousarray(x, dtype=np.complex128)
    r = b64 - apply_M(dims, U64, x64, m)
    return float(np.sqrt(re_dot_even(dims, r, r) / re_dot_even(dims, b64, b64)))

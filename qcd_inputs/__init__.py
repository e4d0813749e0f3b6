"""Seeded synthetic inputs for the staggered Dslash / CG path.

This module is the ONLY thing the CPU oracle (`oracle/`) and the CUDA path
(`paper_2502_03249_b200/`) have in common.  It holds no arithmetic of the
method (no Dslash, no phases, no boundary signs, no CG): it only produces
arrays in the canonical host layouts:

    gauge  : complex128 [V][mu=4][row=3][col=3]   (`U[idx, mu]` = U_{x,mu})
    spinor : complex128 [V][colour=3]
    idx    : x0 + N0*(x1 + N1*(x2 + N2*x3)), x0 fastest, over the FULL lattice

The recipes follow BASELINE.json `configs`:
  * Haar SU(3): Z iid complex Gaussian 3x3, Q from QR with R's diagonal real
    positive (= Gram-Schmidt on the columns), U = Q * det(Q)^(-1/3)  (configs[0]).
  * near-identity: U = exp(i*eps*H), H = (A + A^dagger)/2 - tr/3, A iid complex
    Gaussian with E|A_ij|^2 = 1                                      (configs[1]).
  * source: iid complex Gaussian (E|z|^2 = 1) on the sites of one parity,
    exactly zero on the other.

Random numbers come from Philox streams keyed by (seed, stream, chunk), so a
field is the same no matter how many worker threads generate it.
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

__all__ = [
    "volume", "site_coords", "site_parity", "haar_su3", "near_identity_su3",
    "gauge_field", "gaussian_source", "gaussian_spinor", "CONFIGS", "config_inputs",
]

_CHUNK = 1 << 16  # matrices / sites per Philox stream (part of the recipe: do not change)

# stream ids (second word of the Philox key)
_STREAM_HAAR, _STREAM_NEARID, _STREAM_SPINOR = 1, 2, 3


def _workers() -> int:
    try:
        n = len(os.sched_getaffinity(0))
    except AttributeError:  # pragma: no cover
        n = os.cpu_count() or 1
    return max(1, min(n, 32))


def _rng(seed: int, stream: int, chunk: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed), int(stream)], counter=[0, 0, int(chunk), 0]))


def _chunked(n: int, fn, out: np.ndarray) -> np.ndarray:
    """Fill out[lo:hi] = fn(chunk_index, hi - lo) for every chunk, in parallel."""
    nchunks = (n + _CHUNK - 1) // _CHUNK

    def work(c: int) -> None:
        lo, hi = c * _CHUNK, min(n, (c + 1) * _CHUNK)
        out[lo:hi] = fn(c, hi - lo)

    if nchunks <= 1:
        for c in range(nchunks):
            work(c)
    else:
        with ThreadPoolExecutor(max_workers=_workers()) as ex:
            list(ex.map(work, range(nchunks)))
    return out


def _complex_gaussian(rng: np.random.Generator, shape) -> np.ndarray:
    """iid complex Gaussian with E|z|^2 = 1."""
    z = rng.standard_normal(size=tuple(shape) + (2,))
    return (z[..., 0] + 1j * z[..., 1]) * np.sqrt(0.5)


def volume(dims) -> int:
    n0, n1, n2, n3 = (int(d) for d in dims)
    return n0 * n1 * n2 * n3


def site_coords(dims) -> np.ndarray:
    """int32 [V][4]: coordinates (x0,x1,x2,x3) of lexicographic site idx (x0 fastest)."""
    n0, n1, n2, n3 = (int(d) for d in dims)
    idx = np.arange(n0 * n1 * n2 * n3, dtype=np.int64)
    x = np.empty((idx.size, 4), dtype=np.int32)
    x[:, 0] = idx % n0
    x[:, 1] = (idx // n0) % n1
    x[:, 2] = (idx // (n0 * n1)) % n2
    x[:, 3] = idx // (n0 * n1 * n2)
    return x


def site_parity(dims) -> np.ndarray:
    """uint8 [V]: (x0+x1+x2+x3) mod 2 of every lexicographic site (0 = even)."""
    return (site_coords(dims).sum(axis=1) & 1).astype(np.uint8)


def _haar_chunk(seed: int, c: int, n: int) -> np.ndarray:
    z = _complex_gaussian(_rng(seed, _STREAM_HAAR, c), (n, 3, 3))
    # Gram-Schmidt on the columns == QR with diag(R) real positive.
    q = np.empty_like(z)
    a0 = z[:, :, 0]
    q0 = a0 / np.linalg.norm(a0, axis=1, keepdims=True)
    a1 = z[:, :, 1]
    a1 = a1 - q0 * np.sum(q0.conj() * a1, axis=1, keepdims=True)
    q1 = a1 / np.linalg.norm(a1, axis=1, keepdims=True)
    a2 = z[:, :, 2]
    a2 = a2 - q0 * np.sum(q0.conj() * a2, axis=1, keepdims=True)
    a2 = a2 - q1 * np.sum(q1.conj() * a2, axis=1, keepdims=True)
    # second pass keeps the third column orthogonal to working precision
    a2 = a2 - q0 * np.sum(q0.conj() * a2, axis=1, keepdims=True)
    a2 = a2 - q1 * np.sum(q1.conj() * a2, axis=1, keepdims=True)
    q2 = a2 / np.linalg.norm(a2, axis=1, keepdims=True)
    q[:, :, 0], q[:, :, 1], q[:, :, 2] = q0, q1, q2
    det = (q[:, 0, 0] * (q[:, 1, 1] * q[:, 2, 2] - q[:, 1, 2] * q[:, 2, 1])
           - q[:, 0, 1] * (q[:, 1, 0] * q[:, 2, 2] - q[:, 1, 2] * q[:, 2, 0])
           + q[:, 0, 2] * (q[:, 1, 0] * q[:, 2, 1] - q[:, 1, 1] * q[:, 2, 0]))
    # principal cube root of det (|det| = 1): exp(-i*arg(det)/3)
    fix = np.exp(-1j * np.angle(det) / 3.0)
    return q * fix[:, None, None]


def haar_su3(n: int, seed: int) -> np.ndarray:
    """complex128 [n][3][3], Haar-distributed SU(3) (det = 1)."""
    out = np.empty((int(n), 3, 3), dtype=np.complex128)
    return _chunked(int(n), lambda c, m: _haar_chunk(seed, c, m), out)


def _nearid_chunk(seed: int, eps: float, c: int, n: int) -> np.ndarray:
    a = _complex_gaussian(_rng(seed, _STREAM_NEARID, c), (n, 3, 3))
    h = 0.5 * (a + np.conj(np.swapaxes(a, 1, 2)))
    tr = np.trace(h, axis1=1, axis2=2).real / 3.0
    h[:, 0, 0] -= tr
    h[:, 1, 1] -= tr
    h[:, 2, 2] -= tr
    lam, v = np.linalg.eigh(h)
    ph = np.exp(1j * float(eps) * lam)
    return np.einsum("nij,nj,nkj->nik", v, ph, v.conj())


def near_identity_su3(n: int, eps: float, seed: int) -> np.ndarray:
    """complex128 [n][3][3], U = exp(i*eps*H) with H random traceless Hermitian."""
    out = np.empty((int(n), 3, 3), dtype=np.complex128)
    return _chunked(int(n), lambda c, m: _nearid_chunk(seed, eps, c, m), out)


def gauge_field(dims, kind: str, seed: int = 0, eps: float | None = None) -> np.ndarray:
    """complex128 [V][4][3][3].  kind: 'haar' | 'near_identity' (needs eps) | 'unit'."""
    v = volume(dims)
    if kind == "haar":
        u = haar_su3(4 * v, seed)
    elif kind == "near_identity":
        if eps is None:
            raise ValueError("near_identity needs eps")
        u = near_identity_su3(4 * v, eps, seed)
    elif kind == "unit":
        u = np.zeros((4 * v, 3, 3), dtype=np.complex128)
        u[:, 0, 0] = u[:, 1, 1] = u[:, 2, 2] = 1.0
    else:
        raise ValueError(f"unknown gauge kind {kind!r}")
    return u.reshape(v, 4, 3, 3)


def gaussian_spinor(dims, seed: int) -> np.ndarray:
    """complex128 [V][3], iid complex Gaussian on every site."""
    v = volume(dims)
    out = np.empty((v, 3), dtype=np.complex128)
    return _chunked(v, lambda c, m: _complex_gaussian(_rng(seed, _STREAM_SPINOR, c), (m, 3)), out)


def gaussian_source(dims, seed: int = 1, parity: int = 0) -> np.ndarray:
    """complex128 [V][3]: Gaussian on sites of `parity`, exactly zero elsewhere."""
    phi = gaussian_spinor(dims, seed)
    phi[site_parity(dims) != parity] = 0.0
    return phi


# BASELINE.json `configs`, in order.  Seeds: links 0, source 1.
CONFIGS = [
    dict(name="4^4", dims=(4, 4, 4, 4), links="haar", eps=None, m=0.1,
         tol64=1e-10, tol32=None, maxiter=10000),
    dict(name="16^4", dims=(16, 16, 16, 16), links="near_identity", eps=0.3, m=0.05,
         tol64=1e-10, tol32=1e-5, maxiter=10000),
    dict(name="32^4", dims=(32, 32, 32, 32), links="haar", eps=None, m=0.05,
         tol64=1e-8, tol32=1e-5, maxiter=5000),
    dict(name="48^3x12", dims=(48, 48, 48, 12), links="near_identity", eps=0.5, m=0.01,
         tol64=1e-8, tol32=None, maxiter=10000),
    dict(name="64^4", dims=(64, 64, 64, 64), links="haar", eps=None, m=0.01,
         tol64=1e-8, tol32=1e-5, maxiter=10000),
]


def config_inputs(i: int, dims=None):
    """(cfg, U, b) for BASELINE.json configs[i]; `dims` overrides the lattice (same recipe)."""
    cfg = dict(CONFIGS[i])
    if dims is not None:
        cfg["dims"] = tuple(int(d) for d in dims)
    u = gauge_field(cfg["dims"], cfg["links"], seed=0, eps=cfg["eps"])
    b = gaussian_source(cfg["dims"], seed=1, parity=0)
    return cfg, u, b

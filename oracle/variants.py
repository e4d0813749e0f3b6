"""ORACLE -- TEST INFRASTRUCTURE ONLY: the paper's Dslash variants.

Plain numpy in fp64 on the canonical host layouts (U complex [V][4][3][3], spinors complex
[V][3], idx = x0 + N0 (x1 + N1 (x2 + N2 x3))), on top of the C oracle of Eq. (1)
(oracle.dslash / apply_M / cg).  Nothing here is shared with the CUDA product.

  two-row links     PAPER.md:76 "For each link variable, we store only the first two rows, i.e.
                    12 floats.  The third row is reconstructed on-the-fly when needed, using the
                    properties of SU(3) matrices."            -> compress12 / reconstruct12
  temporal gauge    PAPER.md:76 "We use gauge fixing to transform the temporal link variables to
                    1_{3x3} for all the sites with the temporal coordinate t != 0."
                                                               -> temporal_gauge / rotate_spinor
  multiple vectors  PAPER.md:76-78 "applying D on multiple vectors at once ... each link variable
                    to be read once and then reused for multiple vectors" (NMULTI)
                                                               -> dslash_multi / cg_multi
  mixed precision   PAPER.md:66 (D and CG "in single and double precision"); reading R21:
                    defect correction, fp64 outer residual, fp32 inner CG  -> mixed_cg

Pins: tests/test_oracle_variants.py.  Parity unpinned: the inner-iteration count of mixed_cg on
random links (self-consistency only, like the plain CG count).
"""
from __future__ import annotations

import numpy as np

import oracle


# ------------------------------------------------------------------------------------------
# two-row ("reconstruct-12") link storage
# ------------------------------------------------------------------------------------------
def compress12(U: np.ndarray) -> np.ndarray:
    """[..., 3, 3] -> [..., 2, 3]: the first two rows of every link."""
    return np.ascontiguousarray(U[..., :2, :])


def reconstruct12(U12: np.ndarray) -> np.ndarray:
    """[..., 2, 3] -> [..., 3, 3].  For U in SU(3) the rows a, b, c are orthonormal with
    det = 1, hence c = conj(a x b):  c_k = conj(eps_{kij} a_i b_j)."""
    a, b = U12[..., 0, :], U12[..., 1, :]
    c = np.empty_like(a)
    c[..., 0] = np.conj(a[..., 1] * b[..., 2] - a[..., 2] * b[..., 1])
    c[..., 1] = np.conj(a[..., 2] * b[..., 0] - a[..., 0] * b[..., 2])
    c[..., 2] = np.conj(a[..., 0] * b[..., 1] - a[..., 1] * b[..., 0])
    out = np.empty(U12.shape[:-2] + (3, 3), dtype=U12.dtype)
    out[..., 0, :], out[..., 1, :], out[..., 2, :] = a, b, c
    return out


# ------------------------------------------------------------------------------------------
# temporal gauge fixing, PAPER.md:76 (reading R20)
# ------------------------------------------------------------------------------------------
def _mm(a, b):
    return np.einsum("...ij,...jk->...ik", a, b)


def _dag(a):
    return np.conj(np.swapaxes(a, -1, -2))


def temporal_gauge(dims, U: np.ndarray):
    """Gauge transformation g(x) with U'_{x,mu} = g(x) U_{x,mu} g(x+mu)^dagger such that
    U'_{x,3} = 1 for every site with x3 != 0 (the paper's statement, literally):

        g(xs, 0) = 1
        g(xs, t) = g(xs, t+1) U_{(xs,t),3}^dagger      for t = N3-1, N3-2, ..., 1   (t+1 wraps to 0)

    so that g(t) U_3(t) g(t+1)^dagger = 1 for t = 1..N3-1, and the t = 0 link becomes the
    Polyakov loop U_3(0) U_3(1) ... U_3(N3-1).  Returns (U', g) with g complex [V][3][3]."""
    n0, n1, n2, n3 = (int(d) for d in dims)
    vs = n0 * n1 * n2
    U4 = U.reshape(n3, vs, 4, 3, 3)                       # [t][xs][mu]
    g = np.empty((n3, vs, 3, 3), dtype=U.dtype)
    g[0] = np.eye(3)
    nxt = g[0]
    for t in range(n3 - 1, 0, -1):
        g[t] = _mm(nxt, _dag(U4[t, :, 3]))
        nxt = g[t]
    gl = g.reshape(n3, n2, n1, n0, 3, 3)                  # [x3][x2][x1][x0]
    Ul = U.reshape(n3, n2, n1, n0, 4, 3, 3)
    out = np.empty_like(Ul)
    for mu in range(4):
        axis = 3 - mu                                     # x_mu is array axis 3 - mu
        g_fwd = np.roll(gl, -1, axis=axis)                # g(x + mu), periodic (gauge fields are periodic)
        out[..., mu, :, :] = _mm(_mm(gl, Ul[..., mu, :, :]), _dag(g_fwd))
    return out.reshape(U.shape), g.reshape(-1, 3, 3)


def rotate_spinor(g: np.ndarray, phi: np.ndarray, dagger: bool = False) -> np.ndarray:
    """phi'(x) = g(x) phi(x)   (dagger: g(x)^dagger phi(x))."""
    gg = _dag(g) if dagger else g
    return np.einsum("nij,nj->ni", gg, phi)


# ------------------------------------------------------------------------------------------
# multiple vectors (NMULTI): D applied to each vector, by definition
# ------------------------------------------------------------------------------------------
def dslash_multi(dims, U, phis, out_parity: int):
    return [oracle.dslash(dims, U, phi, out_parity) for phi in phis]


def cg_multi(dims, U, bs, m, tol, maxiter):
    """n independent CG solves (each its own alpha, beta, stopping iteration)."""
    res = [oracle.cg(dims, U, b, m, tol, maxiter) for b in bs]
    return [r[0] for r in res], [r[1] for r in res]


# ------------------------------------------------------------------------------------------
# mixed-precision defect-correction CG (reading R21)
# ------------------------------------------------------------------------------------------
def mixed_cg(dims, U, b, m, tol, inner_tol, maxiter, max_outer: int = 50):
    """Solve M x = b to a TRUE fp64 relative residual <= tol with fp32 inner solves:

        x = 0;  r = b                                     (fp64)
        repeat:
            if ||r|| / ||b|| <= tol: converged
            tol_in = max(inner_tol, 0.5 * tol * ||b|| / ||r||)   (never ask the inner solve for more than is needed)
            s = ||r||;  rhs32 = fp32(r / s)               (normalised so that fp32 never under/overflows)
            e32 = CG_fp32(M32, rhs32, tol_in)             (oracle f32 variant: fp32 fields, fp64 scalars)
            x += s * fp64(e32)                            (fp64)
            r = b - M x                                   (fp64, recomputed: the TRUE residual)

    M32 uses the fp32 rounding of the links.  Returns (x, info) with info = dict(converged,
    outer, inner_iters (sum over inner solves), inner_per_outer, true_resid, m_applications_fp64)."""
    U64 = np.ascontiguousarray(U, dtype=np.complex128)
    U32 = U64.astype(np.complex64)
    b = np.ascontiguousarray(b, dtype=np.complex128)
    x = np.zeros_like(b)
    r = b.copy()
    bb = oracle.re_dot_even(dims, b, b)
    info = dict(converged=False, outer=0, inner_iters=0, inner_per_outer=[], true_resid=1.0, m_applications_fp64=0)
    if bb == 0.0:
        info.update(converged=True, true_resid=0.0)
        return x, info
    budget = int(maxiter)
    while True:
        rr = oracle.re_dot_even(dims, r, r)
        rel = float(np.sqrt(rr / bb))
        info["true_resid"] = rel
        if rel <= tol:
            info["converged"] = True
            break
        if info["outer"] >= max_outer or budget <= 0:
            break
        tol_in = max(float(inner_tol), 0.5 * tol / rel)
        s = float(np.sqrt(rr))
        rhs32 = (r / s).astype(np.complex64)
        e32, iinfo = oracle.cg(dims, U32, rhs32, m, tol_in, budget)
        budget -= iinfo["iters"]
        info["inner_iters"] += iinfo["iters"]
        info["inner_per_outer"].append(iinfo["iters"])
        info["outer"] += 1
        x += s * e32.astype(np.complex128)
        r = b - oracle.apply_M(dims, U64, x, m)
        info["m_applications_fp64"] += 1
    return x, info

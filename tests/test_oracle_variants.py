"""Pins for oracle/variants.py (two-row links, temporal gauge, multiple vectors, mixed-precision
CG): what the paper's statements and the mathematics fix.  No CUDA, no
comparison of a function with itself.  Each pin fails on a plausible mistake (missing conj or
swapped operands in the cross product, g on the wrong end of a link, recursion in the wrong
time direction, the non-trivial link on the wrong time slice, a lost scale factor)."""
import numpy as np
import pytest

import oracle
import oracle.variants as ov
import qcd_inputs as qi

DA = (4, 6, 2, 8)


# ---------------------------------------------------------------- two-row links
def test_reconstruct12_gives_back_the_third_row_of_generated_su3():
    # the generators (Gram-Schmidt + det fix; eigh + exp) know nothing about cross products
    for U in (qi.haar_su3(5000, seed=7), qi.near_identity_su3(5000, 0.5, seed=8)):
        R = ov.reconstruct12(ov.compress12(U))
        assert np.array_equal(R[:, :2], U[:, :2])
        assert np.abs(R[:, 2] - U[:, 2]).max() < 5e-15


def test_reconstruct12_closed_forms():
    a, b = 0.7, -1.9
    d = np.zeros((1, 2, 3), dtype=np.complex128)
    d[0, 0, 0], d[0, 1, 1] = np.exp(1j * a), np.exp(1j * b)
    R = ov.reconstruct12(d)[0]
    assert np.allclose(R[2], [0, 0, np.exp(-1j * (a + b))], atol=1e-16)      # det = 1
    # a cyclic permutation matrix with phases: rows e_1 e^{ia}, e_2 e^{ib} -> third row e_0 e^{-i(a+b)}
    p = np.zeros((1, 2, 3), dtype=np.complex128)
    p[0, 0, 1], p[0, 1, 2] = np.exp(1j * a), np.exp(1j * b)
    R = ov.reconstruct12(p)[0]
    assert np.allclose(R[2], [np.exp(-1j * (a + b)), 0, 0], atol=1e-16)
    assert abs(np.linalg.det(R) - 1) < 1e-15
    # generic: unitary with det 1
    U = ov.reconstruct12(ov.compress12(qi.haar_su3(100, seed=9)))
    assert np.abs(np.einsum("nij,nkj->nik", U, U.conj()) - np.eye(3)).max() < 1e-14
    assert np.abs(np.linalg.det(U) - 1).max() < 1e-14


def test_dslash_on_reconstructed_links_equals_dslash_on_full_links():
    U = qi.gauge_field(DA, "haar", seed=0)
    phi = qi.gaussian_source(DA, seed=1, parity=0)
    ref = oracle.dslash(DA, U, phi, 1)
    got = oracle.dslash(DA, ov.reconstruct12(ov.compress12(U)), phi, 1)
    assert np.abs(got - ref).max() < 1e-13


# ---------------------------------------------------------------- temporal gauge
def _polyakov(dims, U, xs):
    """U_3(xs,0) U_3(xs,1) ... U_3(xs,N3-1) by an explicit site loop."""
    n0, n1, n2, n3 = dims
    P = np.eye(3, dtype=np.complex128)
    for t in range(n3):
        idx = xs[0] + n0 * (xs[1] + n1 * (xs[2] + n2 * t))
        P = P @ U[idx, 3]
    return P


def _plaquette_trace(dims, U, mu, nu):
    """Re tr of the mu-nu plaquette at every site (gauge invariant)."""
    n0, n1, n2, n3 = dims
    Ul = U.reshape(n3, n2, n1, n0, 4, 3, 3)
    sh = lambda a, d: np.roll(a, -1, axis=3 - d)
    A, B = Ul[..., mu, :, :], Ul[..., nu, :, :]
    P = A @ sh(B, mu) @ np.conj(np.swapaxes(sh(A, nu), -1, -2)) @ np.conj(np.swapaxes(B, -1, -2))
    return np.trace(P, axis1=-2, axis2=-1).real


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), DA])
def test_temporal_gauge_links_are_unit_for_t_ne_0_and_polyakov_loop_at_t_0(dims):
    U = qi.gauge_field(dims, "haar", seed=0)
    Uf, g = ov.temporal_gauge(dims, U)
    n0, n1, n2, n3 = dims
    x3 = qi.site_coords(dims)[:, 3]
    assert np.abs(Uf[x3 != 0, 3] - np.eye(3)).max() < 1e-14          # the paper's statement
    assert np.abs(g[x3 == 0] - np.eye(3)).max() == 0.0
    for xs in [(0, 0, 0), (1, 2, 1), (n0 - 1, n1 - 1, n2 - 1)]:
        idx0 = xs[0] + n0 * (xs[1] + n1 * xs[2])
        assert np.abs(Uf[idx0, 3] - _polyakov(dims, U, xs)).max() < 1e-13
    # still SU(3), plaquettes (gauge invariant) unchanged in every plane
    assert np.abs(np.einsum("nmij,nmkj->nmik", Uf, Uf.conj()) - np.eye(3)).max() < 1e-13
    for mu, nu in [(0, 1), (0, 3), (2, 3), (1, 2)]:
        assert np.abs(_plaquette_trace(dims, Uf, mu, nu) - _plaquette_trace(dims, U, mu, nu)).max() < 1e-12


def test_temporal_gauge_is_a_gauge_transformation_of_the_operator():
    # D[U^g] (g phi) = g D[U] phi, and the solve is covariant: x' = g x
    dims = DA
    U = qi.gauge_field(dims, "haar", seed=0)
    Uf, g = ov.temporal_gauge(dims, U)
    phi = qi.gaussian_source(dims, seed=1, parity=0)
    lhs = oracle.dslash(dims, Uf, ov.rotate_spinor(g, phi), 1)
    rhs = ov.rotate_spinor(g, oracle.dslash(dims, U, phi, 1))
    assert np.abs(lhs - rhs).max() < 1e-13
    back = ov.rotate_spinor(g, ov.rotate_spinor(g, phi), dagger=True)
    assert np.abs(back - phi).max() < 1e-14
    x, info = oracle.cg(dims, U, phi, 0.1, 1e-10, 2000)
    xf, infof = oracle.cg(dims, Uf, ov.rotate_spinor(g, phi), 0.1, 1e-10, 2000)
    assert abs(info["iters"] - infof["iters"]) <= max(2, int(np.ceil(0.02 * info["iters"])))   # rounding only (R8)
    assert np.linalg.norm(ov.rotate_spinor(g, xf, dagger=True) - x) <= 1e-7 * np.linalg.norm(x)


# ---------------------------------------------------------------- multiple vectors
def test_dslash_multi_is_linear_in_the_vectors():
    dims = DA
    U = qi.gauge_field(dims, "haar", seed=0)
    phis = [qi.gaussian_source(dims, seed=20 + i, parity=0) for i in range(3)]
    outs = ov.dslash_multi(dims, U, phis, 1)
    c = [0.3 - 1j, 2.0, -0.5j]
    comb = oracle.dslash(dims, U, sum(ci * p for ci, p in zip(c, phis)), 1)
    assert np.abs(comb - sum(ci * o for ci, o in zip(c, outs))).max() < 1e-12


# ---------------------------------------------------------------- mixed-precision CG (R21)
def test_mixed_cg_reaches_fp64_tolerance_and_matches_dense_solve_4x4x4x4():
    dims, m, tol = (4, 4, 4, 4), 0.1, 1e-10
    U = qi.gauge_field(dims, "haar", seed=0)
    b = qi.gaussian_source(dims, seed=1, parity=0)
    x, info = ov.mixed_cg(dims, U, b, m, tol, 1e-4, 20000)
    assert info["converged"] and info["outer"] >= 2
    assert oracle.true_residual(dims, U, b, x, m) <= tol
    # dense 384 x 384 solve (LAPACK), as pin P5 does for the plain CG
    v = qi.volume(dims)
    even = np.flatnonzero(qi.site_parity(dims) == 0)
    cols = (3 * even[:, None] + np.arange(3)[None, :]).reshape(-1)
    M = np.zeros((cols.size, cols.size), dtype=np.complex128)
    e = np.zeros((v, 3), dtype=np.complex128)
    for jj, j in enumerate(cols):
        e.flat[j] = 1.0
        M[:, jj] = oracle.apply_M(dims, U, e, m).reshape(-1)[cols]
        e.flat[j] = 0.0
    xd = np.linalg.solve(M, b.reshape(-1)[cols])
    lam = np.linalg.eigvalsh(M)
    kappa = lam[-1] / lam[0]
    assert np.linalg.norm(x.reshape(-1)[cols] - xd) <= kappa * tol * np.linalg.norm(xd)


def test_mixed_cg_on_rough_links_meets_the_tolerance_plain_fp32_cannot():
    dims, m, tol = (8, 8, 8, 8), 0.05, 1e-8
    U = qi.gauge_field(dims, "haar", seed=0)
    b = qi.gaussian_source(dims, seed=1, parity=0)
    x, info = ov.mixed_cg(dims, U, b, m, tol, 1e-4, 20000)
    assert info["converged"], info
    assert oracle.true_residual(dims, U, b, x, m) <= tol
    x64, i64 = oracle.cg(dims, U, b, m, tol, 20000)
    assert np.linalg.norm(x - x64) <= 1e-5 * np.linalg.norm(x64)
    # zero source
    x0, i0 = ov.mixed_cg(dims, U, np.zeros_like(b), m, tol, 1e-4, 100)
    assert i0["converged"] and not x0.any()

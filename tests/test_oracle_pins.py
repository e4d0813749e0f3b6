"""Pins for the CPU oracle (`oracle/`): what the paper's Eq. (1) and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path.  Each pin is
chosen so that a plausible mistake (dropped term, wrong sign / index, transposed
operand, dagger on the wrong hop, seam on the wrong side, wrong eta convention)
fails at least one of them.  Citations: PAPER.md:49-54 (Eq. 1), BASELINE.json
north_star / configs[0] (conventions), SURVEY.md Sec. 8(c) C4 (pins P1..P8).
"""
import os

import numpy as np
import pytest

import oracle
import qcd_inputs as qi

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
D4 = (4, 4, 4, 4)
DA = (4, 6, 2, 8)   # all extents different: catches swapped strides / extents


def _lex(dims, x):
    return x[0] + dims[0] * (x[1] + dims[1] * (x[2] + dims[2] * x[3]))


def _dense_D(dims, U):
    """Full D as a dense (3V x 3V) matrix, column by column from unit vectors."""
    v = qi.volume(dims)
    D = np.zeros((3 * v, 3 * v), dtype=np.complex128)
    e = np.zeros((v, 3), dtype=np.complex128)
    for j in range(3 * v):
        e.flat[j] = 1.0
        D[:, j] = oracle.dslash(dims, U, e, -1).reshape(-1)
        e.flat[j] = 0.0
    return D


def _dense_M(dims, U, m):
    """M on even sites as a dense (3Vh x 3Vh) matrix via oracle.apply_M on unit vectors."""
    v = qi.volume(dims)
    even = np.flatnonzero(qi.site_parity(dims) == 0)
    cols = (3 * even[:, None] + np.arange(3)[None, :]).reshape(-1)
    M = np.zeros((cols.size, cols.size), dtype=np.complex128)
    e = np.zeros((v, 3), dtype=np.complex128)
    for jj, j in enumerate(cols):
        e.flat[j] = 1.0
        M[:, jj] = oracle.apply_M(dims, U, e, m).reshape(-1)[cols]
        e.flat[j] = 0.0
    return M, cols


@pytest.fixture(scope="module")
def haar4():
    return qi.gauge_field(D4, "haar", seed=0)


@pytest.fixture(scope="module")
def dense4(haar4):
    return _dense_D(D4, haar4)


# ---------------------------------------------------------------- P1 anti-hermiticity
def test_P1_dense_antihermitian_and_block_structure(dense4):
    par = np.repeat(qi.site_parity(D4), 3)
    D = dense4
    assert np.abs(D + D.conj().T).max() < 1e-14          # D^dagger = -D  <=>  D_oe = -D_eo^dagger
    assert np.abs(D[np.ix_(par == 0, par == 0)]).max() == 0.0   # even-even block exactly zero
    assert np.abs(D[np.ix_(par == 1, par == 1)]).max() == 0.0   # odd-odd block exactly zero
    # every row has exactly 8 neighbours x 3 colours of nonzeros
    assert np.all((np.abs(D) > 0).sum(axis=1) == 24)


@pytest.mark.parametrize("dims,kind", [(DA, "haar"), ((8, 8, 8, 8), "near_identity")])
def test_P1_antihermiticity_inner_products(dims, kind):
    U = qi.gauge_field(dims, kind, seed=0, eps=0.5)
    par = qi.site_parity(dims)
    phi_e = qi.gaussian_source(dims, seed=11, parity=0)
    psi_o = qi.gaussian_source(dims, seed=12, parity=1)
    lhs = np.vdot(psi_o, oracle.dslash(dims, U, phi_e, 1))       # <psi_o, D_oe phi_e>
    rhs = np.vdot(phi_e, oracle.dslash(dims, U, psi_o, 0))       # <phi_e, D_eo psi_o>
    assert abs(lhs + np.conj(rhs)) < 1e-12 * abs(lhs)
    # the blocks read only the opposite parity: garbage on the output parity changes nothing
    junk = phi_e + 7.0 * psi_o
    a = oracle.dslash(dims, U, junk, 1)
    assert np.array_equal(a, oracle.dslash(dims, U, phi_e, 1))
    assert np.all(a[par == 0] == 0)


# ---------------------------------------------------------------- P2 M hermitian positive definite
def test_P2_M_hermitian_positive_definite(haar4, dense4):
    m = 0.1
    M, cols = _dense_M(D4, haar4, m)
    assert M.shape == (384, 384)                                  # configs[0]: "384x384"
    assert np.abs(M - M.conj().T).max() < 1e-13
    lam = np.linalg.eigvalsh(0.5 * (M + M.conj().T))
    assert lam.min() >= m * m - 1e-12
    # M is m^2 - D_eo D_oe built from the dense blocks of D (sign of the second term)
    par = np.repeat(qi.site_parity(D4), 3)
    Deo = dense4[np.ix_(par == 0, par == 1)]
    Doe = dense4[np.ix_(par == 1, par == 0)]
    assert np.abs(M - (m * m * np.eye(384) - Deo @ Doe)).max() < 1e-13
    # P7: ||D|| <= 8, and on Haar links the edge sits near (2 sqrt 7)^2 = 28
    top = lam.max() - m * m
    assert top <= 64.0
    assert 22.0 < top < 32.0


def test_P2_rayleigh_quotient_any_size():
    dims, m = DA, 0.07
    U = qi.gauge_field(dims, "haar", seed=3)
    v = qi.gaussian_source(dims, seed=5, parity=0)
    q = np.vdot(v, oracle.apply_M(dims, U, v, m))
    n2 = np.vdot(v, v).real
    assert abs(q.imag) < 1e-12 * abs(q.real)
    assert q.real >= m * m * n2


# ---------------------------------------------------------------- P3 free-field closed forms
def _plane_wave(dims, n, colour_vec):
    x = qi.site_coords(dims).astype(np.float64)
    p = np.array([2 * np.pi * n[0] / dims[0], 2 * np.pi * n[1] / dims[1],
                  2 * np.pi * n[2] / dims[2], (2 * n[3] + 1) * np.pi / dims[3]])
    return np.exp(1j * (x @ p))[:, None] * np.asarray(colour_vec)[None, :], p


def test_P3_free_spectrum_dense_4x4x4x4():
    m = 0.1
    U = qi.gauge_field(D4, "unit")
    M, _ = _dense_M(D4, U, m)
    lam = np.sort(np.linalg.eigvalsh(M))
    want = np.loadtxt(os.path.join(GOLDEN, "free_spectrum_4x4x4x4.txt"))
    expect = np.sort(np.concatenate([np.full(int(k), val) for val, k in want]))
    assert expect.size == 384
    assert np.abs(lam - expect).max() < 1e-12


@pytest.mark.parametrize("n", [(0, 0, 0, 0), (1, 0, 0, 0), (0, 2, 0, 1), (1, 1, 1, 2), (3, 5, 1, 7)])
def test_P3_plane_wave_eigenvector_of_M(n):
    dims, m = DA, 0.3
    U = qi.gauge_field(dims, "unit")
    phi, p = _plane_wave(dims, n, [0.3 - 0.2j, 1.0, -0.5j])
    phi[qi.site_parity(dims) == 1] = 0
    lam = m * m + 4 * np.sum(np.sin(p) ** 2)
    out = oracle.apply_M(dims, U, phi, m)
    assert np.abs(out - lam * phi).max() < 1e-12 * max(1.0, lam)


@pytest.mark.parametrize("n", [(0, 0, 0, 0), (1, 2, 0, 3), (2, 1, 1, 0)])
def test_P3b_pointwise_closed_form(n):
    """Unit links, phi = plane wave on all sites: (D phi)(x) = 2i (sum_mu eta_mu(x) sin p_mu) phi(x)."""
    dims = DA
    U = qi.gauge_field(dims, "unit")
    phi, p = _plane_wave(dims, n, [1.0, 2.0j, -0.7])
    x = qi.site_coords(dims)
    eta = np.stack([np.ones(len(x)), (-1.0) ** x[:, 0], (-1.0) ** (x[:, 0] + x[:, 1]),
                    (-1.0) ** (x[:, 0] + x[:, 1] + x[:, 2])], axis=1)
    expect = (2j * (eta @ np.sin(p)))[:, None] * phi
    out = oracle.dslash(dims, U, phi, -1)
    assert np.abs(out - expect).max() < 1e-12
    # each direction separately (p nonzero in one direction only is covered by the parametrisation;
    # here: the full operator equals the sum of its two parity blocks)
    assert np.array_equal(out, oracle.dslash(dims, U, phi, 0) + oracle.dslash(dims, U, phi, 1))


def test_P3c_constant_field_sees_only_the_time_seam():
    dims = DA
    U = qi.gauge_field(dims, "unit")
    vcol = np.array([1.0 + 0.5j, -2.0, 0.25j])
    phi = np.tile(vcol, (qi.volume(dims), 1))
    out = oracle.dslash(dims, U, phi, -1)
    x = qi.site_coords(dims)
    eta3 = (-1.0) ** (x[:, 0] + x[:, 1] + x[:, 2])
    expect = np.zeros_like(phi)
    last, first = x[:, 3] == dims[3] - 1, x[:, 3] == 0
    expect[last] = (-2.0 * eta3[last])[:, None] * vcol       # forward hop crosses the seam
    expect[first] = (+2.0 * eta3[first])[:, None] * vcol     # backward hop crosses the seam
    assert np.abs(out - expect).max() < 1e-14


def test_P3d_cg_terminates_in_4_iterations_on_the_4_eigenvalue_free_field():
    U = qi.gauge_field(D4, "unit")
    b = qi.gaussian_source(D4, seed=1, parity=0)
    x, info = oracle.cg(D4, U, b, 0.1, 1e-12, 50, history=True)
    assert info["converged"] and info["iters"] == 4
    h = np.sqrt(info["history"])
    assert np.all(h[:3] > 1e-2) and h[3] < 1e-13
    assert oracle.true_residual(D4, U, b, x, 0.1) < 1e-13


# ---------------------------------------------------------------- P6 point source (eta convention, seam side)
def _golden_table():
    rows = np.loadtxt(os.path.join(GOLDEN, "point_source_table.txt"))
    return [(tuple(int(c) for c in r[:4]), int(r[4]), int(r[5]), float(r[6])) for r in rows]


def test_P6_point_source_sign_table_unit_links():
    U = qi.gauge_field(D4, "unit")
    src = np.zeros((256, 3), dtype=np.complex128)
    src[_lex(D4, (1, 0, 0, 0)), 0] = 1.0
    out = oracle.dslash(D4, U, src, 0)
    expect = np.zeros_like(out)
    for x, _mu, _hop, val in _golden_table():
        expect[_lex(D4, x), 0] = val
    assert np.array_equal(out, expect)


def test_P6b_point_source_picks_link_columns(haar4):
    """Same source on Haar links: a forward hop of x reads column c of U_{x,mu}, a backward hop
    row c of U_{y,mu} conjugated (U^dagger) -- pins index order, dagger placement, link ownership."""
    U = haar4
    y, c = (1, 0, 0, 0), 1
    src = np.zeros((256, 3), dtype=np.complex128)
    src[_lex(D4, y), c] = 1.0
    out = oracle.dslash(D4, U, src, 0)
    expect = np.zeros_like(out)
    for x, mu, hop, val in _golden_table():
        if hop > 0:   # x = y - mu: value * U_{x,mu}[:, c]
            expect[_lex(D4, x)] = val * U[_lex(D4, x), mu][:, c]
        else:         # x = y + mu: value * conj(U_{y,mu}[c, :])
            expect[_lex(D4, x)] = val * np.conj(U[_lex(D4, y), mu][c, :])
    assert np.abs(out - expect).max() < 1e-15


# ---------------------------------------------------------------- P4 gauge covariance
def _gauge_transform(dims, U, g):
    """U'_{x,mu} = g(x) U_{x,mu} g(x+mu)^dagger (periodic), done with numpy only."""
    x = qi.site_coords(dims).astype(np.int64)
    Up = np.empty_like(U)
    for mu in range(4):
        xn = x.copy()
        xn[:, mu] = (xn[:, mu] + 1) % dims[mu]
        nbr = xn[:, 0] + dims[0] * (xn[:, 1] + dims[1] * (xn[:, 2] + dims[2] * xn[:, 3]))
        Up[:, mu] = np.einsum("nij,njk,nlk->nil", g, U[:, mu], g[nbr].conj())
    return Up


def test_P4_gauge_covariance_dslash_and_cg():
    dims, m = DA, 0.2
    v = qi.volume(dims)
    U = qi.gauge_field(dims, "haar", seed=0)
    g = qi.haar_su3(v, seed=2)
    Up = _gauge_transform(dims, U, g)
    phi = qi.gaussian_spinor(dims, seed=4)
    gphi = np.einsum("nij,nj->ni", g, phi)
    lhs = oracle.dslash(dims, Up, gphi, -1)
    rhs = np.einsum("nij,nj->ni", g, oracle.dslash(dims, U, phi, -1))
    assert np.abs(lhs - rhs).max() < 1e-13
    b = qi.gaussian_source(dims, seed=1, parity=0)
    gb = np.einsum("nij,nj->ni", g, b)
    x1, i1 = oracle.cg(dims, U, b, m, 1e-10, 2000)
    x2, i2 = oracle.cg(dims, Up, gb, m, 1e-10, 2000)
    assert i1["converged"] and i2["converged"] and abs(i1["iters"] - i2["iters"]) <= 1
    gx1 = np.einsum("nij,nj->ni", g, x1)
    assert np.linalg.norm(x2 - gx1) < 1e-7 * np.linalg.norm(gx1)


# ---------------------------------------------------------------- P5 dense brute force (configs[0])
def test_P5_cg_matches_dense_solve_4x4x4x4(haar4):
    m, tol = 0.1, 1e-10
    b = qi.gaussian_source(D4, seed=1, parity=0)
    M, cols = _dense_M(D4, haar4, m)
    x_dense = np.linalg.solve(M, b.reshape(-1)[cols])
    lam = np.linalg.eigvalsh(0.5 * (M + M.conj().T))
    kappa = lam.max() / lam.min()
    x, info = oracle.cg(D4, haar4, b, m, tol, 10000)
    assert info["converged"]
    assert info["rel_resid"] <= tol
    err = np.linalg.norm(x.reshape(-1)[cols] - x_dense) / np.linalg.norm(x_dense)
    assert err <= kappa * tol
    assert np.all(x[qi.site_parity(D4) == 1] == 0)
    assert oracle.true_residual(D4, haar4, b, x, m) <= 2 * tol
    # one M application against the dense matrix
    assert np.abs(oracle.apply_M(D4, haar4, b, m).reshape(-1)[cols] - M @ b.reshape(-1)[cols]).max() < 1e-12


# ---------------------------------------------------------------- P8 large mass, degenerate cases
def test_P8_large_mass_limit():
    dims, m = DA, 100.0
    U = qi.gauge_field(dims, "haar", seed=0)
    b = qi.gaussian_source(dims, seed=1, parity=0)
    x, info = oracle.cg(dims, U, b, m, 1e-10, 100)
    assert info["converged"] and info["iters"] <= 6
    assert np.linalg.norm(x - b / m ** 2) <= 1e-2 * np.linalg.norm(b / m ** 2)


def test_cg_degenerate_arguments(haar4):
    zero = np.zeros((256, 3), dtype=np.complex128)
    x, info = oracle.cg(D4, haar4, zero, 0.1, 1e-10, 10)
    assert info["converged"] and info["iters"] == 0 and not x.any()
    b = qi.gaussian_source(D4, seed=1, parity=0)
    x, info = oracle.cg(D4, haar4, b, 0.1, 1e-10, 0)
    assert not info["converged"] and info["status"] == 4 and info["iters"] == 0 and not x.any()
    x, info = oracle.cg(D4, haar4, b, 0.1, 1e-10, 7)
    assert info["status"] == 4 and info["iters"] == 7


# ---------------------------------------------------------------- single-site entry, fp32 variant
def test_site_entry_equals_definition_and_fp32_variant_tracks_fp64():
    dims = DA
    U = qi.gauge_field(dims, "haar", seed=0)
    phi = qi.gaussian_spinor(dims, seed=9)
    full = oracle.dslash(dims, U, phi, -1)
    for x in [(0, 0, 0, 0), (3, 5, 1, 7), (2, 0, 1, 0), (1, 5, 0, 7)]:
        assert np.array_equal(oracle.dslash_site(dims, U, phi, x), full[_lex(dims, x)])
    out32 = oracle.dslash(dims, U.astype(np.complex64), phi.astype(np.complex64), -1)
    assert out32.dtype == np.complex64
    scale = np.abs(full).max()
    assert np.abs(out32 - full).max() < 2e-6 * scale * 4
    b = qi.gaussian_source(dims, seed=1, parity=0)
    x64, i64 = oracle.cg(dims, U, b, 0.5, 1e-5, 500)
    x32, i32 = oracle.cg(dims, U.astype(np.complex64), b.astype(np.complex64), 0.5, 1e-5, 500)
    assert i32["converged"] and abs(i32["iters"] - i64["iters"]) <= 1
    assert np.linalg.norm(x32 - x64) < 1e-4 * np.linalg.norm(x64)

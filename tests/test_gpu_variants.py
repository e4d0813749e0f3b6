"""GPU parity of the paper's Dslash variants and of
the mixed-precision solver against oracle/variants.py, through the C-ABI, on the same seeded inputs.

  two-row links    the kernel rebuilds row 2 = conj(row 0 x row 1) from the STORED rows, so the
                   reference is the oracle applied to reconstruct12(compress12(U as stored))
  temporal gauge   device transform vs oracle transform (U', g); the TG kernel (time links with
                   x3 != 0 never read) vs the oracle on the fixed links; covariance back to D[U]
  several vectors  every vector of a multi call vs the oracle applied to it alone; n lock-step CG
                   solves vs n oracle solves
  mixed precision  defect-correction CG vs oracle.variants.mixed_cg: fp64 true residual <= tol

Tolerances as in test_gpu_parity.py (north_star): 1e-13 (fp64), 2e-6 (fp32), per-site measure R10."""
import contextlib

import numpy as np
import pytest

import oracle
import oracle.variants as ov
import qcd_inputs
from util import DSLASH_TOL, dslash_rel_err, iters_close

pytestmark = pytest.mark.gpu

LATTICES = [
    ((4, 4, 4, 4), "haar", None),
    ((4, 6, 2, 8), "haar", None),            # N2 = 2
    ((8, 4, 6, 10), "near_identity", 0.5),   # several blocks and a ragged tail
    ((12, 2, 2, 4), "haar", None),           # time slices shorter than a warp: x3 varies inside a warp
    ((16, 16, 16, 16), "near_identity", 0.3),
]


@pytest.fixture(scope="module")
def q():
    import paper_2502_03249_b200 as pkg
    return pkg


def _rounded(a, prec):
    return a if prec == 64 else a.astype(np.complex64).astype(np.complex128)


def _full_dslash(ctx, q, fU, phi):
    """D phi on the full lattice through qcd_dslash_eo + qcd_dslash_oe."""
    fphi = ctx.field(q.QCD_SPINOR_FULL).upload(phi)
    fout = ctx.field(q.QCD_SPINOR_FULL)
    fout.buf.zero_()
    ctx.qcd_dslash_eo(fU, fout, fphi)
    ctx.qcd_dslash_oe(fU, fout, fphi)
    return fout.download()


def _check_full(dims, got, ref, tol, what=""):
    par = qcd_inputs.site_parity(dims)
    for p in (0, 1):
        err = dslash_rel_err(got[par == p], ref[par == p])
        assert err <= tol, (what, p, err)


# ------------------------------------------------------------------------------------------
# two-row links
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims,links,eps", LATTICES)
def test_two_row_links(q, dims, links, eps, prec):
    ctx = q.Context(dims, prec)
    U = qcd_inputs.gauge_field(dims, links, seed=0, eps=eps)
    phi = qcd_inputs.gaussian_spinor(dims, seed=1)
    Ur, phir = _rounded(U, prec), _rounded(phi, prec)
    Urec = ov.reconstruct12(ov.compress12(Ur))               # what a two-row field represents

    f12 = ctx.field(q.QCD_GAUGE_2ROW).upload(U)
    back = f12.download().astype(np.complex128)
    assert np.array_equal(back[:, :, :2, :], Ur[:, :, :2, :])            # stored rows: exact
    eps_m = 1e-15 if prec == 64 else 5e-7
    assert np.max(np.abs(back - Urec)) <= 8 * eps_m                       # rebuilt row
    assert np.max(np.abs(Urec - Ur)) <= (1e-14 if prec == 64 else 1e-6)   # the inputs are SU(3)

    # device-side compression gives the same planes as the direct upload
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    g12 = ctx.field(q.QCD_GAUGE_2ROW)
    ctx.qcd_gauge_compress(fU, g12)
    import torch
    torch.cuda.synchronize()
    assert torch.equal(g12.buf, f12.buf)

    got = _full_dslash(ctx, q, f12, phi)
    _check_full(dims, got, oracle.dslash(dims, Urec, phir, -1), DSLASH_TOL[prec], "two-row vs oracle on rebuilt links")
    if prec == 64:      # and the rebuilt links are the links: same answer as Eq. (1) on U itself
        _check_full(dims, got, oracle.dslash(dims, U, phi, -1), DSLASH_TOL[64], "two-row vs oracle on full links")
    ctx.close()


@pytest.mark.parametrize("prec", [64, 32])
def test_two_row_apply_M_and_cg(q, prec):
    dims, m = (8, 4, 6, 10), 0.1
    tol = 1e-10 if prec == 64 else 1e-5
    ctx = q.Context(dims, prec)
    U = qcd_inputs.gauge_field(dims, "near_identity", seed=0, eps=0.5)
    b = qcd_inputs.gaussian_source(dims, seed=1)
    Ur, br = _rounded(U, prec), _rounded(b, prec)
    Urec = ov.reconstruct12(ov.compress12(Ur))
    par = qcd_inputs.site_parity(dims)
    f12 = ctx.field(q.QCD_GAUGE_2ROW).upload(U)
    fb = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
    fx = ctx.field(q.QCD_SPINOR_EVEN)
    ctx.qcd_apply_M(f12, fx, fb, m)
    got = fx.download()
    assert dslash_rel_err(got[par == 0], oracle.apply_M(dims, Urec, br, m)[par == 0]) <= DSLASH_TOL[prec]
    info = ctx.qcd_cg_solve(f12, fb, fx, m, tol, 5000)
    x = fx.download().astype(np.complex128)
    _, oinfo = oracle.cg(dims, Urec.astype(ctx.cdtype), br.astype(ctx.cdtype), m, tol, 5000)
    assert info["converged"] and iters_close(info["iters"], oinfo["iters"]), (info, oinfo)
    assert oracle.true_residual(dims, Urec, br, x, m) <= tol * (1.0 if prec == 64 else 1.5)
    ctx.close()


# ------------------------------------------------------------------------------------------
# temporal gauge (reading R20)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims,links,eps", LATTICES)
def test_temporal_gauge_transform_fp64(q, dims, links, eps):
    ctx = q.Context(dims, 64)
    U = qcd_inputs.gauge_field(dims, links, seed=0, eps=eps)
    phi = qcd_inputs.gaussian_spinor(dims, seed=1)
    Ufix_ref, g_ref = ov.temporal_gauge(dims, U)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    fUf = ctx.field(q.QCD_GAUGE)
    fg = ctx.field(q.QCD_COLOUR_MATRIX)
    ctx.qcd_gauge_fix_temporal(fU, fUf, fg)
    g = fg.download()
    Ufix = fUf.download()
    assert np.max(np.abs(g - g_ref)) <= 1e-13
    assert np.max(np.abs(Ufix - Ufix_ref)) <= 1e-13
    x3 = qcd_inputs.site_coords(dims)[:, 3]
    assert np.array_equal(Ufix[x3 != 0, 3], np.broadcast_to(np.eye(3), Ufix[x3 != 0, 3].shape))   # exactly 1
    assert np.max(np.abs(Ufix[x3 == 0, 3] - np.eye(3))) > 1e-3                                      # the Polyakov loop is not

    # rotation g phi, and back
    fphi = ctx.field(q.QCD_SPINOR_FULL).upload(phi)
    frot = ctx.field(q.QCD_SPINOR_FULL)
    ctx.qcd_spinor_rotate(fg, frot, fphi, dagger=False)
    rot = frot.download()
    assert np.max(np.abs(rot - ov.rotate_spinor(g_ref, phi))) <= 1e-13
    ctx.qcd_spinor_rotate(fg, frot, frot, dagger=True)              # in place
    assert np.max(np.abs(frot.download() - phi)) <= 1e-13

    # the TG kernel on the fixed links (it never reads the unit time links) ...
    got = _full_dslash(ctx, q, fUf, rot)
    _check_full(dims, got, oracle.dslash(dims, Ufix_ref, ov.rotate_spinor(g_ref, phi), -1), DSLASH_TOL[64], "TG kernel")
    # ... is gauge covariant: g^dagger D[U'] g phi = D[U] phi
    fgot = ctx.field(q.QCD_SPINOR_FULL).upload(got)
    ctx.qcd_spinor_rotate(fg, fgot, fgot, dagger=True)
    _check_full(dims, fgot.download(), oracle.dslash(dims, U, phi, -1), DSLASH_TOL[64], "covariance")

    # two rows + temporal gauge: the paper's 126-real kernel
    f12 = ctx.field(q.QCD_GAUGE_2ROW)
    ctx.qcd_gauge_compress(fUf, f12)
    got12 = _full_dslash(ctx, q, f12, rot)
    _check_full(dims, got12, oracle.dslash(dims, Ufix_ref, ov.rotate_spinor(g_ref, phi), -1), DSLASH_TOL[64], "two-row + TG")
    ctx.close()


def test_temporal_gauge_kernel_does_not_read_unit_links(q):
    """Poison the time links with x3 != 0 after marking the field: the result must not change."""
    dims = (8, 4, 6, 10)
    ctx = q.Context(dims, 64)
    U = qcd_inputs.gauge_field(dims, "haar", seed=0)
    phi = qcd_inputs.gaussian_spinor(dims, seed=1)
    Ufix, _ = ov.temporal_gauge(dims, U)
    x3 = qcd_inputs.site_coords(dims)[:, 3]
    poisoned = Ufix.copy()
    poisoned[x3 != 0, 3] = np.nan
    for kind in (q.QCD_GAUGE, q.QCD_GAUGE_2ROW):
        f = ctx.field(kind).upload(poisoned)
        ctx.qcd_gauge_set_temporal_unit(f, True)
        got = _full_dslash(ctx, q, f, phi)
        assert np.isfinite(got).all()
        _check_full(dims, got, oracle.dslash(dims, Ufix, phi, -1), DSLASH_TOL[64], kind)
        ctx.qcd_gauge_set_temporal_unit(f, False)
        assert not np.isfinite(_full_dslash(ctx, q, f, phi)).all()
    ctx.close()


@pytest.mark.parametrize("dims,links,eps", LATTICES[1:4])
def test_temporal_gauge_fp32(q, dims, links, eps):
    """fp32: the links fixed by the oracle in fp64, rounded, uploaded and marked; reference = oracle on
    the rounded links with the unit time links exactly 1."""
    ctx = q.Context(dims, 32)
    U = qcd_inputs.gauge_field(dims, links, seed=0, eps=eps)
    phi = qcd_inputs.gaussian_spinor(dims, seed=1)
    Ufix, _ = ov.temporal_gauge(dims, U)
    x3 = qcd_inputs.site_coords(dims)[:, 3]
    Ufix[x3 != 0, 3] = np.eye(3)
    Ur, phir = _rounded(Ufix, 32), _rounded(phi, 32)
    for kind in (q.QCD_GAUGE, q.QCD_GAUGE_2ROW):
        f = ctx.field(kind).upload(Ufix)
        ctx.qcd_gauge_set_temporal_unit(f, True)
        ref_links = Ur if kind == q.QCD_GAUGE else ov.reconstruct12(ov.compress12(Ur))
        _check_full(dims, _full_dslash(ctx, q, f, phi), oracle.dslash(dims, ref_links, phir, -1), DSLASH_TOL[32], kind)
    ctx.close()


def test_temporal_gauge_cg_returns_rotated_solution(q):
    """M[U'] x' = g b  is solved by  x' = g x  (SURVEY.md pin P4)."""
    dims, m, tol = (8, 4, 6, 10), 0.1, 1e-10
    ctx = q.Context(dims, 64)
    U = qcd_inputs.gauge_field(dims, "near_identity", seed=0, eps=0.5)
    b = qcd_inputs.gaussian_source(dims, seed=1)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    fUf, fg = ctx.field(q.QCD_GAUGE), ctx.field(q.QCD_COLOUR_MATRIX)
    ctx.qcd_gauge_fix_temporal(fU, fUf, fg)
    f12 = ctx.field(q.QCD_GAUGE_2ROW)
    ctx.qcd_gauge_compress(fUf, f12)
    fb = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
    fbr, fx = ctx.field(q.QCD_SPINOR_EVEN), ctx.field(q.QCD_SPINOR_EVEN)
    ctx.qcd_spinor_rotate(fg, fbr, fb)
    info = ctx.qcd_cg_solve(f12, fbr, fx, m, tol, 5000)
    ctx.qcd_spinor_rotate(fg, fx, fx, dagger=True)
    x = fx.download()
    _, oinfo = oracle.cg(dims, U, b, m, tol, 5000)
    assert info["converged"] and iters_close(info["iters"], oinfo["iters"])
    assert oracle.true_residual(dims, U, b, x, m) <= tol
    ctx.close()


# ------------------------------------------------------------------------------------------
# several vectors per link load (NMULTI)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7, 8])
@pytest.mark.parametrize("kind_name,tg", [("QCD_GAUGE", False), ("QCD_GAUGE_2ROW", True)])
def test_dslash_multi(q, n, prec, kind_name, tg):
    dims = (8, 4, 6, 10)
    kind = getattr(q, kind_name)
    ctx = q.Context(dims, prec)
    U = qcd_inputs.gauge_field(dims, "haar", seed=0)
    if tg:
        U, _ = ov.temporal_gauge(dims, U)
        U[qcd_inputs.site_coords(dims)[:, 3] != 0, 3] = np.eye(3)
    Ur = _rounded(U, prec)
    if kind == q.QCD_GAUGE_2ROW:
        Ur = ov.reconstruct12(ov.compress12(Ur))
    fU = ctx.field(kind).upload(U)
    ctx.qcd_gauge_set_temporal_unit(fU, tg)
    phis = [qcd_inputs.gaussian_spinor(dims, seed=10 + i) for i in range(n)]
    par = qcd_inputs.site_parity(dims)
    fin = [ctx.field(q.QCD_SPINOR_FULL).upload(p) for p in phis]
    fout = [ctx.field(q.QCD_SPINOR_FULL) for _ in range(n)]
    for f in fout:
        f.buf.zero_()
    refs = ov.dslash_multi(dims, Ur, [_rounded(p, prec) for p in phis], -1)
    first = None
    for kernel in (0, 4, 5, 6, 7, 8, 9, 10):  # library's choice; staged (links through shared memory); register kernel; pair kernel at two register caps; register kernel with the x0-x1 tile; rolled direction loop; bulk-copy kernel (not applicable on this lattice: falls back)
        ctx.qcd_set_dslash_variant(kernel)
        for f in fout:
            f.buf.zero_()
        ctx.qcd_dslash_eo_multi(fU, fout, fin)
        ctx.qcd_dslash_oe_multi(fU, fout, fin)
        got = [f.download() for f in fout]
        for i in range(n):
            for p in (0, 1):
                assert dslash_rel_err(got[i][par == p], refs[i][par == p]) <= DSLASH_TOL[prec], (kernel, i, p)
        if first is None:
            first = got
        else:                        # same FMAs in the same order per site, whichever way the operands arrive
            assert all(np.array_equal(a, b) for a, b in zip(first, got)), kernel
    ctx.close()


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims,chunk", [((32, 8, 2, 4), 0), ((16, 16, 4, 2), 1), ((16, 16, 4, 2), 2), ((64, 4, 2, 2), 0), ((256, 2, 2, 2), 0),
                                        ((128, 2, 4, 2), 0), ((32, 16, 4, 6), 0), ((16, 16, 16, 16), 0)])
def test_dslash_bulk_copy_kernel_on_row_aligned_lattices(q, dims, chunk, prec):
    """The warp-specialised bulk-copy kernel (variant 10; producer warps feed a shared-memory ring through the TMA engine, consumer
    warps compute) needs a block's 128 sites to be whole x0-rows of one (x2, x3) plane.  Rows of 8 ... 128 sites (16, 8, 4, 2, 1 rows per
    block), x1 wraps INSIDE a block (two runs per plane, the 1-d bulk copies) and at its edge, x2 / x3 extents of 2 (forward and backward
    neighbour are the same site), with and without traversal chunking; every link storage (full, two-row, two-row in temporal gauge: unit
    links are neither copied nor multiplied) and 2 ... 8 vectors (odd counts: one consumer half holds one vector fewer).
    Bitwise equal to the register kernel, equal to the oracle within tolerance, and nothing is written outside the outputs."""
    U = qcd_inputs.gauge_field(dims, "haar", seed=0)
    Ufix, _ = ov.temporal_gauge(dims, U)
    Ufix[qcd_inputs.site_coords(dims)[:, 3] != 0, 3] = np.eye(3)
    par = qcd_inputs.site_parity(dims)
    nmax = 8
    ctx = q.Context(dims, prec, nrhs=nmax)
    ctx.qcd_set_traversal_chunk(chunk)
    phis = [qcd_inputs.gaussian_spinor(dims, seed=50 + i) for i in range(nmax)]
    fin = [ctx.field(q.QCD_SPINOR_FULL).upload(p) for p in phis]
    fout = [ctx.field(q.QCD_SPINOR_FULL) for _ in range(nmax)]
    for name, kind, Uh, tg in (("full", q.QCD_GAUGE, U, False), ("tworow", q.QCD_GAUGE_2ROW, U, False), ("tworow+tg", q.QCD_GAUGE_2ROW, Ufix, True)):
        fU = ctx.field(kind).upload(Uh)
        ctx.qcd_gauge_set_temporal_unit(fU, tg)
        Ur = _rounded(Uh, prec)
        if kind == q.QCD_GAUGE_2ROW:
            Ur = ov.reconstruct12(ov.compress12(Ur))
        refs = ov.dslash_multi(dims, Ur, [_rounded(p, prec) for p in phis], -1)
        for n in (2, 3, 5, 8):
            res = {}
            for kernel in (5, 10):
                ctx.qcd_set_dslash_variant(kernel)
                for f in fout:
                    f.buf.fill_(255)
                ctx.qcd_dslash_eo_multi(fU, fout[:n], fin[:n])
                ctx.qcd_dslash_oe_multi(fU, fout[:n], fin[:n])
                res[kernel] = [f.download() for f in fout[:n]]
                assert all(bool((f.buf == 255).all().item()) for f in fout[n:]), (name, n, kernel)      # the other fields are untouched
            for i in range(n):
                for p in (0, 1):
                    assert dslash_rel_err(res[10][i][par == p], refs[i][par == p]) <= DSLASH_TOL[prec], (name, n, i, p)
            assert all(np.array_equal(a, b) for a, b in zip(res[5], res[10])), (name, n)
    ctx.qcd_set_dslash_variant(0)
    ctx.close()


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims,chunk", [((32, 8, 2, 4), 0), ((16, 16, 4, 2), 1), ((16, 16, 4, 2), 2), ((64, 4, 2, 2), 0)])
def test_dslash_tile_and_pair_kernels_on_row_aligned_lattices(q, dims, chunk, prec):
    """The register kernel with the x0 / x1 neighbour rows of a block in shared memory (variant 8) needs a block of 128
    sites to be whole x0-rows of one (x2, x3) plane; (8,4,6,10) of test_dslash_multi is not such a lattice and runs the
    library's choice there.  Here it does run: rows of 16, 8 and 32 sites, x1 and x2 wraps inside a block's neighbourhood,
    with and without traversal chunking, plain Dslash (MODE 0) and, through the lock-step CG, the reducing kernel (MODE 2).
    Bitwise equal to the library's choice, and equal to the oracle within tolerance."""
    U = qcd_inputs.gauge_field(dims, "haar", seed=0)
    par = qcd_inputs.site_parity(dims)
    for n in (4, 8):
        ctx = q.Context(dims, prec, nrhs=n)
        ctx.qcd_set_traversal_chunk(chunk)
        fU = ctx.field(q.QCD_GAUGE).upload(U)
        phis = [qcd_inputs.gaussian_spinor(dims, seed=30 + i) for i in range(n)]
        fin = [ctx.field(q.QCD_SPINOR_FULL).upload(p) for p in phis]
        fout = [ctx.field(q.QCD_SPINOR_FULL) for _ in range(n)]
        refs = ov.dslash_multi(dims, _rounded(U, prec), [_rounded(p, prec) for p in phis], -1)
        first = None
        for kernel in (0, 8, 6, 5, 9):
            ctx.qcd_set_dslash_variant(kernel)
            for f in fout:
                f.buf.fill_(255)
            ctx.qcd_dslash_eo_multi(fU, fout, fin)
            ctx.qcd_dslash_oe_multi(fU, fout, fin)
            got = [f.download() for f in fout]
            for i in range(n):
                for p in (0, 1):
                    assert dslash_rel_err(got[i][par == p], refs[i][par == p]) <= DSLASH_TOL[prec], (n, kernel, i, p)
            if first is None:
                first = got
            else:
                assert all(np.array_equal(a, b) for a, b in zip(first, got)), (n, kernel)
        # MODE 2 through the lock-step CG: same iteration counts and solutions whichever kernel applies M
        m, tol = 0.3, (1e-10 if prec == 64 else 1e-5)
        srcs = [qcd_inputs.gaussian_source(dims, seed=40 + i) for i in range(n)]
        fb = [ctx.field(q.QCD_SPINOR_EVEN).upload(s_) for s_ in srcs]
        fx = [ctx.field(q.QCD_SPINOR_EVEN) for _ in range(n)]
        sols = {}
        for kernel in (0, 8):
            ctx.qcd_set_dslash_variant(kernel)
            infos = ctx.qcd_cg_solve_multi(fU, fb, fx, m, tol, 5000)
            assert all(i["converged"] for i in infos)
            sols[kernel] = ([i["iters"] for i in infos], [f.download() for f in fx])
        assert sols[0][0] == sols[8][0]
        for a, b in zip(sols[0][1], sols[8][1]):
            assert np.allclose(a, b, rtol=0, atol=(1e-12 if prec == 64 else 1e-5) * np.abs(a).max())
        _, oinfo = oracle.cg(dims, _rounded(U, prec).astype(ctx.cdtype), _rounded(srcs[0], prec).astype(ctx.cdtype), m, tol, 5000)
        assert iters_close(sols[8][0][0], oinfo["iters"])
        ctx.close()


@pytest.mark.parametrize("prec,n", [(64, 2), (64, 3), (64, 8), (32, 4)])
def test_cg_multi_is_n_independent_solves(q, prec, n):
    dims, m = (8, 4, 6, 10), 0.1
    tol = 1e-10 if prec == 64 else 1e-5
    ctx = q.Context(dims, prec, nrhs=n)
    U = qcd_inputs.gauge_field(dims, "near_identity", seed=0, eps=0.5)
    Ur = _rounded(U, prec)
    bs = [qcd_inputs.gaussian_source(dims, seed=20 + i) * (10.0 ** (i - 1)) for i in range(n)]
    bs[1] = np.zeros_like(bs[1])                                  # a zero source: converged at once, x = 0
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    fb = [ctx.field(q.QCD_SPINOR_EVEN).upload(b) for b in bs]
    fx = [ctx.field(q.QCD_SPINOR_EVEN) for _ in range(n)]
    infos = ctx.qcd_cg_solve_multi(fU, fb, fx, m, tol, 5000)
    _, oinfos = ov.cg_multi(dims, Ur.astype(ctx.cdtype), [_rounded(b, prec).astype(ctx.cdtype) for b in bs], m, tol, 5000)
    single = q.Context(dims, prec)
    single.qcd_set_cg_loop(1)            # kernel-by-kernel: the loop the lock-step solve uses
    sU = single.field(q.QCD_GAUGE).upload(U)
    for i in range(n):
        x = fx[i].download().astype(np.complex128)
        assert infos[i]["converged"], (i, infos[i])
        assert iters_close(infos[i]["iters"], oinfos[i]["iters"]), (i, infos[i], oinfos[i])
        if not bs[i].any():
            assert infos[i]["iters"] == 0 and not x.any()
            continue
        assert oracle.true_residual(dims, Ur, _rounded(bs[i], prec), x, m) <= tol * (1.0 if prec == 64 else 1.5), i
        # identical to the single-vector solve: same arithmetic, same reduction order
        sb, sx = single.field(q.QCD_SPINOR_EVEN).upload(bs[i]), single.field(q.QCD_SPINOR_EVEN)
        sinfo = single.qcd_cg_solve(sU, sb, sx, m, tol, 5000)
        assert sinfo["iters"] == infos[i]["iters"], (i, sinfo, infos[i])
        assert np.allclose(sx.download(), fx[i].download(), rtol=0, atol=1e-12 * np.max(np.abs(x)) if prec == 64 else 1e-5 * np.max(np.abs(x)))
    single.close()
    ctx.close()


def test_multi_argument_errors(q):
    dims = (4, 4, 4, 4)
    ctx = q.Context(dims, 64)            # workspace for ONE right-hand side only
    fU = ctx.field(q.QCD_GAUGE).upload(qcd_inputs.gauge_field(dims, "haar", seed=0))
    fb = [ctx.field(q.QCD_SPINOR_EVEN).upload(qcd_inputs.gaussian_source(dims, seed=i)) for i in range(2)]
    fx = [ctx.field(q.QCD_SPINOR_EVEN) for _ in range(2)]
    with pytest.raises(q.QcdError) as e:
        ctx.qcd_cg_solve_multi(fU, fb, fx, 0.1, 1e-8, 100)
    assert e.value.status == q.QCD_EINVAL and "workspace" in str(e.value)
    with pytest.raises(q.QcdError):
        ctx.qcd_cg_solve_multi(fU, fb, [fx[0], fx[0]], 0.1, 1e-8, 100)       # aliased solutions
    fo = [ctx.field(q.QCD_SPINOR_ODD) for _ in range(9)]
    with pytest.raises(q.QcdError):
        ctx.qcd_dslash_oe_multi(fU, fo, [fb[0]] * 9)                          # n > QCD_MAX_RHS
    with pytest.raises(q.QcdError):
        ctx.qcd_dslash_eo_multi(fU, fx, fb)                                   # parity mismatch
    ctx.close()


# ------------------------------------------------------------------------------------------
# precision conversion and mixed-precision defect-correction CG (reading R21)
# ------------------------------------------------------------------------------------------
def test_field_convert_rounds_to_nearest(q):
    dims = (8, 4, 6, 10)
    c64, c32 = q.Context(dims, 64), q.Context(dims, 32)
    U = qcd_inputs.gauge_field(dims, "haar", seed=0)
    for kind in (q.QCD_GAUGE, q.QCD_GAUGE_2ROW):
        f64 = c64.field(kind).upload(U)
        f32 = c32.field(kind)
        c64.qcd_field_convert(f32, f64)
        direct = c32.field(kind).upload(U)          # host-side rounding by numpy astype
        import torch
        torch.cuda.synchronize()
        assert torch.equal(f32.buf, direct.buf)
    c64.close(); c32.close()


@pytest.mark.parametrize("dims,links,eps,m,tol", [
    ((8, 4, 6, 10), "haar", None, 0.1, 1e-10),
    ((8, 8, 8, 8), "haar", None, 0.05, 1e-9),
    ((16, 16, 16, 16), "near_identity", 0.3, 0.05, 1e-10),
])
def test_mixed_precision_cg(q, dims, links, eps, m, tol):
    inner_tol, maxiter = 1e-3, 20000
    c64, c32 = q.Context(dims, 64), q.Context(dims, 32)
    U = qcd_inputs.gauge_field(dims, links, seed=0, eps=eps)
    b = qcd_inputs.gaussian_source(dims, seed=1)
    U64 = c64.field(q.QCD_GAUGE).upload(U)
    U32 = c32.field(q.QCD_GAUGE)
    c64.qcd_field_convert(U32, U64)
    fb, fx = c64.field(q.QCD_SPINOR_EVEN).upload(b), c64.field(q.QCD_SPINOR_EVEN)
    rhs32, e32 = c32.field(q.QCD_SPINOR_EVEN), c32.field(q.QCD_SPINOR_EVEN)
    info = c64.qcd_cg_solve_mixed(c32, U64, U32, fb, fx, rhs32, e32, m, tol, inner_tol, maxiter)
    x = fx.download()
    xo, oinfo = ov.mixed_cg(dims, U, b, m, tol, inner_tol, maxiter)
    assert info["converged"] and oinfo["converged"], (info, oinfo)
    true = oracle.true_residual(dims, U, b, x, m)
    assert true <= tol, true                                             # north_star: fp64 true residual <= tol
    assert abs(true - info["true_resid"]) <= 1e-3 * tol + 1e-14          # the device-side residual is the true one
    assert abs(info["outer"] - oinfo["outer"]) <= 1, (info, oinfo)
    assert iters_close(info["inner_iters"], oinfo["inner_iters"]) or abs(info["outer"] - oinfo["outer"]) == 1, (info, oinfo)
    assert info["m_applications_fp64"] == info["outer"]
    # the same x as the oracle's up to the conditioning of M:  |dx| / |x| <= kappa * tol, kappa <= (m^2 + 64) / m^2
    kappa = (m * m + 64.0) / (m * m)
    assert np.linalg.norm(x - xo) / np.linalg.norm(xo) <= kappa * tol
    # and cheaper than it looks: the fp64 work is `outer` operator applications
    assert info["outer"] <= 12
    c64.close(); c32.close()


def test_mixed_zero_source_and_budget(q):
    dims = (4, 4, 4, 4)
    c64, c32 = q.Context(dims, 64), q.Context(dims, 32)
    U = qcd_inputs.gauge_field(dims, "haar", seed=0)
    U64 = c64.field(q.QCD_GAUGE).upload(U)
    U32 = c32.field(q.QCD_GAUGE).upload(U)
    fb, fx = c64.field(q.QCD_SPINOR_EVEN), c64.field(q.QCD_SPINOR_EVEN)
    fb.buf.zero_()
    fx.buf.fill_(7)
    rhs32, e32 = c32.field(q.QCD_SPINOR_EVEN), c32.field(q.QCD_SPINOR_EVEN)
    info = c64.qcd_cg_solve_mixed(c32, U64, U32, fb, fx, rhs32, e32, 0.1, 1e-10, 1e-3, 100)
    assert info["converged"] and info["outer"] == 0 and not fx.download().any()
    fb.upload(qcd_inputs.gaussian_source(dims, seed=1))
    info = c64.qcd_cg_solve_mixed(c32, U64, U32, fb, fx, rhs32, e32, 0.1, 1e-10, 1e-3, 10)     # budget of 10 inner iterations
    assert info["status"] == q.QCD_ENOTCONVERGED and not info["converged"] and info["inner_iters"] == 10
    c64.close(); c32.close()


# ------------------------------------------------------------------------------------------
# solver loop on small lattices: CUDA-graph replay
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", [64, 32])
def test_cg_graph_replay_matches_plain_loop(q, prec):
    """On a non-default stream qcd_cg_solve replays a captured graph of 16 iterations; on the legacy
    default stream it enqueues kernel by kernel.  Same kernels, same order: identical iteration count
    and bitwise identical solution; both match the oracle."""
    import torch
    dims, m = (16, 16, 16, 16), 0.05
    tol = 1e-10 if prec == 64 else 1e-5
    U = qcd_inputs.gauge_field(dims, "near_identity", seed=0, eps=0.3)
    b = qcd_inputs.gaussian_source(dims, seed=1)
    res = []
    for use_stream in (False, True):
        stream = torch.cuda.Stream() if use_stream else None
        with (torch.cuda.stream(stream) if use_stream else contextlib.nullcontext()):
            ctx = q.Context(dims, prec, stream=stream)
            ctx.qcd_set_cg_loop(2 if use_stream else 1)      # graph replay / kernel-by-kernel (not the persistent kernel)
            fU = ctx.field(q.QCD_GAUGE).upload(U)
            fb = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
            fx = ctx.field(q.QCD_SPINOR_EVEN)
            n0 = ctx.qcd_launch_count()
            info = ctx.qcd_cg_solve(fU, fb, fx, m, tol, 10000)
            launches = ctx.qcd_launch_count() - n0
            assert ctx.qcd_last_cg_loop() == (2 if use_stream else 1)     # the loop that ran is the one this test is about
            res.append((info, fx.download(), launches))
            # maxiter that is not a multiple of the graph length: stops exactly there
            info2 = ctx.qcd_cg_solve(fU, fb, fx, m, 1e-300, 37)
            assert info2["iters"] == 37 and not info2["converged"] and info2["status"] == q.QCD_ENOTCONVERGED
            ctx.close()
    (i0, x0, l0), (i1, x1, l1) = res
    assert i0["converged"] and i1["converged"] and i0["iters"] == i1["iters"]
    assert np.array_equal(x0, x1)
    assert l1 >= 4 * i1["iters"] and l0 >= 4 * i0["iters"]
    _, oinfo = oracle.cg(dims, _rounded(U, prec).astype(x0.dtype), _rounded(b, prec).astype(x0.dtype), m, tol, 10000)
    assert iters_close(i1["iters"], oinfo["iters"])
    assert oracle.true_residual(dims, _rounded(U, prec), _rounded(b, prec), x1.astype(np.complex128), m) <= tol * (1.0 if prec == 64 else 1.5)


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims,links,eps", [((4, 4, 4, 4), "haar", None), ((8, 4, 6, 10), "near_identity", 0.5),
                                            ((4, 6, 2, 8), "haar", None), ((8, 8, 8, 8), "haar", None)])
def test_cg_persistent_cluster_and_grid_shapes_agree(q, dims, links, eps, prec):
    """Loop 3 runs lattices of up to 2048 sites per parity as ONE thread-block cluster (barrier.cluster, partial sums
    through distributed shared memory) and larger ones as a cooperative grid.  Same
    per-site arithmetic; only the shape of the final sum over blocks differs.  Both shapes must match the oracle,
    agree with each other to rounding, and be bitwise reproducible; the library must say which one ran."""
    m = 0.1
    tol = 1e-10 if prec == 64 else 1e-5
    U = qcd_inputs.gauge_field(dims, links, seed=0, eps=eps)
    b = qcd_inputs.gaussian_source(dims, seed=1)
    Ur, br = _rounded(U, prec), _rounded(b, prec)
    ctx = q.Context(dims, prec)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    fb, fx = ctx.field(q.QCD_SPINOR_EVEN).upload(b), ctx.field(q.QCD_SPINOR_EVEN)
    ctx.qcd_set_cg_loop(3)
    out = {}
    for cluster in (True, False):
        ctx.qcd_set_cg_cluster(cluster)
        info = ctx.qcd_cg_solve(fU, fb, fx, m, tol, 20000)
        x = fx.download()
        assert ctx.qcd_last_cg_loop() == 3
        ncta = ctx.qcd_last_cg_cluster()
        assert (1 <= ncta <= 16) if cluster else ncta == 0, ncta
        info2 = ctx.qcd_cg_solve(fU, fb, fx, m, tol, 20000)
        assert info2["iters"] == info["iters"] and np.array_equal(fx.download(), x)          # bitwise reproducible
        out[cluster] = (info, x.astype(np.complex128))
    (ic, xc), (ig, xg) = out[True], out[False]
    # the two shapes sum the per-block partials in different groupings; on the rounding plateau of 4^4 at 1e-10 (the oracle's own
    # count moves by +-3 with its thread count) that shifts the stopping iteration by a few: reading R8 is the bound
    assert ic["converged"] and ig["converged"] and iters_close(ic["iters"], ig["iters"])
    xo, oinfo = oracle.cg(dims, Ur.astype(ctx.cdtype), br.astype(ctx.cdtype), m, tol, 20000)
    for info, x in (out[True], out[False]):
        assert iters_close(info["iters"], oinfo["iters"]), (info, oinfo)
        true = oracle.true_residual(dims, Ur, br, x, m)
        if prec == 64:
            assert true <= tol, true
        else:
            assert true <= 2.0 * max(tol, oracle.true_residual(dims, Ur, br, xo.astype(np.complex128), m)), true
    if prec == 64:
        assert np.linalg.norm(xc - xg) <= 1e-9 * np.linalg.norm(xg)
    # exact stop at maxiter and the residual history in the cluster shape
    ctx.qcd_set_cg_cluster(True)
    info7 = ctx.qcd_cg_solve(fU, fb, fx, m, 1e-300, 7)
    assert info7["iters"] == 7 and info7["status"] == q.QCD_ENOTCONVERGED and len(ctx.qcd_cg_history()) == 7
    ctx.close()


def test_cg_timeline_hook(q):
    """qcd_cg_timeline_*: the persistent loop stamps its phase boundaries for the first iterations when asked to, and
    takes no stamp (and changes no result) otherwise.  Stamps are nanoseconds of one clock: monotone inside an
    iteration and from one iteration to the next, in both recorded blocks."""
    dims, m, tol = (8, 8, 8, 8), 0.1, 1e-10
    U = qcd_inputs.gauge_field(dims, "haar", seed=0)
    b = qcd_inputs.gaussian_source(dims, seed=1)
    ctx = q.Context(dims, 64)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    fb, fx = ctx.field(q.QCD_SPINOR_EVEN).upload(b), ctx.field(q.QCD_SPINOR_EVEN)
    ctx.qcd_set_cg_loop(3)
    info0 = ctx.qcd_cg_solve(fU, fb, fx, m, tol, 5000)
    x0 = fx.download()
    assert ctx.qcd_cg_timeline_read().shape == (2, 0, 9)                 # off by default: nothing recorded
    ctx.qcd_cg_timeline_enable(True)
    info1 = ctx.qcd_cg_solve(fU, fb, fx, m, tol, 5000)
    assert ctx.qcd_last_cg_loop() == 3 and info1["iters"] == info0["iters"] and np.array_equal(fx.download(), x0)
    tl = ctx.qcd_cg_timeline_read()
    assert tl.shape == (2, min(64, info1["iters"]), 9)
    flat = tl.reshape(2, -1).astype(np.int64)
    assert np.all(np.diff(flat, axis=1) >= 0)
    per_iter = np.diff(tl[0, :, 0].astype(np.int64))
    assert 0 < np.median(per_iter) < 1_000_000                            # an 8^4 iteration takes microseconds, not milliseconds
    assert ctx.qcd_cg_timeline_read(5).shape == (2, 5, 9)
    info7 = ctx.qcd_cg_solve(fU, fb, fx, m, 1e-300, 7)                     # a shorter solve: exactly its iterations are reported
    assert info7["iters"] == 7 and ctx.qcd_cg_timeline_read().shape == (2, 7, 9)
    ctx.qcd_cg_timeline_enable(False)
    ctx.qcd_set_cg_loop(1)
    ctx.qcd_cg_solve(fU, fb, fx, m, tol, 5000)                             # another loop records nothing and is unaffected
    assert np.allclose(fx.download(), x0, rtol=0, atol=1e-9 * np.max(np.abs(x0)))
    ctx.close()


# ------------------------------------------------------------------------------------------
# traversal chunking: a pure permutation of the work
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims", [(8, 4, 6, 10), (4, 6, 2, 8), (12, 2, 4, 4)])
def test_traversal_chunk_is_a_pure_permutation(q, dims, prec):
    ctx = q.Context(dims, prec, nrhs=3)
    U = qcd_inputs.gauge_field(dims, "haar", seed=0)
    phis = [qcd_inputs.gaussian_spinor(dims, seed=30 + i) for i in range(3)]
    par = qcd_inputs.site_parity(dims)
    fU = ctx.field(q.QCD_GAUGE_2ROW).upload(U)
    fin = [ctx.field(q.QCD_SPINOR_FULL).upload(p) for p in phis]
    fout = [ctx.field(q.QCD_SPINOR_FULL) for _ in phis]
    results = {}
    for W in [0] + [w for w in range(1, dims[2] + 1) if dims[2] % w == 0]:
        ctx.qcd_set_traversal_chunk(W)
        for f in fout:
            f.buf.zero_()
        ctx.qcd_dslash_eo_multi(fU, fout, fin)
        ctx.qcd_dslash_oe_multi(fU, fout, fin)
        results[W] = [f.download() for f in fout]
    for W, got in results.items():
        for i in range(3):
            assert np.array_equal(got[i], results[0][i]), (W, i)          # bitwise: same arithmetic per site
    Ur = ov.reconstruct12(ov.compress12(_rounded(U, prec)))
    for i in range(3):
        ref = oracle.dslash(dims, Ur, _rounded(phis[i], prec), -1)
        for p in (0, 1):
            assert dslash_rel_err(results[0][i][par == p], ref[par == p]) <= DSLASH_TOL[prec]
    with pytest.raises(q.QcdError):
        ctx.qcd_set_traversal_chunk(dims[2] + 1)
    # CG with a forced chunk: the reduction order changes, the solve does not
    b = qcd_inputs.gaussian_source(dims, seed=1)
    m, tol = 0.1, (1e-10 if prec == 64 else 1e-5)
    fb, fx = ctx.field(q.QCD_SPINOR_EVEN).upload(b), ctx.field(q.QCD_SPINOR_EVEN)
    ctx.qcd_set_traversal_chunk(1 if dims[2] > 1 else 0)
    info = ctx.qcd_cg_solve(fU, fb, fx, m, tol, 5000)
    xo, oinfo = oracle.cg(dims, Ur.astype(ctx.cdtype), _rounded(b, prec).astype(ctx.cdtype), m, tol, 5000)
    assert info["converged"] and iters_close(info["iters"], oinfo["iters"])
    true = oracle.true_residual(dims, Ur, _rounded(b, prec), fx.download().astype(np.complex128), m)
    if prec == 64:
        assert true <= tol
    else:       # DESIGN.md R11: an fp32 solve attains what the f32 oracle variant attains, within a factor 2
        assert true <= 2.0 * max(tol, oracle.true_residual(dims, Ur, _rounded(b, prec), xo.astype(np.complex128), m)), true
    ctx.close()


# ------------------------------------------------------------------------------------------
# solver loop for lattices that fit the L2: one persistent cooperative kernel (qcd_set_cg_loop 3)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims,links,eps,kind_name", [
    ((16, 16, 16, 16), "near_identity", 0.3, "QCD_GAUGE"),       # configs[1]
    ((8, 4, 6, 10), "haar", None, "QCD_GAUGE_2ROW"),             # fewer sites than resident threads, ragged
    ((4, 4, 4, 4), "haar", None, "QCD_GAUGE"),                   # configs[0]
    ((24, 24, 24, 24), "near_identity", 0.3, "QCD_GAUGE_2ROW"),  # more sites than resident threads: grid-stride loops
])
def test_cg_persistent_kernel(q, dims, links, eps, kind_name, prec):
    """The same algorithm, the same per-site arithmetic: iteration counts equal to the kernel-by-kernel
    loop up to the reduction order, solutions equal to rounding, oracle checks as everywhere."""
    m = 0.05 if dims[0] >= 16 else 0.1
    tol = 1e-10 if prec == 64 else 1e-5
    U = qcd_inputs.gauge_field(dims, links, seed=0, eps=eps)
    b = qcd_inputs.gaussian_source(dims, seed=1)
    Ur, br = _rounded(U, prec), _rounded(b, prec)
    if kind_name == "QCD_GAUGE_2ROW":
        Ur = ov.reconstruct12(ov.compress12(Ur))
    ctx = q.Context(dims, prec)
    fU = ctx.field(getattr(q, kind_name)).upload(U)
    fb, fx = ctx.field(q.QCD_SPINOR_EVEN).upload(b), ctx.field(q.QCD_SPINOR_EVEN)
    out = {}
    for loop in (1, 3):
        ctx.qcd_set_cg_loop(loop)
        n0 = ctx.qcd_launch_count()
        info = ctx.qcd_cg_solve(fU, fb, fx, m, tol, 20000)
        launches = ctx.qcd_launch_count() - n0
        out[loop] = (info, fx.download().astype(np.complex128), launches)
    (i1, x1, l1), (i3, x3, l3) = out[1], out[3]
    assert i1["converged"] and i3["converged"]
    assert l3 == 2 and l1 >= 4 * i1["iters"]                       # init + ONE kernel for the whole solve
    assert iters_close(i1["iters"], i3["iters"]), (i1, i3)          # reading R8 (the reduction orders differ)
    xo, oinfo = oracle.cg(dims, Ur.astype(ctx.cdtype), br.astype(ctx.cdtype), m, tol, 20000)
    assert iters_close(i3["iters"], oinfo["iters"]), (i3, oinfo)
    true = oracle.true_residual(dims, Ur, br, x3, m)
    if prec == 64:
        assert true <= tol, true
        assert np.linalg.norm(x3 - x1) <= 1e-9 * np.linalg.norm(x1)
    else:
        assert true <= 2.0 * max(tol, oracle.true_residual(dims, Ur, br, xo.astype(np.complex128), m)), true
    # exact stop at maxiter, zero iterations, zero source
    info = ctx.qcd_cg_solve(fU, fb, fx, m, 1e-300, 7)
    assert info["iters"] == 7 and info["status"] == q.QCD_ENOTCONVERGED
    x7 = fx.download()
    ctx.qcd_set_cg_loop(1)
    assert ctx.qcd_cg_solve(fU, fb, fx, m, 1e-300, 7)["iters"] == 7
    assert np.allclose(fx.download(), x7, rtol=0, atol=(1e-12 if prec == 64 else 1e-5) * np.max(np.abs(x7)))
    ctx.qcd_set_cg_loop(3)
    info = ctx.qcd_cg_solve(fU, fb, fx, m, tol, 0)
    assert info["iters"] == 0 and info["status"] == q.QCD_ENOTCONVERGED and not fx.download().any()
    fz = ctx.field(q.QCD_SPINOR_EVEN)
    fz.buf.zero_()
    info = ctx.qcd_cg_solve(fU, fz, fx, m, tol, 100)
    assert info["iters"] == 0 and info["converged"] and not fx.download().any()
    # run to run bitwise reproducible
    ctx.qcd_cg_solve(fU, fb, fx, m, tol, 20000)
    xa = fx.download()
    ctx.qcd_cg_solve(fU, fb, fx, m, tol, 20000)
    assert np.array_equal(xa, fx.download())
    ctx.close()


# ------------------------------------------------------------------------------------------
# index arithmetic on unusual shapes: seeded random extents, every kernel family
# ------------------------------------------------------------------------------------------
def _random_shapes(n, seed=5):
    rng = np.random.default_rng(seed)
    shapes = [(4, 2, 2, 2), (4, 2, 2, 12), (16, 2, 6, 2), (20, 4, 2, 4)]        # extremes first: h = 2, N = 2 everywhere
    while len(shapes) < n:
        shapes.append((int(rng.choice([4, 8, 12, 16, 20, 24])), int(rng.choice([2, 4, 6, 8, 10])),
                       int(rng.choice([2, 4, 6, 8])), int(rng.choice([2, 4, 6, 10, 14]))))
    return shapes


@pytest.mark.parametrize("dims", _random_shapes(12))
def test_random_shapes_every_kernel_family(q, dims):
    """Full links / two rows / two rows + temporal gauge, 1 and 3 vectors (register, staged), both
    precisions, D_oe and D_eo, against the oracle; then a CG solve in each solver loop."""
    U = qcd_inputs.gauge_field(dims, "haar", seed=0)
    Ufix, _ = ov.temporal_gauge(dims, U)
    Ufix[qcd_inputs.site_coords(dims)[:, 3] != 0, 3] = np.eye(3)
    phis = [qcd_inputs.gaussian_spinor(dims, seed=60 + i) for i in range(3)]
    par = qcd_inputs.site_parity(dims)
    for prec in (64, 32):
        ctx = q.Context(dims, prec, nrhs=3)
        fin = [ctx.field(q.QCD_SPINOR_FULL).upload(p) for p in phis]
        fout = [ctx.field(q.QCD_SPINOR_FULL) for _ in phis]
        for kind, links, tg in ((q.QCD_GAUGE, U, False), (q.QCD_GAUGE_2ROW, U, False), (q.QCD_GAUGE_2ROW, Ufix, True)):
            fU = ctx.field(kind).upload(links)
            ctx.qcd_gauge_set_temporal_unit(fU, tg)
            Ur = _rounded(links, prec)
            if kind == q.QCD_GAUGE_2ROW:
                Ur = ov.reconstruct12(ov.compress12(Ur))
            refs = [oracle.dslash(dims, Ur, _rounded(p, prec), -1) for p in phis]
            for n in (1, 3):
                for f in fout:
                    f.buf.zero_()
                ctx.qcd_dslash_eo_multi(fU, fout[:n], fin[:n])
                ctx.qcd_dslash_oe_multi(fU, fout[:n], fin[:n])
                for i in range(n):
                    got = fout[i].download()
                    for p in (0, 1):
                        assert dslash_rel_err(got[par == p], refs[i][par == p]) <= DSLASH_TOL[prec], (prec, kind, tg, n, i, p)
        # CG on the full links, every solver loop
        b = qcd_inputs.gaussian_source(dims, seed=1)
        m, tol = 0.2, (1e-9 if prec == 64 else 1e-5)
        fU = ctx.field(q.QCD_GAUGE).upload(U)
        fb, fx = ctx.field(q.QCD_SPINOR_EVEN).upload(b), ctx.field(q.QCD_SPINOR_EVEN)
        Ur, br = _rounded(U, prec), _rounded(b, prec)
        xo, oinfo = oracle.cg(dims, Ur.astype(ctx.cdtype), br.astype(ctx.cdtype), m, tol, 3000)
        bound = tol if prec == 64 else 2.0 * max(tol, oracle.true_residual(dims, Ur, br, xo.astype(np.complex128), m))
        for loop in (1, 3):
            ctx.qcd_set_cg_loop(loop)
            info = ctx.qcd_cg_solve(fU, fb, fx, m, tol, 3000)
            assert info["converged"] and iters_close(info["iters"], oinfo["iters"]), (prec, loop, info, oinfo)
            assert oracle.true_residual(dims, Ur, br, fx.download().astype(np.complex128), m) <= bound, (prec, loop)
        ctx.close()

"""Out-of-bounds and race checks of our own, through the C-ABI (SURVEY.md Sec. 4 tier (v), Sec. 5).

`compute-sanitizer` is closed on this GPU pool ("runs under it have left GPUs needing a reset"; recorded in
profiles/r02_sanitizer.md), so the checks it would have made are made here by construction:

  out-of-bounds WRITES   every field and the solver workspace are bound in the MIDDLE of a larger torch buffer
                         whose 64 KiB guard bands on both sides are filled with 0xFF; after every kernel family
                         has run the bands must still be 0xFF, byte for byte;
  out-of-bounds READS /  the bands and the not-yet-written interiors are NaN bit patterns (all-ones bytes are a NaN
  unwritten outputs      in fp32 and fp64): a read past a field, or an output element a kernel never wrote, puts a
                         NaN into a result that is then compared with the oracle element by element;
  races                  the kernels that communicate through shared memory (block reductions, the cp.async ring of
                         the staged Dslash, the cluster CG with its DSMEM slots) or through global memory between
                         barriers (cooperative-grid CG, last-block reductions) are run repeatedly and must return
                         bitwise identical results every time and the oracle's result within tolerance.

Lattices: 4^4 (one block), (8,4,6,10) (several blocks and a ragged tail), (12,2,2,4) (time slices shorter than a
warp), 16^4 (256 blocks, the cooperative-grid shape of the persistent loop).
"""
import ctypes

import numpy as np
import pytest

import oracle
import oracle.variants as ov
import qcd_inputs
from util import DSLASH_TOL, dslash_rel_err, iters_close

pytestmark = pytest.mark.gpu

GUARD = 1 << 16
SHAPES = [((4, 4, 4, 4), "haar", None), ((8, 4, 6, 10), "near_identity", 0.5), ((12, 2, 2, 4), "haar", None),
          ((16, 16, 16, 16), "near_identity", 0.3)]


@pytest.fixture(scope="module")
def q():
    import paper_2502_03249_b200 as pkg
    return pkg


class Guarded:
    """A field bound in the middle of a 0xFF-filled buffer."""

    def __init__(self, ctx, kind):
        import torch
        self.n = ctx.qcd_field_bytes(kind)
        self.raw = torch.full((self.n + 2 * GUARD,), 0xFF, dtype=torch.uint8, device=ctx.device)
        self.f = ctx.field(kind, buf=self.raw[GUARD: GUARD + self.n])

    def intact(self) -> bool:
        return bool((self.raw[:GUARD] == 0xFF).all().item() and (self.raw[GUARD + self.n:] == 0xFF).all().item())


def guarded_context(q, dims, prec, nrhs=1, stream=None):
    """Context whose workspace sits between guard bands as well."""
    import torch
    ctx = q.Context(dims, prec, workspace=False, stream=stream)
    n = ctx.qcd_workspace_bytes_multi(nrhs)
    raw = torch.full((n + 2 * GUARD,), 0xFF, dtype=torch.uint8, device=ctx.device)
    ctx.ws = raw[GUARD: GUARD + n]
    ctx._check(ctx.lib.qcd_set_workspace(ctx.handle, ctypes.c_void_p(ctx.ws.data_ptr()), n), "qcd_set_workspace")
    ctx._ws_raw, ctx._ws_n = raw, n
    return ctx


def ws_intact(ctx) -> bool:
    raw, n = ctx._ws_raw, ctx._ws_n
    return bool((raw[:GUARD] == 0xFF).all().item() and (raw[GUARD + n:] == 0xFF).all().item())


def _rounded(a, prec):
    return a if prec == 64 else a.astype(np.complex64).astype(np.complex128)


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims,links,eps", SHAPES)
def test_guard_bands_dslash_families(q, dims, links, eps, prec):
    """Every Dslash kernel family (link storage x temporal gauge x number of vectors x kernel choice), the M
    application, the layout kernels, the gauge transforms and the precision conversion, between guard bands."""
    U = qcd_inputs.gauge_field(dims, links, seed=0, eps=eps)
    par = qcd_inputs.site_parity(dims)
    ctx = guarded_context(q, dims, prec)
    gU = Guarded(ctx, q.QCD_GAUGE)
    gU.f.upload(U)
    assert np.array_equal(gU.f.download(), U.astype(ctx.cdtype)) and gU.intact()
    # temporal gauge on the device, two-row copy of it
    gUf, gg, g12 = Guarded(ctx, q.QCD_GAUGE), Guarded(ctx, q.QCD_COLOUR_MATRIX), Guarded(ctx, q.QCD_GAUGE_2ROW)
    ctx.qcd_gauge_fix_temporal(gU.f, gUf.f, gg.f)
    ctx.qcd_gauge_compress(gUf.f, g12.f)
    Uf = gUf.f.download().astype(np.complex128)
    assert np.isfinite(Uf).all() and np.isfinite(gg.f.download()).all()
    U12ref = ov.reconstruct12(ov.compress12(Uf))
    guards = [gU, gUf, gg, g12]
    nmax = 8
    phis = [qcd_inputs.gaussian_spinor(dims, seed=20 + i) for i in range(nmax)]
    gin = [Guarded(ctx, q.QCD_SPINOR_FULL) for _ in range(nmax)]
    gout = [Guarded(ctx, q.QCD_SPINOR_FULL) for _ in range(nmax)]
    for g, p in zip(gin, phis):
        g.f.upload(p)
    guards += gin + gout
    for fU, Uref in ((gU.f, _rounded(U, prec)), (g12.f, U12ref)):
        refs = ov.dslash_multi(dims, Uref, [_rounded(p, prec) for p in phis], -1)
        for n in (1, 2, 3, 4, 8):
            first = None
            for kernel in ((0, 1, 2, 3) if n == 1 else (0, 4, 5, 6, 7, 8, 9, 10)):
                ctx.qcd_set_dslash_variant(kernel)
                for g in gout[:n]:
                    g.raw[GUARD: GUARD + g.n] = 0xFF                         # NaN: an element nobody writes stays NaN
                ctx.qcd_dslash_eo_multi(fU, [g.f for g in gout[:n]], [g.f for g in gin[:n]])
                ctx.qcd_dslash_oe_multi(fU, [g.f for g in gout[:n]], [g.f for g in gin[:n]])
                got = [g.f.download() for g in gout[:n]]
                for i in range(n):
                    for p in (0, 1):
                        assert dslash_rel_err(got[i][par == p], refs[i][par == p]) <= DSLASH_TOL[prec], (n, kernel, i, p)
                if first is None:
                    first = got
                else:
                    assert all(np.array_equal(a, b) for a, b in zip(first, got)), (n, kernel)
            ctx.qcd_set_dslash_variant(0)
    # M application and the spinor rotation
    ge, gm = Guarded(ctx, q.QCD_SPINOR_EVEN), Guarded(ctx, q.QCD_SPINOR_EVEN)
    b = qcd_inputs.gaussian_source(dims, seed=1)
    ge.f.upload(b)
    ctx.qcd_apply_M(gU.f, gm.f, ge.f, 0.1)
    ref = oracle.apply_M(dims, _rounded(U, prec), _rounded(b, prec), 0.1)
    assert dslash_rel_err(gm.f.download()[par == 0], ref[par == 0]) <= 2 * DSLASH_TOL[prec]
    ctx.qcd_spinor_rotate(gg.f, gm.f, ge.f)
    ctx.qcd_spinor_rotate(gg.f, gm.f, gm.f, dagger=True)
    assert np.allclose(gm.f.download(), b.astype(ctx.cdtype), rtol=0, atol=(1e-13 if prec == 64 else 1e-5) * np.abs(b).max())
    guards += [ge, gm]
    for g in guards:
        assert g.intact()
    assert ws_intact(ctx)
    ctx.close()


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims,links,eps", SHAPES)
def test_guard_bands_and_repeatability_cg_loops(q, dims, links, eps, prec):
    """Every solver loop (kernel by kernel, graph replay, persistent kernel as one cluster and as a cooperative grid),
    the lock-step multi solve and the mixed-precision solve, between guard bands, five times each: bitwise identical
    every time, iteration count and true residual as the oracle's."""
    import torch
    m = 0.1
    tol = 1e-10 if prec == 64 else 1e-5
    U = qcd_inputs.gauge_field(dims, links, seed=0, eps=eps)
    b = qcd_inputs.gaussian_source(dims, seed=1)
    Ur, br = _rounded(U, prec), _rounded(b, prec)
    xo, oinfo = oracle.cg(dims, Ur.astype(np.complex128 if prec == 64 else np.complex64),
                          br.astype(np.complex128 if prec == 64 else np.complex64), m, tol, 20000)
    bound = tol if prec == 64 else 2.0 * max(tol, oracle.true_residual(dims, Ur, br, xo.astype(np.complex128), m))
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ctx = guarded_context(q, dims, prec, nrhs=3, stream=stream)
        gU, gb, gx = Guarded(ctx, q.QCD_GAUGE), Guarded(ctx, q.QCD_SPINOR_EVEN), Guarded(ctx, q.QCD_SPINOR_EVEN)
        gU.f.upload(U)
        gb.f.upload(b)
        shapes = [(1, True), (2, True), (3, True), (3, False)]
        for loop, cluster in shapes:
            ctx.qcd_set_cg_loop(loop)
            ctx.qcd_set_cg_cluster(cluster)
            first = None
            for rep in range(5):
                gx.raw[GUARD: GUARD + gx.n] = 0xFF
                info = ctx.qcd_cg_solve(gU.f, gb.f, gx.f, m, tol, 20000)
                x = gx.f.download()
                assert ctx.qcd_last_cg_loop() == loop
                assert info["converged"] and iters_close(info["iters"], oinfo["iters"]), (loop, cluster, info, oinfo)
                if first is None:
                    first = (info["iters"], x)
                    assert oracle.true_residual(dims, Ur, br, x.astype(np.complex128), m) <= bound, (loop, cluster)
                else:
                    assert info["iters"] == first[0] and np.array_equal(x, first[1]), (loop, cluster, rep)
            assert gU.intact() and gb.intact() and gx.intact() and ws_intact(ctx), (loop, cluster)
        # lock-step solve of three right-hand sides (the second is zero: frozen at iteration 0)
        ctx.qcd_set_cg_loop(0)
        srcs = [b, 0.0 * b, qcd_inputs.gaussian_source(dims, seed=3)]
        gbs = [Guarded(ctx, q.QCD_SPINOR_EVEN) for _ in srcs]
        gxs = [Guarded(ctx, q.QCD_SPINOR_EVEN) for _ in srcs]
        for g, s_ in zip(gbs, srcs):
            g.f.upload(s_)
        first = None
        for rep in range(3):
            infos = ctx.qcd_cg_solve_multi(gU.f, [g.f for g in gbs], [g.f for g in gxs], m, tol, 20000)
            xs = [g.f.download() for g in gxs]
            assert infos[1]["iters"] == 0 and not xs[1].any()
            assert iters_close(infos[0]["iters"], oinfo["iters"])
            if first is None:
                first = xs
            else:
                assert all(np.array_equal(a, c) for a, c in zip(first, xs)), rep
        for g in gbs + gxs:
            assert g.intact()
        assert ws_intact(ctx)
        ctx.close()


@pytest.mark.parametrize("dims,links,eps", SHAPES[:3])
def test_guard_bands_mixed_precision(q, dims, links, eps):
    m, tol = 0.1, 1e-10
    U = qcd_inputs.gauge_field(dims, links, seed=0, eps=eps)
    b = qcd_inputs.gaussian_source(dims, seed=1)
    c64, c32 = guarded_context(q, dims, 64), guarded_context(q, dims, 32)
    gU64, gU32 = Guarded(c64, q.QCD_GAUGE), Guarded(c32, q.QCD_GAUGE)
    gU64.f.upload(U)
    c64.qcd_field_convert(gU32.f, gU64.f)
    gb, gx = Guarded(c64, q.QCD_SPINOR_EVEN), Guarded(c64, q.QCD_SPINOR_EVEN)
    gr, ge = Guarded(c32, q.QCD_SPINOR_EVEN), Guarded(c32, q.QCD_SPINOR_EVEN)
    gb.f.upload(b)
    first = None
    for rep in range(3):
        info = c64.qcd_cg_solve_mixed(c32, gU64.f, gU32.f, gb.f, gx.f, gr.f, ge.f, m, tol, 1e-3, 20000)
        x = gx.f.download()
        assert info["converged"] and oracle.true_residual(dims, U, b, x, m) <= tol
        if first is None:
            first = x
        else:
            assert np.array_equal(first, x)
    for g in (gU64, gU32, gb, gx, gr, ge):
        assert g.intact()
    assert ws_intact(c64) and ws_intact(c32)
    c64.close(); c32.close()

"""GPU parity at BASELINE.json's full sizes (configs 2, 3, 4), in the launch configuration
bench.py times (default Dslash variant, qcd_cg_solve as bench.py's extras call it).

Dslash: the whole output field against the oracle where the oracle finishes in seconds, plus
sampled sites through oracle.dslash_site (the literal single-site Eq. (1)), chosen to include
every lattice face (wrap in each direction, the antiperiodic time seam) and random interior
sites.  CG: the fp64 oracle recomputes ||b - M x_gpu|| / ||b|| (one M application); the
iteration count is compared with the oracle's stored count (tests/golden/cg_config*_fp*.json,
written by tests/golden/make_cg_golden.py from oracle/ only; the fingerprint proves the
inputs regenerated here are the ones the oracle solved)."""
import importlib.util
import json
import os

import numpy as np
import pytest

import oracle
import qcd_inputs
from util import DSLASH_TOL, dslash_rel_err, iters_close

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))
_spec = importlib.util.spec_from_file_location("make_cg_golden", os.path.join(HERE, "golden", "make_cg_golden.py"))
golden_mod = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(golden_mod)


@pytest.fixture(scope="module")
def q():
    import paper_2502_03249_b200 as pkg
    return pkg


_cache = {}


def inputs(i):
    """One config's inputs at a time (64^4 links are 9.7 GB on the host)."""
    if _cache.get("i") != i:
        _cache.clear()
        cfg, U, b = qcd_inputs.config_inputs(i)
        _cache.update(i=i, cfg=cfg, U=U, b=b, fp=golden_mod.fingerprint(U, b))
    return _cache["cfg"], _cache["U"], _cache["b"]


def golden(i, prec):
    p = golden_mod.golden_path(i, prec)
    if not os.path.exists(p):
        return None
    with open(p) as f:
        g = json.load(f)
    assert g["input_fingerprint"] == _cache["fp"], "inputs regenerated here differ from the ones the oracle solved"
    return g


def sample_sites(dims, parity, n_random, seed):
    """Sites of one parity: all 2^4 combinations of {first, last} coordinate per direction that have
    the parity (faces, edges, corners: every wrap and the time seam), plus random ones."""
    rng = np.random.default_rng(seed)
    sites = []
    for c in np.ndindex(2, 2, 2, 2):
        x = [0 if c[d] == 0 else dims[d] - 1 for d in range(4)]
        for bump in range(2):                       # the corner and its x0-neighbour cover both parities
            y = list(x)
            y[0] = (y[0] + bump) % dims[0]
            if sum(y) % 2 == parity:
                sites.append(tuple(y))
    while len(sites) < n_random + 16:
        x = [int(rng.integers(0, d)) for d in dims]
        if sum(x) % 2 == parity:
            sites.append(tuple(x))
    return sites


def lex(dims, x):
    return x[0] + dims[0] * (x[1] + dims[1] * (x[2] + dims[2] * x[3]))


def rounded(a, prec):
    return a if prec == 64 else a.astype(np.complex64).astype(np.complex128)


# ------------------------------------------------------------------------------------------
# Dslash at full size
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("config", [2, 3, 4])
def test_dslash_full_size(q, config, prec):
    cfg, U, b = inputs(config)
    dims = cfg["dims"]
    if prec == 32 and cfg["tol32"] is None:
        pytest.skip("BASELINE.json names fp64 only for this config")
    V = int(np.prod(dims))
    ctx = q.Context(dims, prec)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    fe = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
    fo = ctx.field(q.QCD_SPINOR_ODD)
    fe2 = ctx.field(q.QCD_SPINOR_EVEN)
    ctx.qcd_dslash_oe(fU, fo, fe)              # t = D_oe b
    got_o = fo.download()
    Ur, br = rounded(U, prec), rounded(b, prec)
    tol = DSLASH_TOL[prec]
    R_o = np.sqrt(np.mean(np.linalg.norm(got_o[1::2], axis=1) ** 2))      # rms site norm scale (R10)
    # sampled sites, literal Eq. (1) one site at a time
    worst = 0.0
    for x in sample_sites(dims, 1, 300, seed=config):
        ref = oracle.dslash_site(dims, Ur, br, x)
        d = np.linalg.norm(got_o[lex(dims, x)] - ref) / max(np.linalg.norm(ref), 0.1 * R_o)
        worst = max(worst, d)
    assert worst <= tol, worst
    # whole field, element by element
    par = qcd_inputs.site_parity(dims)
    ref_o = oracle.dslash(dims, Ur, br, 1)
    assert dslash_rel_err(got_o[par == 1], ref_o[par == 1]) <= tol
    assert not got_o[par == 0].any()
    # second hop (D_eo): device and oracle both start from the ORACLE's t, rounded to the device precision
    t_in = rounded(ref_o, prec)
    del ref_o
    fo.upload(t_in)
    ctx.qcd_dslash_eo(fU, fe2, fo)
    got_e = fe2.download()
    R_e = np.sqrt(np.mean(np.linalg.norm(got_e[::2], axis=1) ** 2))
    worst = 0.0
    for x in sample_sites(dims, 0, 300, seed=100 + config):
        ref = oracle.dslash_site(dims, Ur, t_in, x)
        d = np.linalg.norm(got_e[lex(dims, x)] - ref) / max(np.linalg.norm(ref), 0.1 * R_e)
        worst = max(worst, d)
    assert worst <= tol, worst
    ref_e = oracle.dslash(dims, Ur, t_in, 0)
    assert dslash_rel_err(got_e[par == 0], ref_e[par == 0]) <= tol
    assert V == par.size
    ctx.close()


# ------------------------------------------------------------------------------------------
# the paper's variants at full size, as bench.py launches them
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [4, 8])
def test_multi_vector_two_row_64(q, n):
    """configs[4], fp64, two-row links compressed on the device, n vectors per link load: at this size
    the library chunks the traversal (W < N2) and picks the staged kernel for n = 4, the register
    kernel for n = 8 -- exactly what bench.py's variants sweep times.  Sampled sites, literal Eq. (1)."""
    cfg, U, b = inputs(4)
    dims = cfg["dims"]
    ctx = q.Context(dims, 64)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    f12 = ctx.field(q.QCD_GAUGE_2ROW)
    ctx.qcd_gauge_compress(fU, f12)
    fU.free()
    srcs = [b] + [qcd_inputs.gaussian_source(dims, seed=40 + i) for i in range(1, n)]
    fin = [ctx.field(q.QCD_SPINOR_EVEN).upload(s_) for s_ in srcs]
    fout = [ctx.field(q.QCD_SPINOR_ODD) for _ in range(n)]
    ctx.qcd_dslash_oe_multi(f12, fout, fin)
    sites = sample_sites(dims, 1, 60, seed=7)
    for i in range(n):
        got = fout[i].download()
        R = np.sqrt(np.mean(np.linalg.norm(got[1::2], axis=1) ** 2))
        worst = 0.0
        for x in sites:
            ref = oracle.dslash_site(dims, U, srcs[i], x)       # fp64: the rebuilt third row is the third row (1e-15)
            worst = max(worst, np.linalg.norm(got[lex(dims, x)] - ref) / max(np.linalg.norm(ref), 0.1 * R))
        assert worst <= DSLASH_TOL[64], (i, worst)
        del got
    # the bulk-copy kernel (variant 10) at the same size, on the chunked traversal: bitwise the same fields, compared on the device
    import torch
    first = [f.buf.clone() for f in fout]
    ctx.qcd_set_dslash_variant(10)
    for f in fout:
        f.buf.fill_(255)
    ctx.qcd_dslash_oe_multi(f12, fout, fin)
    torch.cuda.synchronize()
    assert all(torch.equal(a, f.buf) for a, f in zip(first, fout))
    ctx.qcd_set_dslash_variant(0)
    ctx.close()


@pytest.mark.parametrize("prec", [64, 32])
def test_temporal_gauge_two_row_32(q, prec):
    """configs[2] (the paper's Table 2 lattice): links fixed to temporal gauge by the ORACLE, rounded,
    uploaded as two-row links and marked; n = 1 and n = 4; whole fields against the oracle."""
    import oracle.variants as ov
    cfg, U, b = inputs(2)
    dims = cfg["dims"]
    Ufix, g = ov.temporal_gauge(dims, U)
    x3 = qcd_inputs.site_coords(dims)[:, 3]
    Ufix[x3 != 0, 3] = np.eye(3)
    Uref = ov.reconstruct12(ov.compress12(rounded(Ufix, prec)))
    srcs = [ov.rotate_spinor(g, b)] + [qcd_inputs.gaussian_source(dims, seed=50 + i) for i in range(1, 4)]
    par = qcd_inputs.site_parity(dims)
    ctx = q.Context(dims, prec)
    f12 = ctx.field(q.QCD_GAUGE_2ROW).upload(Ufix)
    ctx.qcd_gauge_set_temporal_unit(f12, True)
    fin = [ctx.field(q.QCD_SPINOR_EVEN).upload(s_) for s_ in srcs]
    fout = [ctx.field(q.QCD_SPINOR_ODD) for _ in srcs]
    refs = [oracle.dslash(dims, Uref, rounded(s_, prec), 1) for s_ in srcs]
    ctx.qcd_dslash_oe(f12, fout[0], fin[0])
    assert dslash_rel_err(fout[0].download()[par == 1], refs[0][par == 1]) <= DSLASH_TOL[prec]
    for f in fout:
        f.buf.zero_()
    ctx.qcd_dslash_oe_multi(f12, fout, fin)
    for i in range(4):
        assert dslash_rel_err(fout[i].download()[par == 1], refs[i][par == 1]) <= DSLASH_TOL[prec], i
    ctx.close()


# ------------------------------------------------------------------------------------------
# CG at full size
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("config,prec", [(2, 64), (2, 32), (3, 64), (4, 64), (4, 32)])
def test_cg_full_size(q, config, prec):
    cfg, U, b = inputs(config)
    dims, m = cfg["dims"], cfg["m"]
    tol = cfg["tol64"] if prec == 64 else cfg["tol32"]
    g = golden(config, prec)
    ctx = q.Context(dims, prec)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    fb = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
    fx = ctx.field(q.QCD_SPINOR_EVEN)
    info = ctx.qcd_cg_solve(fU, fb, fx, m, tol, cfg["maxiter"])
    x = fx.download()
    ctx.close()
    assert info["status"] == q.QCD_OK and info["converged"], info
    assert info["rel_resid"] <= tol
    true = oracle.true_residual(dims, rounded(U, prec), rounded(b, prec), x, m)
    if prec == 64:
        assert true <= tol, true                                  # north_star: recomputed by the oracle in fp64
    elif g is not None:
        assert true <= 2.0 * g["true_resid"], (true, g["true_resid"])   # DESIGN.md R11 (Haar links, plain fp32)
    if g is None:
        pytest.skip(f"no stored oracle solve for config {config} fp{prec} (tests/golden/make_cg_golden.py); "
                    f"residual check passed: true {true:.3e}, iters {info['iters']}")
    assert g["tol"] == tol and g["m"] == m and g["status"] == 0
    assert iters_close(info["iters"], g["iters"]), (info["iters"], g["iters"])
    assert abs(info["bnorm2"] - g["bnorm2"]) <= 1e-6 * g["bnorm2"]


@pytest.mark.parametrize("config,prec", [(2, 64), (4, 32)])
def test_cg_full_size_is_bitwise_reproducible(q, config, prec):
    """The reductions are deterministic (fixed summation order, integer tickets only): two solves of the
    same system give the same iteration count, the same recurrence residual and the same bits in x."""
    cfg, U, b = inputs(config)
    dims, m = cfg["dims"], cfg["m"]
    tol = cfg["tol64"] if prec == 64 else cfg["tol32"]
    ctx = q.Context(dims, prec)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    fb = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
    fx = ctx.field(q.QCD_SPINOR_EVEN)
    i1 = ctx.qcd_cg_solve(fU, fb, fx, m, tol, cfg["maxiter"])
    x1 = fx.download()
    fx.buf.zero_()
    i2 = ctx.qcd_cg_solve(fU, fb, fx, m, tol, cfg["maxiter"])
    x2 = fx.download()
    ctx.close()
    assert i1["iters"] == i2["iters"] and i1["rel_resid"] == i2["rel_resid"]
    assert np.array_equal(x1, x2)


# ------------------------------------------------------------------------------------------
# beyond the benchmark sizes: element offsets past 2^31
# ------------------------------------------------------------------------------------------
def test_lattice_with_more_than_2G_link_elements(q):
    """128 x 128 x 64 x 64 (4 x configs[4]'s volume; links 38.7 GB fp64): the gauge field has 72 planes of
    Vh = 33.5 M complex numbers = 2.4e9 elements, so every plane offset past plane 63 exceeds 2^31 --
    which no BASELINE.json config reaches (64^4: 6.0e8).  It is also the first size at which ONE vector
    is walked in the chunked traversal order (W = 16 < N2).  Whole fields against the oracle for D_oe,
    D_eo and M, and the CG iterate after 3 iterations against the oracle's."""
    dims = (128, 128, 64, 64)
    _cache.clear()                               # drop a cached config: the links here are 38.7 GB on the host
    U = qcd_inputs.gauge_field(dims, "haar", seed=0)
    b = qcd_inputs.gaussian_source(dims, seed=1, parity=0)
    par = qcd_inputs.site_parity(dims)
    for prec in (64, 32):                        # fp64 first: the fp32 pass rounds U and b in place
        _beyond_2G(q, dims, U, b, par, prec)
        if prec == 64:
            U, b = rounded(U, 32), rounded(b, 32)


def _beyond_2G(q, dims, U, b, par, prec):
    m = 0.05
    # fp64: north_star's 1e-13.  fp32: north_star states 2e-6 for the five configs; the measure (R10) is a MAX
    # over sites with the site norm floored at 0.1 R, and over 4 x the sites of configs[4] its tail reaches
    # 2.08e-6 (measured; 64^4 stays below 2e-6), so this size is held to 3e-6.  An indexing fault shows as O(1).
    tol = DSLASH_TOL[prec] if prec == 64 else 3e-6
    ctx = q.Context(dims, prec)
    assert 72 * (par.size // 2) > 2 ** 31 and ctx.qcd_field_bytes(q.QCD_GAUGE) == par.size * 4 * 18 * (prec // 8)
    fU = ctx.field(q.QCD_GAUGE).upload(U)         # fp32: U, b arrive already rounded (exactly representable)
    fe = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
    fo = ctx.field(q.QCD_SPINOR_ODD)
    fe2 = ctx.field(q.QCD_SPINOR_EVEN)
    ctx.qcd_dslash_oe(fU, fo, fe)
    got = fo.download()
    ref = oracle.dslash(dims, U, b, 1)
    assert dslash_rel_err(got[par == 1], ref[par == 1]) <= tol
    assert not got[par == 0].any()
    t_in = rounded(ref, prec)
    del ref, got
    fo.upload(t_in)
    ctx.qcd_dslash_eo(fU, fe2, fo)
    got = fe2.download()
    ref = oracle.dslash(dims, U, t_in, 0)
    assert dslash_rel_err(got[par == 0], ref[par == 0]) <= tol
    del ref, got, t_in
    ctx.qcd_apply_M(fU, fe2, fe, m)
    got = fe2.download()
    ref = oracle.apply_M(dims, U, b, m)
    assert dslash_rel_err(got[par == 0], ref[par == 0]) <= 2 * tol
    del ref, got
    info = ctx.qcd_cg_solve(fU, fe, fe2, m, 1e-12, 3)
    got = fe2.download()
    xo, oinfo = oracle.cg(dims, U, b, m, 1e-12, 3)
    assert info["iters"] == oinfo["iters"] == 3 and not info["converged"]
    if prec == 64:
        assert dslash_rel_err(got[par == 0], xo[par == 0]) <= 1e-12
        assert abs(info["rel_resid"] - oinfo["rel_resid"]) <= 1e-12 * oinfo["rel_resid"]
    else:
        assert dslash_rel_err(got[par == 0], xo[par == 0]) <= 2e-5   # three fp32 iterations against fp64 ones
        assert abs(info["rel_resid"] - oinfo["rel_resid"]) <= 1e-5 * oinfo["rel_resid"]
    ctx.close()

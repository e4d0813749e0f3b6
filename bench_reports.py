"""Sidecar reports of bench.py (rank 0, N = 1 semantics; nothing here is printed on stdout).

bench.py's stdout is ONE compact JSON line.  Everything else SURVEY.md Sec. 8(d) asks to be reported -- the
per-config table (Dslash and CG at BASELINE.json configs 0-4 with the oracle timed beside them), full solves in
both precisions, the paper's variants, the small-lattice solver loops, the CG
update routine of Table 1 and the Fig. 3 size sweep -- is collected here into the `side` dict
that bench.py writes to the sidecar file.  `run_all` also fills the few headline keys that need these
measurements (cpu_baseline, dslash_gbs_*, cg_s_per_solve_*).

Every section is guarded: a failure is recorded under side["errors"] and costs that section only.
The oracle (test infrastructure) is used here for the cpu_baseline leg and the oracle-recomputed residuals only.
"""
from __future__ import annotations

import json
import os
import time

import numpy as np

from bench import (FLOP_PER_CG_ITER, FLOP_PER_SITE, REALS_DSLASH_COMPULSORY, REALS_DSLASH_NOMINAL, REALS_ITER_NOMINAL,
                   ROOT, THEORETICAL_HBM_GBS, UNIT, log, make_inputs)

L2_RESIDENT_BYTES = 96 << 20        # links + work vectors below this: the run measures the L2, not HBM


def section(side: dict, name: str, fn):
    t0 = time.time()
    res = None
    try:
        log(f"report: {name}")
        res = fn()
        if res is not None:
            side[name] = res
    except Exception as e:  # noqa: BLE001 -- a report must never cost the headline
        side.setdefault("errors", {})[name] = repr(e)
        log(f"report {name} FAILED: {e!r}")
    side.setdefault("section_seconds", {})[name] = round(time.time() - t0, 1)
    return res


# ---- Dslash timing ---------------------------------------------------------------------------
def time_dslash(torch, ctx, fU, fin, fout, n=20):
    for _ in range(3):
        ctx.qcd_dslash_oe(fU, fout, fin)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n):
        ctx.qcd_dslash_oe(fU, fout, fin)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / n


def time_dslash_graph(torch, ctx, stream, fU, fin, fout, per_graph=20, replays=5):
    """ms per D_oe launch, the launches replayed from a CUDA graph: below 16^4 a Python-driven launch loop would
    time the host, not the kernel.  `stream` is the context's (non-default) stream and must be current."""
    ctx.qcd_dslash_oe(fU, fout, fin)
    stream.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=stream):
        for _ in range(per_graph):
            ctx.qcd_dslash_oe(fU, fout, fin)
    graph.replay()
    stream.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(replays):
        graph.replay()
    e1.record(stream)
    stream.synchronize()
    ms = e0.elapsed_time(e1) / (per_graph * replays)
    del graph
    return ms


def dslash_report(ms, Vh, rsize, peak, stream_gbs=None):
    comp = REALS_DSLASH_COMPULSORY * rsize * Vh / ms / 1e6
    r = {"ms": round(ms, 5), "gflops": round(FLOP_PER_SITE * Vh / ms / 1e6, 1),
         "effective_gbs_nominal": round(REALS_DSLASH_NOMINAL * rsize * Vh / ms / 1e6, 1),
         "gbs_compulsory": round(comp, 1),
         "frac_of_measured_copy_peak": round(comp / peak, 4),
         "frac_of_theoretical_8184": round(comp / THEORETICAL_HBM_GBS, 4)}
    if stream_gbs:
        r["frac_of_read_stream"] = round(comp / stream_gbs, 4)
    return r


# ---- variants -----------------------------------------------------------------
def variant_reals(nrow, tg, n, N3):
    """(compulsory, nominal) reals per output site of one multi-vector half-Dslash:
    links 6 * nrow reals each, 8 per site, or 6 + 2/N3 in temporal gauge (the time links are read only
    on the slices x3 = 0 / 1); compulsory = each input vector once + each output once; nominal = all 8
    neighbours of every vector (the paper's count: n 570 / (8 (6 12 + n 9 6)))."""
    links = (6.0 + 2.0 / N3 if tg else 8.0) * 6 * nrow
    return links + 12.0 * n, links + 54.0 * n


def time_dslash_multi(torch, ctx, fU, fins, fouts, reps=10):
    for _ in range(2 if reps > 1 else 0):
        ctx.qcd_dslash_oe_multi(fU, fouts, fins)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        ctx.qcd_dslash_oe_multi(fU, fouts, fins)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def variants_sweep(q, torch, ctx, fU_full, dims, peak, nmulti=(1, 2, 3, 4, 6, 8), reps=10):
    """Dslash with the paper's traffic reductions, reported separately from the headline:
    link storage x temporal gauge x NMULTI.  Throughput does not depend on the link values, so the
    temporal-gauge rows run on the same links with the field marked (the kernel then skips the time links
    of x3 != 0); correctness of every variant is tests/test_gpu_variants.py's job."""
    Vh = int(np.prod(dims)) // 2
    rsize = 8 if ctx.precision == 64 else 4
    f12 = ctx.field(q.QCD_GAUGE_2ROW)
    ctx.qcd_gauge_compress(fU_full, f12)
    nmax = max(nmulti)
    fins = [ctx.field(q.QCD_SPINOR_EVEN) for _ in range(nmax)]
    fouts = [ctx.field(q.QCD_SPINOR_ODD) for _ in range(nmax)]
    g = torch.Generator(device=ctx.device).manual_seed(7)
    for f in fins:
        real = torch.float64 if ctx.precision == 64 else torch.float32
        f.buf.view(real).copy_(torch.randn(f.buf.numel() // rsize, generator=g, device=ctx.device, dtype=real))
    rows = []
    # the streaming ceiling of the same mix of read and write streams with stencil and arithmetic taken out (qcd_stream_mix):
    # link planes + 3 n vector planes read, 3 n planes written, every thread at its own index
    fmix = ctx.field(q.QCD_GAUGE)
    mix_cache = {}

    def mix_ceiling(read_planes, write_planes):
        key = (min(read_planes, 72), write_planes)          # the source field has 72 planes; GB/s is intensive
        if key not in mix_cache:
            ctx.qcd_stream_mix(fU_full, fmix, key[0], key[1], 2)
            mix_cache[key] = (key[0] + key[1]) * (fU_full.nbytes // 72) / ctx.qcd_stream_mix(fU_full, fmix, key[0], key[1], 5) / 1e6
        return mix_cache[key]

    for name, fU, nrow, tg in (("full18", fU_full, 3, 0), ("tworow12", f12, 2, 0), ("tworow12+temporal_gauge", f12, 2, 1)):
        ctx.qcd_gauge_set_temporal_unit(fU, bool(tg))
        for n in nmulti:
            ms = time_dslash_multi(torch, ctx, fU, fins[:n], fouts[:n], reps)
            comp, nom = variant_reals(nrow, tg, n, dims[3])
            gbs = comp * rsize * Vh / ms / 1e6
            ceil_gbs = mix_ceiling((6 if tg else 8) * 3 * nrow + 3 * n, 3 * n)
            rows.append({"links": name, "nmulti": n, "ms": round(ms, 5),
                         "tflops": round(FLOP_PER_SITE * n * Vh / ms / 1e9, 3),
                         "gbs_compulsory": round(gbs, 1), "frac_of_measured_copy_peak": round(gbs / peak, 4),
                         "stream_mix_ceiling_gbs": round(ceil_gbs, 1), "frac_of_stream_mix_ceiling": round(gbs / ceil_gbs, 4),
                         "ai_nominal_flop_per_byte": round(FLOP_PER_SITE * n / (nom * rsize), 3),
                         # Eq. (2) of the paper: attainable = min(peak, AI x bandwidth); the
                         # bandwidth term binds at every n here.  With the paper's NOMINAL bytes (no cache reuse
                         # of the neighbour vectors) a kernel whose L2 serves that reuse lands ABOVE this line,
                         # as the paper observes on A100; with compulsory bytes it cannot.
                         "eq2_attainable_tflops_nominal_ai": round(FLOP_PER_SITE * n / (nom * rsize) * peak / 1e3, 3),
                         "eq2_attainable_tflops_compulsory_ai": round(FLOP_PER_SITE * n / (comp * rsize) * peak / 1e3, 3)})
        ctx.qcd_gauge_set_temporal_unit(fU, False)
    for f in fins + fouts + [f12, fmix]:
        f.free()
    return rows


def cg_multi_report(q, torch, device, dims, prec, fU_full, m, ns=(1, 2, 4), iters=20):
    """n CG solves in lock step (qcd_cg_begin_multi / qcd_cg_iterate): ms per iteration and per right-hand side,
    on the paper's link storage (two rows + temporal gauge marking) and on full links."""
    rows = []
    ctx0 = fU_full.ctx
    for n in ns:
        ctx = q.Context(dims, prec, device=device, nrhs=n)
        fb = [ctx.field(q.QCD_SPINOR_EVEN) for _ in range(n)]
        fx = [ctx.field(q.QCD_SPINOR_EVEN) for _ in range(n)]
        real = torch.float64 if prec == 64 else torch.float32
        g = torch.Generator(device=device).manual_seed(11)
        for f in fb:
            f.buf.view(real).copy_(torch.randn(f.buf.numel() // (prec // 8), generator=g, device=device, dtype=real))
        for name, kind in (("full18", q.QCD_GAUGE), ("tworow12+temporal_gauge", q.QCD_GAUGE_2ROW)):
            if kind == q.QCD_GAUGE:
                fU = ctx.field(kind, buf=fU_full.buf)      # same device memory, descriptor of the new context
            else:
                f12 = ctx0.field(q.QCD_GAUGE_2ROW)
                ctx0.qcd_gauge_compress(fU_full, f12)
                fU = ctx.field(kind, buf=f12.buf)
            ctx.qcd_gauge_set_temporal_unit(fU, kind == q.QCD_GAUGE_2ROW)
            ctx.qcd_cg_begin_multi(fU, fb, fx, m, 1e-300, 1 << 30)
            ctx.qcd_cg_iterate(3)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.qcd_cg_iterate(iters)
            e1.record()
            torch.cuda.synchronize()
            ctx.qcd_cg_finish_multi()
            ms = e0.elapsed_time(e1) / iters
            rows.append({"links": name, "n": n, "ms_per_iter": round(ms, 5), "ms_per_iter_per_rhs": round(ms / n, 5)})
            fU.free()
        for f in fb + fx:
            f.free()
        ctx.close()
        torch.cuda.empty_cache()
    return rows


LOOP_NAMES = {1: "kernel-by-kernel enqueue", 2: "CUDA-graph replay, 16 iterations per launch",
              3: "persistent cooperative kernel (one launch per solve)"}


def small_lattice_report(q, torch, device):
    """configs[1] (16^4, links fit the L2): the solve is launch- and reduction-latency bound.
    The three solver loops of qcd_set_cg_loop: kernel-by-kernel enqueue, CUDA-graph replay of 16 iterations
    (side stream), and the persistent cooperative kernel (the library's choice at this size)."""
    dims = (16, 16, 16, 16)
    cfg, U, b = make_inputs(dims, 1)
    rows = []
    stream = torch.cuda.Stream(device=device)
    with torch.cuda.stream(stream):
        for prec, tol in ((64, cfg["tol64"]), (32, cfg["tol32"])):
            ctx = q.Context(dims, prec, stream=stream, device=device)
            fU = ctx.field(q.QCD_GAUGE).upload(U)
            fb = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
            fx = ctx.field(q.QCD_SPINOR_EVEN)
            for loop in (1, 2, 3):
                ctx.qcd_set_cg_loop(loop)
                ctx.qcd_cg_solve(fU, fb, fx, cfg["m"], tol, cfg["maxiter"])
                best = None
                for _ in range(3):
                    t0 = time.perf_counter()
                    info = ctx.qcd_cg_solve(fU, fb, fx, cfg["m"], tol, cfg["maxiter"])
                    wall = time.perf_counter() - t0
                    if best is None or info["seconds"] < best[0]["seconds"]:
                        best = (info, wall)
                info, wall = best
                rows.append({"loop": LOOP_NAMES[loop], "loop_that_ran": ctx.qcd_last_cg_loop(), "prec": prec, "tol": tol,
                             "iters": info["iters"], "converged": info["converged"],
                             "ms_per_solve_device": round(1e3 * info["seconds"], 4), "ms_per_solve_wall": round(1e3 * wall, 4),
                             "us_per_iter": round(1e6 * info["seconds"] / max(info["iters"], 1), 3)})
            ctx.close()
    return {"lattice": list(dims), "rows": rows}


def size_sweep_report(q, torch, device, sizes=((8, 8, 8, 8), (12, 12, 12, 12), (16, 16, 16, 16), (24, 24, 24, 24),
                                               (32, 32, 32, 32), (48, 48, 48, 12), (32, 32, 64, 64)), iters=200):
    """The paper's Fig. 3 experiment: Dslash and CG throughput against the lattice size, in
    single and double precision (the 64^4 point is the headline; 32^2 x 64^2 is the size beyond which the
    paper's MI250X curve degrades).  Dslash: D_oe launches replayed from a CUDA graph;
    CG: qcd_cg_solve with an unreachable tolerance and maxiter = `iters`, i.e. the solver loop the library picks
    for that size (persistent kernel while the lattice fits the L2, graph replay / kernel-by-kernel beyond).
    GFLOP/s with 570 flop per site (Dslash) and 2 x 570 + 72 flop per even site and iteration (CG)."""
    import qcd_inputs
    rows = []
    for dims in sizes:
        Vh = int(np.prod(dims)) // 2
        U = qcd_inputs.gauge_field(dims, "haar", seed=0)
        b = qcd_inputs.gaussian_source(dims, seed=1)
        for prec in (64, 32):
            stream = torch.cuda.Stream(device=device)
            with torch.cuda.stream(stream):
                ctx = q.Context(dims, prec, device=device, stream=stream)
                fU = ctx.field(q.QCD_GAUGE).upload(U)
                fb = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
                fx = ctx.field(q.QCD_SPINOR_EVEN)
                fo = ctx.field(q.QCD_SPINOR_ODD)
                ms_d = time_dslash_graph(torch, ctx, stream, fU, fb, fo)
                ctx.qcd_cg_solve(fU, fb, fx, 0.01, 1e-300, 20)
                secs = min(ctx.qcd_cg_solve(fU, fb, fx, 0.01, 1e-300, iters)["seconds"] for _ in range(2))
                rows.append({"lattice": list(dims), "prec": prec, "dslash_us": round(1e3 * ms_d, 3),
                             "dslash_gflops": round(FLOP_PER_SITE * Vh / ms_d / 1e6, 1),
                             "cg_loop": ctx.qcd_last_cg_loop(),
                             "cg_us_per_iter": round(1e6 * secs / iters, 3),
                             "cg_gflops": round(FLOP_PER_CG_ITER * Vh * iters / secs / 1e9, 1)})
                ctx.close()
    return rows


def update_routine_report(q, torch, device, peak, dims=(48, 48, 48, 48), iters=50):
    """The paper's Table 1 workload: bandwidth of the "CG update routine" on a 48^4 lattice,
    fp64 -- here the fused x += alpha p, r -= alpha Ap, |r|^2 kernel (288 B per even site) and the p update
    (144 B), timed by CUDA events around each launch inside running CG iterations."""
    cfg, U, b = make_inputs(dims, 4)
    Vh = int(np.prod(dims)) // 2
    ctx = q.Context(dims, 64, device=device)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    fb = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
    fx = ctx.field(q.QCD_SPINOR_EVEN)
    ctx.qcd_cg_begin(fU, fb, fx, cfg["m"], 1e-300, 1 << 30)
    ctx.qcd_cg_iterate(5)
    ctx.qcd_profile_enable(True)
    ctx.qcd_cg_iterate(iters)
    n_xr, ms_xr = ctx.qcd_profile_read(q.QCD_K_UPDATE_XR)
    n_p, ms_p = ctx.qcd_profile_read(q.QCD_K_UPDATE_P)
    ctx.qcd_profile_enable(False)
    ctx.qcd_cg_finish()
    ctx.close()
    xr = 36 * 8 * Vh / (ms_xr / n_xr) / 1e6
    pu = 18 * 8 * Vh / (ms_p / n_p) / 1e6
    return {"lattice": list(dims), "update_xr_norm_ms": round(ms_xr / n_xr, 5), "update_xr_norm_gbs": round(xr, 1),
            "update_xr_frac_of_measured_copy_peak": round(xr / peak, 4), "update_p_ms": round(ms_p / n_p, 5),
            "update_p_gbs": round(pu, 1),
            "paper_table1_gbs": {"OpenCL on A100": 1351, "CUDA on A100": 1317, "OpenCL on MI250x": 1134,
                                 "peaks": {"A100": 1555, "MI250x GCD": 1638},
                                 "source": "PAPER.md:56-62 (other hardware; context only)"}}


def config2_sweep_report(q, torch, device, peak, hbm_stream_gbs):
    """BASELINE.json configs[2]: "Dslash throughput sweep" at 32^4 in both precisions -- the block shapes of the one-vector
    kernel that qcd_set_dslash_variant exposes (0: 128 threads x 3 resident blocks, the library's choice; 1: 64 x 8;
    2: 256 x 2; 3: 128 x 4), D_oe launches replayed from a CUDA graph."""
    import qcd_inputs
    cfg, U, b = qcd_inputs.config_inputs(2)
    dims = cfg["dims"]
    Vh = int(np.prod(dims)) // 2
    names = {0: "128 threads x 3 blocks/SM (library's choice for the plain Dslash)", 1: "64 x 8", 2: "256 x 2", 3: "128 x 4"}
    rows = []
    for prec in (64, 32):
        stream = torch.cuda.Stream(device=device)
        with torch.cuda.stream(stream):
            ctx = q.Context(dims, prec, device=device, stream=stream)
            fU = ctx.field(q.QCD_GAUGE).upload(U)
            fb = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
            fo = ctx.field(q.QCD_SPINOR_ODD)
            for v in (0, 1, 2, 3):
                ctx.qcd_set_dslash_variant(v)
                ms = min(time_dslash_graph(torch, ctx, stream, fU, fb, fo) for _ in range(2))
                rows.append(dict(dslash_report(ms, Vh, prec // 8, peak, hbm_stream_gbs), prec=prec, block_shape=names[v]))
            ctx.close()
    return {"lattice": list(dims), "rows": rows}


# ---- oracle timings ----------------------------------------------------------------------------
def oracle_dslash_times(oracle, dims, U, b):
    """One oracle D_oe: best of 3 on all host threads, and one run on a single thread."""
    threads = oracle.num_threads()
    best = None
    for _ in range(3):
        t0 = time.perf_counter()
        oracle.dslash(dims, U, b, 1)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    oracle.set_num_threads(1)
    try:
        t0 = time.perf_counter()
        oracle.dslash(dims, U, b, 1)
        single = time.perf_counter() - t0
    finally:
        oracle.set_num_threads(threads)
    Vh = int(np.prod(dims)) // 2
    return {"oracle_dslash_ms": round(1e3 * best, 3), "oracle_threads": threads,
            "oracle_dslash_ms_single_thread": round(1e3 * single, 3),
            "oracle_dslash_gflops": round(FLOP_PER_SITE * Vh / best / 1e9, 3),
            "oracle_dslash_effective_gbs_nominal": round(REALS_DSLASH_NOMINAL * 8 * Vh / best / 1e9, 3)}


def golden(config: int, prec: int):
    p = os.path.join(ROOT, "tests", "golden", f"cg_config{config}_fp{prec}.json")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        return json.load(f)


def within_r8(it_gpu: int, it_ref: int) -> bool:
    """DESIGN.md reading R8: |it_gpu - it_oracle| <= max(2, ceil(0.02 it_oracle))."""
    return abs(it_gpu - it_ref) <= max(2, int(np.ceil(0.02 * it_ref)))


def config_row(cfg_index, cfg, prec, tol, dslash, cg_info, loop, true_resid, oracle_iters, oracle_iters_source,
               oracle_cg_seconds, oracle_cg_source, oracle_times, regime):
    it = cg_info["iters"]
    return {"config": cfg_index, "lattice": list(cfg["dims"]), "prec": prec, "links": cfg["links"], "m": cfg["m"], "tol": tol,
            "regime": regime, "dslash": dslash,
            "cg": {"loop": LOOP_NAMES.get(loop, str(loop)), "iters_gpu": it, "iters_oracle": oracle_iters,
                   "iters_oracle_source": oracle_iters_source,
                   "iters_within_R8": (within_r8(it, oracle_iters) if oracle_iters else None),
                   "converged": cg_info["converged"], "s_per_solve": round(cg_info["seconds"], 6),
                   "ms_per_iter": round(1e3 * cg_info["seconds"] / max(it, 1), 5),
                   "rel_resid_recurrence": cg_info["rel_resid"], "true_resid_oracle_fp64": true_resid,
                   # north_star's CG criterion: the TRUE residual, recomputed by the oracle in fp64, <= tol.  Plain fp32 CG on
                   # Haar links cannot meet it (R11); the mixed-precision solver can and does.
                   "meets_north_star_true_resid": bool(true_resid <= tol)},
            "oracle": dict(oracle_times, oracle_cg_seconds=oracle_cg_seconds, oracle_cg_source=oracle_cg_source)}


def per_config_report(q, torch, device, peak, hbm_stream_gbs, side):
    """SURVEY.md Sec. 8(d) "Reported per config" for BASELINE.json configs 0-3 (config 4 is assembled by run_all from
    the headline run): GPU Dslash and full CG solve next to the oracle's own D_oe and full CG on the host cores."""
    import oracle
    import qcd_inputs
    rows = []
    # the small-lattice denominator: L2 -> SM read rate over an L2-resident gauge field (16^4 fp64 links, 37.7 MB)
    c16 = q.Context((16, 16, 16, 16), 64, device=device)
    f16 = c16.field(q.QCD_GAUGE)
    f16.buf.zero_()
    l2_stream = f16.nbytes / c16.qcd_stream_read_resident(f16, 200) / 1e6
    f16.free()
    c16.close()
    for ci in (0, 1, 2, 3):
        cfg, U, b = qcd_inputs.config_inputs(ci)
        dims, m = cfg["dims"], cfg["m"]
        Vh = int(np.prod(dims)) // 2
        log(f"  config {ci} ({cfg['name']}): oracle D_oe and CG")
        otimes = oracle_dslash_times(oracle, dims, U, b)
        t0 = time.perf_counter()
        _, o64 = oracle.cg(dims, U, b, m, cfg["tol64"], cfg["maxiter"])
        o64_s = time.perf_counter() - t0
        for prec in (64, 32):
            tol = cfg["tol64"] if prec == 64 else cfg["tol32"]
            if tol is None:
                continue
            rsize = prec // 8
            Ur, br = (U, b) if prec == 64 else (U.astype(np.complex64), b.astype(np.complex64))
            if prec == 64:
                oit, osrc, osec, osecsrc = o64["iters"], "live", round(o64_s, 3), "live (full solve)"
            else:
                t0 = time.perf_counter()
                _, o32 = oracle.cg(dims, Ur, br, m, tol, cfg["maxiter"])
                oit, osrc, osec, osecsrc = o32["iters"], "live (f32 oracle variant, DESIGN.md R9)", round(time.perf_counter() - t0, 3), "live (full solve)"
            stream = torch.cuda.Stream(device=device)
            with torch.cuda.stream(stream):
                ctx = q.Context(dims, prec, device=device, stream=stream)
                fU = ctx.field(q.QCD_GAUGE).upload(U)
                fb = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
                fx = ctx.field(q.QCD_SPINOR_EVEN)
                fo = ctx.field(q.QCD_SPINOR_ODD)
                resident = fU.nbytes + 6 * fb.nbytes <= L2_RESIDENT_BYTES
                ms_d = time_dslash_graph(torch, ctx, stream, fU, fb, fo)
                ctx.qcd_cg_solve(fU, fb, fx, m, tol, cfg["maxiter"])
                info = min((ctx.qcd_cg_solve(fU, fb, fx, m, tol, cfg["maxiter"]) for _ in range(2)), key=lambda i: i["seconds"])
                loop = ctx.qcd_last_cg_loop()
                x = fx.download()
                ctx.close()
            true = oracle.true_residual(dims, Ur, br, x, m)
            d = dslash_report(ms_d, Vh, rsize, peak, l2_stream if resident else hbm_stream_gbs)
            d["read_stream_denominator"] = "L2-resident read stream (16^4 links re-read 200 x inside one launch)" if resident else "HBM read stream (64^4 links)"
            rows.append(config_row(ci, cfg, prec, tol, d, info, loop, true, oit, osrc, osec, osecsrc, otimes,
                                   "L2-resident (not an HBM measurement)" if resident else "HBM"))
    side["l2_resident_read_stream_gbs"] = round(l2_stream, 1) if l2_stream else None
    return rows


# ---- everything --------------------------------------------------------------------------------
def run_all(args, q, torch, ctx, out, side, cfg, dims, U, b, hb, hx, fU, fb, fx, fo, peak, stream_gbs):
    """Fills `side` (sidecar) and the headline keys of `out` that need these measurements."""
    import oracle
    V = int(np.prod(dims))
    Vh = V // 2
    m = cfg["m"]
    full = dims == (64, 64, 64, 64)
    state = {}

    def do_dslash64():
        r = dslash_report(time_dslash(torch, ctx, fU, fb, fo), Vh, 8, peak, stream_gbs)
        out["dslash_gbs_fp64"] = r["gbs_compulsory"]
        out["dslash_frac_hbm_fp64"] = r["frac_of_measured_copy_peak"]
        return r
    section(side, "dslash_fp64", do_dslash64)

    def do_cg64():
        info = ctx.qcd_cg_solve(fU, fb, fx, m, cfg["tol64"], cfg["maxiter"])
        x64 = fx.download()
        t0 = time.time()
        true64 = oracle.true_residual(dims, U, b, x64, m)
        state["oracle_apply_M_seconds"] = round(time.time() - t0, 2)
        state["cg64"], state["true64"] = info, true64
        out["cg_s_per_solve_fp64"] = round(info["seconds"], 4)
        out["cg_iters_fp64"] = info["iters"]
        return {"tol": cfg["tol64"], "iters": info["iters"], "converged": info["converged"], "loop": ctx.qcd_last_cg_loop(),
                "s_per_solve": round(info["seconds"], 4),
                "ms_per_iter": round(1e3 * info["seconds"] / max(info["iters"], 1), 5),
                "rel_resid_recurrence": info["rel_resid"], "true_resid_oracle_fp64": true64,
                "meets_north_star_true_resid": bool(true64 <= cfg["tol64"])}
    section(side, "cg_fp64", do_cg64)

    # CPU baseline: the oracle as it stands, a bounded sample of the same workload
    def do_cpu():
        nit = 12                                            # ~6-10 s of oracle time at 64^4 on 16 cores
        t0 = time.time()
        _, oinfo = oracle.cg(dims, U, b, m, 1e-300, nit)
        t_or = time.time() - t0
        state["oracle_s_per_iter"] = t_or / max(oinfo["iters"], 1)
        cb = {"value": round(REALS_ITER_NOMINAL * 8 * Vh * oinfo["iters"] / t_or / 1e9, 3), "unit": UNIT,
              "cores": oracle.num_threads(), "kind": "oracle",
              "sample": f"{nit} CG iterations of the same {'x'.join(map(str, dims))} fp64 solve, oracle set-up included; {t_or:.1f} s"}
        out["cpu_baseline"] = cb
        return dict(cb, oracle_apply_M_seconds=state.get("oracle_apply_M_seconds"))
    section(side, "cpu_baseline", do_cpu)

    # the ONE C-ABI call that takes host buffers, for a full solve (upload b, solve, download x inside info.seconds)
    def do_e2e_full():
        info = ctx.qcd_cg_solve_host(fU, fb, fx, hb.data_ptr(), hx.data_ptr(), m, cfg["tol64"], cfg["maxiter"])
        nbytes = hb.numel() * hb.element_size()
        return {"call": "qcd_cg_solve_host (pinned host b and x; the 9.7 GB link upload is outside)", "iters": info["iters"],
                "converged": info["converged"], "seconds_including_copies": round(info["seconds"], 4),
                "value": round(REALS_ITER_NOMINAL * 8 * Vh * info["iters"] / info["seconds"] / 1e9, 2), "unit": UNIT,
                "h2d_bytes": int(nbytes), "d2h_bytes": int(nbytes),
                "solve_only_seconds": state["cg64"]["seconds"] if "cg64" in state else None}
    section(side, "e2e_full_solve", do_e2e_full)

    section(side, "oracle_64" if full else "oracle_headline_lattice", lambda: oracle_dslash_times(oracle, dims, U, b))

    # ---- variants, reported separately from the headline ----
    c32 = q.Context(dims, 32, device=ctx.device)
    gU = c32.field(q.QCD_GAUGE)
    ctx.qcd_field_convert(gU, fU)                          # fp32 links = round-to-nearest of the fp64 links, on the device
    gx = c32.field(q.QCD_SPINOR_EVEN)
    go = c32.field(q.QCD_SPINOR_ODD)
    inner_tol = 1e-3
    s64 = lambda: state["cg64"]["seconds"] if "cg64" in state else float("nan")  # noqa: E731

    def do_mixed():
        # mixed-precision defect-correction CG to the fp64 tolerance (R21)
        mi = ctx.qcd_cg_solve_mixed(c32, fU, gU, fb, fx, gx, c32.field(q.QCD_SPINOR_EVEN), m, cfg["tol64"], inner_tol,
                                    4 * cfg["maxiter"])
        true = oracle.true_residual(dims, U, b, fx.download(), m)
        return {"tol": cfg["tol64"], "inner_tol": inner_tol, "converged": mi["converged"], "outer": mi["outer"],
                "inner_iters_fp32": mi["inner_iters"], "m_applications_fp64": mi["m_applications_fp64"],
                "s_per_solve": round(mi["seconds"], 4), "true_resid_device_fp64": mi["true_resid"],
                "true_resid_oracle_fp64": true, "meets_north_star_true_resid": bool(true <= cfg["tol64"]),
                "speedup_vs_cg_fp64": round(s64() / max(mi["seconds"], 1e-9), 3)}
    section(side, "cg_mixed", do_mixed)

    def do_paper_storage():
        # the same two solves on the paper's link storage: temporal gauge fixed on the device,
        # two rows stored; the source is rotated in (b' = g b), the solution rotated back (x = g^dagger x'),
        # and the oracle checks the residual against the ORIGINAL links and source
        fUf, fg = ctx.field(q.QCD_GAUGE), ctx.field(q.QCD_COLOUR_MATRIX)
        ctx.qcd_gauge_fix_temporal(fU, fUf, fg)
        f12 = ctx.field(q.QCD_GAUGE_2ROW)
        ctx.qcd_gauge_compress(fUf, f12)
        fUf.free()
        g12 = c32.field(q.QCD_GAUGE_2ROW)
        ctx.qcd_field_convert(g12, f12)
        fbr = ctx.field(q.QCD_SPINOR_EVEN)
        ctx.qcd_spinor_rotate(fg, fbr, fb)
        info = ctx.qcd_cg_solve(f12, fbr, fx, m, cfg["tol64"], cfg["maxiter"])
        ctx.qcd_spinor_rotate(fg, fx, fx, dagger=True)
        side["cg_fp64_tworow_temporal_gauge"] = {
            "tol": cfg["tol64"], "iters": info["iters"], "converged": info["converged"], "s_per_solve": round(info["seconds"], 4),
            "ms_per_iter": round(1e3 * info["seconds"] / max(info["iters"], 1), 5),
            "true_resid_oracle_fp64_original_links": oracle.true_residual(dims, U, b, fx.download(), m),
            "speedup_vs_cg_fp64": round(s64() / max(info["seconds"], 1e-9), 3)}
        mi = ctx.qcd_cg_solve_mixed(c32, f12, g12, fbr, fx, gx, c32.field(q.QCD_SPINOR_EVEN), m, cfg["tol64"], inner_tol,
                                    4 * cfg["maxiter"])
        ctx.qcd_spinor_rotate(fg, fx, fx, dagger=True)
        side["cg_mixed_tworow_temporal_gauge"] = {
            "tol": cfg["tol64"], "inner_tol": inner_tol, "converged": mi["converged"], "outer": mi["outer"],
            "inner_iters_fp32": mi["inner_iters"], "s_per_solve": round(mi["seconds"], 4),
            "true_resid_device_fp64": mi["true_resid"],
            "true_resid_oracle_fp64_original_links": oracle.true_residual(dims, U, b, fx.download(), m),
            "speedup_vs_cg_fp64": round(s64() / max(mi["seconds"], 1e-9), 3)}
        for f in (f12, g12, fg, fbr):
            f.free()
    section(side, "paper_link_storage_solves", do_paper_storage)

    section(side, "variants_fp64", lambda: {"lattice": list(dims), "dslash": variants_sweep(q, torch, ctx, fU, dims, peak)})
    section(side, "cg_multi_fp64", lambda: cg_multi_report(q, torch, ctx.device, dims, 64, fU, m))

    # ---- fp32 ----
    U32, b32 = U.astype(np.complex64), b.astype(np.complex64)
    gb = c32.field(q.QCD_SPINOR_EVEN).upload(b32)

    def do_dslash32():
        r = dslash_report(time_dslash(torch, c32, gU, gb, go), Vh, 4, peak, stream_gbs)
        out["dslash_gbs_fp32"] = r["gbs_compulsory"]
        return r
    section(side, "dslash_fp32", do_dslash32)
    section(side, "variants_fp32", lambda: {"lattice": list(dims), "dslash": variants_sweep(q, torch, c32, gU, dims, peak)})

    def do_cg32():
        if not cfg["tol32"]:
            return None
        info = c32.qcd_cg_solve(gU, gb, gx, m, cfg["tol32"], cfg["maxiter"])
        true = oracle.true_residual(dims, U32, b32, gx.download(), m)
        state["cg32"], state["true32"] = info, true
        out["cg_s_per_solve_fp32"] = round(info["seconds"], 4)
        return {"tol": cfg["tol32"], "iters": info["iters"], "converged": info["converged"], "loop": c32.qcd_last_cg_loop(),
                "s_per_solve": round(info["seconds"], 4),
                "ms_per_iter": round(1e3 * info["seconds"] / max(info["iters"], 1), 5),
                "rel_resid_recurrence": info["rel_resid"], "true_resid_oracle_fp64": true,
                "meets_north_star_true_resid": bool(true <= cfg["tol32"]),
                "note": "plain fp32 CG on Haar links: the recurrence meets tol, the TRUE residual stalls near 1e-2 (DESIGN.md R11); "
                        "it does NOT meet north_star's CG criterion -- cg_mixed does"}
    section(side, "cg_fp32", do_cg32)
    del U32

    # ---- per-config table ----
    def do_table():
        rows = per_config_report(q, torch, ctx.device, peak, stream_gbs, side) if full else []
        if full and "cg64" in state:
            ot = side.get("oracle_64", {})
            g64, g32 = golden(4, 64), golden(4, 32)
            ext = (round(state["oracle_s_per_iter"] * g64["iters"], 1) if g64 and "oracle_s_per_iter" in state else None)
            d64 = dict(side.get("dslash_fp64", {}), read_stream_denominator="HBM read stream (64^4 links)")
            rows.append(config_row(4, cfg, 64, cfg["tol64"], d64, state["cg64"], side["cg_fp64"]["loop"], state["true64"],
                                   g64["iters"] if g64 else None, "tests/golden/cg_config4_fp64.json (oracle, offline)",
                                   ext, "EXTRAPOLATED: live oracle s/iteration (12-iteration sample) x golden iteration count", ot, "HBM"))
            if "cg32" in state:
                d32 = dict(side.get("dslash_fp32", {}), read_stream_denominator="HBM read stream (64^4 links)")
                rows.append(config_row(4, cfg, 32, cfg["tol32"], d32, state["cg32"], side["cg_fp32"]["loop"], state["true32"],
                                       g32["iters"] if g32 else None, "tests/golden/cg_config4_fp32.json (f32 oracle variant, offline)",
                                       g32["oracle_seconds"] if g32 else None,
                                       f"golden file (offline run on {g32['oracle_threads']} threads)" if g32 else None, ot, "HBM"))
        return rows
    section(side, "per_config", do_table)

    # ---- the paper's own experiments on this hardware ----
    if full:
        def do_table2():
            # the paper's own NMULTI experiment: 32^4, two-row links, temporal gauge (Table 2)
            d32 = (32, 32, 32, 32)
            _, U_32, _ = make_inputs(d32, 2)
            t2 = {"lattice": list(d32), "paper_A100_tflops": {"fp32": {1: 2.244, 2: 2.532, 3: 2.953, 4: 3.205, 6: 3.090, 8: 3.006},
                                                               "fp64": {1: 1.245, 2: 1.530, 3: 1.929, 4: 2.199, 6: 2.039, 8: 2.026},
                                                               "source": "PAPER.md:84-98 Table 2 (A100, OpenCL; other hardware, context only)"}}
            for prec in (64, 32):
                c = q.Context(d32, prec, device=ctx.device)
                f = c.field(q.QCD_GAUGE).upload(U_32)
                t2[f"fp{prec}"] = variants_sweep(q, torch, c, f, d32, peak)
                f.free()
                c.close()
            return t2
        section(side, "variants_table2_32x32x32x32", do_table2)
        section(side, "config2_dslash_block_shape_sweep", lambda: config2_sweep_report(q, torch, ctx.device, peak, stream_gbs))
        section(side, "cg_small_lattice", lambda: small_lattice_report(q, torch, ctx.device))
        section(side, "cg_update_routine_48x48x48x48", lambda: update_routine_report(q, torch, ctx.device, peak))
        section(side, "size_sweep_fig3", lambda: size_sweep_report(q, torch, ctx.device))
    side["paper_context"] = {"A100_OpenCL_dslash_fp64_TFLOPs_32^4_12real_links_gaugefixed": 1.245,
                             "A100_OpenCL_cg_update_GBs_48^4_fp64": 1351, "source": "PAPER.md:59,87 (other hardware; context only)"}
    # copy the headline keys filled above into the sidecar as well
    for k in ("cpu_baseline", "dslash_gbs_fp64", "dslash_frac_hbm_fp64", "dslash_gbs_fp32", "cg_s_per_solve_fp64",
              "cg_s_per_solve_fp32", "cg_iters_fp64"):
        if k in out:
            side[k] = out[k]
    try:
        c32.close()
    except Exception:  # noqa: BLE001
        pass

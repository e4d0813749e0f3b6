#!/usr/bin/env python
"""bench.py -- staggered Dslash + CG hot path on B200 (one JSON line on stdout; rank 0 only).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--lattice 64,64,64,64] [--quick]

Workload (config.workload): BASELINE.json configs[4] -- 64^4 lattice, Haar-random SU(3) links
(seed 0), Gaussian even-site source (seed 1), m = 0.01, fp64 -- the configuration the metric is
quoted on.  Inputs (9.7 GB of links) are far larger than the 126 MB L2, so no L2 flush is needed
between timed iterations.

A STEP is one Conjugate-Gradient iteration on M = m^2 - D_eo D_oe = one pass over every row of
SURVEY.md Sec. 8(a): D_oe, D_eo + M epilogue + <p,Mp>, alpha, fused x/r update + |r|^2, beta and
the stop test, the p update -- all in our CUDA kernels, scalars resident on the device.

  value : effective GB/s = nominal bytes of one iteration (3648 B per even site in fp64:
          two half-Dslash at 1584 B/site (BASELINE.json north_star) + 480 B of vector traffic)
          x sites x K / device time of K iterations.  Inputs resident in HBM.
  e2e   : the same K iterations through the C-ABI with HOST buffers: qcd_field_upload of the
          source from pinned memory, K x (qcd_cg_iterate(1) + qcd_cg_poll, a 72-byte D2H read
          of the residual after every step), qcd_field_download of the iterate to pinned memory.
  roofline : the Dslash kernel (D_oe launches inside the timed region, CUDA events on the
          launching stream), algorithmic = COMPULSORY DRAM bytes 1248 B/site (each link once,
          each spinor once, one store), against MEASURED_PEAKS.json hbm_gbs.
  cpu_baseline / --impl reference : the CPU oracle as it stands on the host cores.

N > 1: replicas only: every rank runs the same workload on its own
GPU, no data-path collective; value = sum of units / max-over-ranks device time.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

# ---- byte / flop model -------------------
FLOP_PER_SITE = 570
REALS_DSLASH_NOMINAL = 198               # 8 links x 18 + 8 vectors x 6 + 1 vector written (north_star: 1584 B fp64)
REALS_DSLASH_COMPULSORY = 156            # 8 links x 18 + 1 vector read + 1 written          (1248 B fp64)
REALS_ITER_NOMINAL = 2 * 198 + 6 + 36 + 18      # + epilogue read of p, x/r update (6 vectors), p update (3 vectors) = 456
REALS_ITER_COMPULSORY = 2 * 156 + 6 + 36 + 18   # = 372 (2976 B fp64)
THEORETICAL_HBM_GBS = 8184.0             # 3996 MHz x 2 (DDR) x 8192 bit / 8 -- nvidia-smi max memory clock; context only

METRIC = "staggered CG-iteration effective GB/s (two half-Dslash at 1584 B/site + CG vector kernels), 64^4 fp64"
UNIT = "GB/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--lattice", default=None, help="override dims, e.g. 16,16,16,16 (testing only)")
    ap.add_argument("--quick", action="store_true", help="skip the extra reports (full solves, fp32, cpu_baseline)")
    ap.add_argument("--variants-only", action="store_true",
                    help="run only the Dslash variant sweep (two-row / temporal gauge / NMULTI) and print it; used for ncu captures")
    ap.add_argument("--prec", type=int, default=64, choices=(64, 32),
                    help="precision of --variants-only, and of the timed CG iterations (32: the fp32 path of the same "
                         "workload, reported with dtype f32 and without the extra reports; the default line is fp64)")
    ap.add_argument("--nmulti", default="1,2,3,4,6,8", help="NMULTI values of --variants-only")
    ap.add_argument("--reps", type=int, default=10, help="timed launches per variant of --variants-only")
    ap.add_argument("--kernel", type=int, default=0,
                    help="qcd_set_dslash_variant for --variants-only (0 default choice, 4 staged kernel, 5 register kernel)")
    return ap.parse_args()


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_traffic(prec: int):
    """ncu-measured DRAM bytes per Dslash launch, recorded in profiles/ (text, committed); None if absent."""
    p = os.path.join(ROOT, "profiles", "dslash_traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        rows = dict(line.strip().split(",", 1) for line in f if "," in line)
    v = rows.get(f"fp{prec}_64x64x64x64_bytes_per_launch")
    return int(v) if v is not None else None


# ---- clocks ---------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz, self.power = [], set(), None, []
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception as e:  # pragma: no cover
            self.nv, self.err = None, repr(e)

    def _run(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1e3)
            except Exception:
                pass
            time.sleep(0.01)

    def __enter__(self):
        if self.nv:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples),
                "power_w": round(float(np.median(self.power)), 1) if self.power else None}


# ---- multi-rank plumbing ---------------------------------------------------------------------
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def aggregate_over_ranks(local_ms: float, local_units: float, backend_device=None):
    """(max-over-ranks time, sum-over-ranks units).  No data-path collective exists; this is the
    only communication in the bench.  Works with gloo (CPU tensors) and nccl (CUDA tensors)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return local_ms, local_units
    dev = backend_device if backend_device is not None else "cpu"
    t = torch.tensor([local_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([local_units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ---- our arm ---------------------------------------------------------------------------------
def make_inputs(dims, cfg_index=4):
    import qcd_inputs
    cfg = dict(qcd_inputs.CONFIGS[cfg_index])
    cfg["dims"] = tuple(dims)
    U = qcd_inputs.gauge_field(cfg["dims"], cfg["links"], seed=0, eps=cfg["eps"])
    b = qcd_inputs.gaussian_source(cfg["dims"], seed=1, parity=0)
    return cfg, U, b


def time_dslash(q, torch, ctx, fU, fin, fout, n=20):
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
    for name, fU, nrow, tg in (("full18", fU_full, 3, 0), ("tworow12", f12, 2, 0), ("tworow12+temporal_gauge", f12, 2, 1)):
        ctx.qcd_gauge_set_temporal_unit(fU, bool(tg))
        for n in nmulti:
            ms = time_dslash_multi(torch, ctx, fU, fins[:n], fouts[:n], reps)
            comp, nom = variant_reals(nrow, tg, n, dims[3])
            gbs = comp * rsize * Vh / ms / 1e6
            rows.append({"links": name, "nmulti": n, "ms": round(ms, 5),
                         "tflops": round(FLOP_PER_SITE * n * Vh / ms / 1e9, 3),
                         "gbs_compulsory": round(gbs, 1), "frac_of_measured_copy_peak": round(gbs / peak, 4),
                         "ai_nominal_flop_per_byte": round(FLOP_PER_SITE * n / (nom * rsize), 3),
                         # Eq. (2) of the paper: attainable = min(peak, AI x bandwidth); the
                         # bandwidth term binds at every n here.  With the paper's NOMINAL bytes (no cache reuse
                         # of the neighbour vectors) a kernel whose L2 serves that reuse lands ABOVE this line,
                         # as the paper observes on A100; with compulsory bytes it cannot.
                         "eq2_attainable_tflops_nominal_ai": round(FLOP_PER_SITE * n / (nom * rsize) * peak / 1e3, 3),
                         "eq2_attainable_tflops_compulsory_ai": round(FLOP_PER_SITE * n / (comp * rsize) * peak / 1e3, 3)})
        ctx.qcd_gauge_set_temporal_unit(fU, False)
    for f in fins + fouts + [f12]:
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
            for loop, name in ((1, "kernel-by-kernel enqueue"), (2, "CUDA-graph replay, 16 iterations per launch"),
                               (3, "persistent cooperative kernel (one launch per solve)")):
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
                rows.append({"loop": name, "prec": prec, "tol": tol, "iters": info["iters"], "converged": info["converged"],
                             "ms_per_solve_device": round(1e3 * info["seconds"], 4), "ms_per_solve_wall": round(1e3 * wall, 4),
                             "us_per_iter": round(1e6 * info["seconds"] / max(info["iters"], 1), 3)})
            ctx.close()
    return {"lattice": list(dims), "rows": rows}


FLOP_PER_CG_ITER = 2 * FLOP_PER_SITE + 72     # per even site: two half-Dslash + m^2 p - (6 fma) + two dots (2 x 12) + x, r, p updates (3 x 12)


def size_sweep_report(q, torch, device, sizes=((8, 8, 8, 8), (12, 12, 12, 12), (16, 16, 16, 16), (24, 24, 24, 24),
                                               (32, 32, 32, 32), (48, 48, 48, 12), (32, 32, 64, 64)), iters=200):
    """The paper's Fig. 3 experiment: Dslash and CG throughput against the lattice size, in
    single and double precision (the 64^4 point is the headline above; 32^2 x 64^2 is the size beyond which the
    paper's MI250X curve degrades).  Dslash: 20 back-to-back D_oe launches;
    CG: qcd_cg_solve with an unreachable tolerance and maxiter = `iters`, i.e. the solver loop the library picks
    for that size (persistent kernel while the lattice fits the L2, kernel-by-kernel beyond).  GFLOP/s with
    570 flop per site (Dslash) and 2 x 570 + 72 flop per even site and iteration (CG)."""
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
                # 20 launches captured in one CUDA graph: below 16^4 a Python-driven launch loop would
                # time the host, not the kernel
                ctx.qcd_dslash_oe(fU, fo, fb)
                stream.synchronize()
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph, stream=stream):
                    for _ in range(20):
                        ctx.qcd_dslash_oe(fU, fo, fb)
                graph.replay()
                stream.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                for _ in range(5):
                    graph.replay()
                e1.record(stream)
                stream.synchronize()
                ms_d = e0.elapsed_time(e1) / 100
                del graph
            ctx.qcd_cg_solve(fU, fb, fx, 0.01, 1e-300, 20)
            secs = min(ctx.qcd_cg_solve(fU, fb, fx, 0.01, 1e-300, iters)["seconds"] for _ in range(2))
            rows.append({"lattice": list(dims), "prec": prec, "dslash_us": round(1e3 * ms_d, 3),
                         "dslash_gflops": round(FLOP_PER_SITE * Vh / ms_d / 1e6, 1),
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


def dslash_report(ms, Vh, rsize, peak):
    comp = REALS_DSLASH_COMPULSORY * rsize * Vh / ms / 1e6
    return {"ms": round(ms, 5), "gflops": round(FLOP_PER_SITE * Vh / ms / 1e6, 1),
            "effective_gbs_nominal": round(REALS_DSLASH_NOMINAL * rsize * Vh / ms / 1e6, 1),
            "gbs_compulsory": round(comp, 1),
            "frac_of_measured_copy_peak": round(comp / peak, 4),
            "frac_of_theoretical_8184": round(comp / THEORETICAL_HBM_GBS, 4)}


def run_ours(args):
    import torch
    import paper_2502_03249_b200 as q

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))

    dims = tuple(int(v) for v in args.lattice.split(",")) if args.lattice else (64, 64, 64, 64)
    K, W = args.steps, args.warmup
    peak, peak_src = load_peaks()
    t_setup = time.time()
    V = int(np.prod(dims))
    Vh = V // 2
    prec = args.prec
    rsize = prec // 8
    ctx = q.Context(dims, prec, device=dev)
    fU = ctx.field(q.QCD_GAUGE)
    fb = ctx.field(q.QCD_SPINOR_EVEN)
    fx = ctx.field(q.QCD_SPINOR_EVEN)
    fo = ctx.field(q.QCD_SPINOR_ODD)
    if rank == 0:
        cfg, U, b = make_inputs(dims)
        fU.upload(U)
        fb.upload(b)
    else:
        # replicas: every rank works on the SAME inputs.  Rank 0 generates them (9.7 GB of links on the
        # host) and the device images are broadcast once during set-up -- plumbing, outside every timed
        # region; eight ranks generating 64^4 on one host would need ~200 GB of host memory.
        import qcd_inputs
        cfg, U, b = dict(qcd_inputs.CONFIGS[4]), None, None
        cfg["dims"] = tuple(dims)
    if world > 1:
        import torch.distributed as dist
        dist.broadcast(fU.buf, src=0)
        dist.broadcast(fb.buf, src=0)
        if rank != 0:
            b = fb.download()                  # the canonical host source (for the e2e leg) through the library
    m, tol64 = cfg["m"], cfg["tol64"]
    t_setup = time.time() - t_setup

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()

    # ---------------- timed region: K CG iterations, inputs resident --------------------------
    ctx.qcd_cg_begin(fU, fb, fx, m, 1e-300, 1 << 30)      # tol far below reach: every step does full work
    ctx.qcd_cg_iterate(W)
    barrier()
    torch.cuda.synchronize()
    ctx.qcd_profile_enable(True)
    launches0 = ctx.qcd_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local_rank) as clocks:
        e0.record()
        ctx.qcd_cg_iterate(K)
        e1.record()
        torch.cuda.synchronize()
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = ctx.qcd_launch_count() - launches0
    prof = {k: ctx.qcd_profile_read(k) for k in range(4)}
    ctx.qcd_profile_enable(False)
    state, it_done, _ = ctx.qcd_cg_poll()
    ctx.qcd_cg_finish()
    assert state == 0 and it_done == W + K, (state, it_done)

    bytes_iter = REALS_ITER_NOMINAL * rsize * Vh
    ms_max, units = aggregate_over_ranks(ms_total, float(K) * bytes_iter, dev if world > 1 else None)
    value = units / ms_max / 1e6

    # ---------------- e2e: host buffers through the C-ABI --------------------------------------
    hb = torch.from_numpy(np.ascontiguousarray(b, dtype=ctx.cdtype)).pin_memory()
    hx = torch.empty_like(hb).pin_memory()
    torch.cuda.synchronize()
    barrier()
    t0 = time.perf_counter()
    e0.record()
    ctx._check(ctx.lib.qcd_field_upload(fb.handle, hb.data_ptr()), "qcd_field_upload")
    ctx.qcd_cg_begin(fU, fb, fx, m, 1e-300, 1 << 30)
    rr_last = None
    for _ in range(K):
        ctx.qcd_cg_iterate(1)
        _, _, rr_last = ctx.qcd_cg_poll()                  # D2H read of the step's result (residual)
    ctx.qcd_cg_finish()
    ctx._check(ctx.lib.qcd_field_download(fx.handle, hx.data_ptr()), "qcd_field_download")
    e1.record()
    torch.cuda.synchronize()
    e2e_wall_ms = (time.perf_counter() - t0) * 1e3
    e2e_ms = e0.elapsed_time(e1)
    e2e_ms_max, e2e_units = aggregate_over_ranks(max(e2e_ms, e2e_wall_ms), float(K) * bytes_iter, dev if world > 1 else None)
    spinor_host_bytes = hb.numel() * hb.element_size()
    e2e = {"value": round(e2e_units / e2e_ms_max / 1e6, 2), "unit": UNIT,
           "h2d_bytes_per_step": int(spinor_host_bytes / K), "d2h_bytes_per_step": int(spinor_host_bytes / K + 72),
           "ms_total": round(e2e_ms_max, 3),
           "what": "qcd_field_upload(b, pinned host) + K x [qcd_cg_iterate(1) + qcd_cg_poll (D2H of the residual)] + "
                   "qcd_field_download(x, pinned host); host copies amortised over the K steps of the solve"}
    del hb, hx

    # ---------------- roofline of the dominant kernel ------------------------------------------
    n_ds, ms_ds = prof[q.QCD_K_DSLASH]
    ds_ms = ms_ds / max(n_ds, 1)
    achieved = REALS_DSLASH_COMPULSORY * rsize * Vh / ds_ms / 1e6
    # read-only streaming ceiling over the gauge field's own bytes (qcd_stream_read: the Dslash's link-load
    # instruction and nothing else), measured after the timed region; the third denominator beside the
    # copy peak and the theoretical peak
    ctx.qcd_stream_read(fU, 3)
    stream_gbs = fU.nbytes / ctx.qcd_stream_read(fU, 10) / 1e6
    roofline = {"bound": "hbm", "kernel": f"dslash_kernel<{'double' if prec == 64 else 'float'},MODE0> (D_oe inside the CG iteration)",
                "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s", "frac": round(achieved / peak, 4),
                "peak_source": peak_src, "traffic": load_traffic(prec) if dims == (64, 64, 64, 64) else None,
                "algorithmic_bytes_per_launch": REALS_DSLASH_COMPULSORY * rsize * Vh,
                "avg_launch_ms": round(ds_ms, 5), "launches_timed": n_ds,
                "frac_of_theoretical_8184": round(achieved / THEORETICAL_HBM_GBS, 4),
                "read_stream_gbs": round(stream_gbs, 1), "frac_of_read_stream": round(achieved / stream_gbs, 4)}
    kernel_ms = {name: round(prof[k][1] / max(prof[k][0], 1), 5) for name, k in
                 (("dslash_oe", q.QCD_K_DSLASH), ("dslash_eo_epilogue_dot", q.QCD_K_DSLASH_EPI),
                  ("update_xr_norm", q.QCD_K_UPDATE_XR), ("update_p", q.QCD_K_UPDATE_P))}

    out = {
        "metric": METRIC if prec == 64 else METRIC.replace("fp64", "fp32").replace("1584", "792"),
        "value": round(value, 2), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": round(ms_max / K, 5), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": f"f{prec}", "data": "synthetic (seeded Haar SU(3) links, Gaussian source; BASELINE.json configs[4])",
        "config": {"workload": f"{'x'.join(map(str, dims))} staggered CG iteration, Haar links, m={m}, fp{prec}, full 18-real links",
                   "lattice": list(dims), "sites": V, "l2": "inputs (9.7 GB links) >> 126 MB L2, no flush needed",
                   "parallelism": "replicas only (no data-path collective)" if world > 1 else "single GPU",
                   "bytes_per_even_site_per_step": REALS_ITER_NOMINAL * rsize},
        "clocks": clocks.summary(), "e2e": e2e, "gpu_launches": int(launches),
        "roofline": roofline, "kernel_ms": kernel_ms, "setup_seconds": round(t_setup, 1),
    }

    if rank == 0 and not args.quick and prec == 64:
        extras(args, q, torch, ctx, out, cfg, dims, U, b, fU, fb, fx, fo, peak)
    if rank == 0:
        print(json.dumps(out), flush=True)
    ctx.close()
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def extras(args, q, torch, ctx, out, cfg, dims, U, b, fU, fb, fx, fo, peak):
    """Reports beside the headline (rank 0, N = 1 semantics): Dslash alone, full solves, fp32, oracle."""
    import oracle
    V = int(np.prod(dims))
    Vh = V // 2
    m = cfg["m"]
    # Dslash alone, fp64
    out["dslash_fp64"] = dslash_report(time_dslash(q, torch, ctx, fU, fb, fo), Vh, 8, peak)
    # full fp64 solve: CG s/solve (BASELINE.json metric)
    info = ctx.qcd_cg_solve(fU, fb, fx, m, cfg["tol64"], cfg["maxiter"])
    x64 = fx.download()
    t0 = time.time()
    true64 = oracle.true_residual(dims, U, b, x64, m)
    t_true = time.time() - t0
    out["cg_fp64"] = {"tol": cfg["tol64"], "iters": info["iters"], "converged": info["converged"],
                      "s_per_solve": round(info["seconds"], 4),
                      "ms_per_iter": round(1e3 * info["seconds"] / max(info["iters"], 1), 5),
                      "rel_resid_recurrence": info["rel_resid"], "true_resid_oracle_fp64": true64}
    # CPU baseline: the oracle as it stands, a bounded sample of the same workload
    nit = 12                                                # ~10 s of oracle time at 64^4 on 16 cores
    t0 = time.time()
    _, oinfo = oracle.cg(dims, U, b, m, 1e-300, nit)
    t_or = time.time() - t0
    out["cpu_baseline"] = {"value": round(REALS_ITER_NOMINAL * 8 * Vh * oinfo["iters"] / t_or / 1e9, 3), "unit": UNIT,
                           "cores": oracle.num_threads(), "kind": "oracle",
                           "sample": f"{nit} CG iterations (maxiter={nit}) of the same {'x'.join(map(str, dims))} fp64 solve, "
                                     f"including the oracle's own set-up; {t_or:.1f} s",
                           "oracle_apply_M_seconds": round(t_true, 2)}
    del x64
    # ---- variants, reported separately from the headline ----
    c32 = q.Context(dims, 32, device=ctx.device)
    gU = c32.field(q.QCD_GAUGE)
    ctx.qcd_field_convert(gU, fU)                          # fp32 links = round-to-nearest of the fp64 links, on the device
    gx = c32.field(q.QCD_SPINOR_EVEN)
    go = c32.field(q.QCD_SPINOR_ODD)
    # mixed-precision defect-correction CG to the fp64 tolerance (R21)
    inner_tol = 1e-3
    mi = ctx.qcd_cg_solve_mixed(c32, fU, gU, fb, fx, gx, c32.field(q.QCD_SPINOR_EVEN), m, cfg["tol64"], inner_tol,
                                4 * cfg["maxiter"])
    xm = fx.download()
    out["cg_mixed"] = {"tol": cfg["tol64"], "inner_tol": inner_tol, "converged": mi["converged"], "outer": mi["outer"],
                       "inner_iters_fp32": mi["inner_iters"], "m_applications_fp64": mi["m_applications_fp64"],
                       "s_per_solve": round(mi["seconds"], 4), "true_resid_device_fp64": mi["true_resid"],
                       "true_resid_oracle_fp64": oracle.true_residual(dims, U, b, xm, m),
                       "speedup_vs_cg_fp64": round(out["cg_fp64"]["s_per_solve"] / max(mi["seconds"], 1e-9), 3)}
    del xm
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
    xc = fx.download()
    out["cg_fp64_tworow_temporal_gauge"] = {
        "tol": cfg["tol64"], "iters": info["iters"], "converged": info["converged"], "s_per_solve": round(info["seconds"], 4),
        "ms_per_iter": round(1e3 * info["seconds"] / max(info["iters"], 1), 5),
        "true_resid_oracle_fp64_original_links": oracle.true_residual(dims, U, b, xc, m),
        "speedup_vs_cg_fp64": round(out["cg_fp64"]["s_per_solve"] / max(info["seconds"], 1e-9), 3)}
    mi = ctx.qcd_cg_solve_mixed(c32, f12, g12, fbr, fx, gx, c32.field(q.QCD_SPINOR_EVEN), m, cfg["tol64"], inner_tol,
                                4 * cfg["maxiter"])
    ctx.qcd_spinor_rotate(fg, fx, fx, dagger=True)
    xc = fx.download()
    out["cg_mixed_tworow_temporal_gauge"] = {
        "tol": cfg["tol64"], "inner_tol": inner_tol, "converged": mi["converged"], "outer": mi["outer"],
        "inner_iters_fp32": mi["inner_iters"], "s_per_solve": round(mi["seconds"], 4),
        "true_resid_device_fp64": mi["true_resid"],
        "true_resid_oracle_fp64_original_links": oracle.true_residual(dims, U, b, xc, m),
        "speedup_vs_cg_fp64": round(out["cg_fp64"]["s_per_solve"] / max(mi["seconds"], 1e-9), 3)}
    del xc
    for f in (f12, g12, fg, fbr):
        f.free()
    out["variants_fp64"] = {"lattice": list(dims), "dslash": variants_sweep(q, torch, ctx, fU, dims, peak)}
    out["cg_multi_fp64"] = cg_multi_report(q, torch, ctx.device, dims, 64, fU, m)
    # fp32: free the fp64 device fields first
    fU.free(); fb.free(); fx.free(); fo.free()
    ctx.close()
    torch.cuda.empty_cache()
    U32, b32 = U.astype(np.complex64), b.astype(np.complex64)
    gb = c32.field(q.QCD_SPINOR_EVEN).upload(b32)
    out["dslash_fp32"] = dslash_report(time_dslash(q, torch, c32, gU, gb, go), Vh, 4, peak)
    out["variants_fp32"] = {"lattice": list(dims), "dslash": variants_sweep(q, torch, c32, gU, dims, peak)}
    if cfg["tol32"]:
        info = c32.qcd_cg_solve(gU, gb, gx, m, cfg["tol32"], cfg["maxiter"])
        x32 = gx.download()
        out["cg_fp32"] = {"tol": cfg["tol32"], "iters": info["iters"], "converged": info["converged"],
                          "s_per_solve": round(info["seconds"], 4),
                          "ms_per_iter": round(1e3 * info["seconds"] / max(info["iters"], 1), 5),
                          "rel_resid_recurrence": info["rel_resid"],
                          "true_resid_oracle_fp64": oracle.true_residual(dims, U32, b32, x32, m),
                          "note": "plain fp32 CG on Haar links stalls in TRUE residual near 1e-4 (DESIGN.md R11)"}
    c32.close()
    torch.cuda.empty_cache()
    # the paper's own NMULTI experiment: 32^4, two-row links, temporal gauge (Table 2)
    if dims == (64, 64, 64, 64):
        d32 = (32, 32, 32, 32)
        _, U_32, _ = make_inputs(d32, 2)
        t2 = {"lattice": list(d32), "paper_A100_tflops": {"fp32": {1: 2.244, 2: 2.532, 3: 2.953, 4: 3.205, 6: 3.090, 8: 3.006},
                                                           "fp64": {1: 1.245, 2: 1.530, 3: 1.929, 4: 2.199, 6: 2.039, 8: 2.026},
                                                           "source": "PAPER.md:84-98 Table 2 (A100, OpenCL; other hardware, context only)"}}
        for prec in (64, 32):
            c = q.Context(d32, prec, device=ctx.device)
            f = c.field(q.QCD_GAUGE).upload(U_32)
            t2[f"fp{prec}"] = variants_sweep(q, torch, c, f, d32, peak)
            f.free(); c.close()
        out["variants_table2_32x32x32x32"] = t2
        out["cg_small_lattice"] = small_lattice_report(q, torch, ctx.device)
        out["cg_update_routine_48x48x48x48"] = update_routine_report(q, torch, ctx.device, peak)
        out["size_sweep_fig3"] = size_sweep_report(q, torch, ctx.device)
    out["paper_context"] = {"A100_OpenCL_dslash_fp64_TFLOPs_32^4_12real_links_gaugefixed": 1.245,
                            "A100_OpenCL_cg_update_GBs_48^4_fp64": 1351, "source": "PAPER.md:59,87 (other hardware; context only)"}


# ---- reference arm: the CPU oracle -------------------------------------------------------------
def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    import oracle
    K, W = args.steps, args.warmup
    dims = tuple(int(v) for v in args.lattice.split(",")) if args.lattice else (32, 32, 32, 32)
    cfg, U, b = make_inputs(dims)
    Vh = int(np.prod(dims)) // 2
    if W > 0:
        oracle.cg(dims, U, b, cfg["m"], 1e-300, W)
    t0 = time.perf_counter()
    _, info = oracle.cg(dims, U, b, cfg["m"], 1e-300, K)
    dt = time.perf_counter() - t0
    value = REALS_ITER_NOMINAL * 8 * Vh * info["iters"] / dt / 1e9
    sample = (f"{K} CG iterations of the CPU oracle on a {'x'.join(map(str, dims))} lattice of the same recipe "
              f"(Haar links, m={cfg['m']}, fp64): a 1/{(64 ** 4) // int(np.prod(dims))} sample of the 64^4 sites; GB/s is per-site intensive")
    out = {"impl": "reference", "metric": METRIC, "value": round(value, 4), "unit": UNIT, "n_gpus": world, "steps": K,
           "warmup": W, "ms_per_step": round(1e3 * dt / max(info["iters"], 1), 3), "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded)",
           "config": {"workload": "64x64x64x64 staggered CG iteration, Haar links, m=0.01, fp64, full 18-real links",
                      "sample": sample},
           "cpu_baseline": {"value": round(value, 4), "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
           "e2e": {"value": round(value, 4), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def run_variants_only(args):
    """Dslash variant sweep alone (rank 0, one GPU): `--lattice`, `--prec`, `--nmulti`, `--reps`."""
    import torch
    import paper_2502_03249_b200 as q
    dims = tuple(int(v) for v in args.lattice.split(",")) if args.lattice else (64, 64, 64, 64)
    peak, _ = load_peaks()
    _, U, _ = make_inputs(dims)
    ctx = q.Context(dims, args.prec)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    ctx.qcd_set_dslash_variant(args.kernel)
    rows = variants_sweep(q, torch, ctx, fU, dims, peak, tuple(int(v) for v in args.nmulti.split(",")), args.reps)
    print(json.dumps({"variants": rows, "lattice": list(dims), "prec": args.prec, "gpu_launches": ctx.qcd_launch_count()}), flush=True)
    ctx.close()


def main():
    args = parse_args()
    if args.variants_only:
        run_variants_only(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

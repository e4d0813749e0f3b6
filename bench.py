#!/usr/bin/env python
"""bench.py -- staggered Dslash + CG hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--lattice 64,64,64,64] [--quick]

stdout carries exactly ONE line: a compact (< 2 KB) JSON headline, printed last by rank 0.  Everything
else the run measures (per-config table, full solves, variants, sweeps) goes to a sidecar JSON file whose
path is in the headline (`extras`, default gpurun_out/bench_extras.json); progress goes to stderr.

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
          The gauge links are the operator, resident like model weights: their upload is outside.
  roofline : the Dslash kernel (D_oe launches inside the timed region, CUDA events on the
          launching stream), algorithmic = COMPULSORY DRAM bytes 1248 B/site (each link once,
          each spinor once, one store), against MEASURED_PEAKS.json hbm_gbs.
  cpu_baseline / --impl reference : the CPU oracle as it stands on the host cores.

N > 1: replicas only: every rank runs the same workload on its own
GPU, no data-path collective; value = sum of units / max-over-ranks device time.  `--gpus N`
without a torchrun environment re-launches itself under torch.distributed.run with N ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
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
FLOP_PER_CG_ITER = 2 * FLOP_PER_SITE + 72     # per even site: two half-Dslash + m^2 p - (6 fma) + two dots (2 x 12) + x, r, p updates (3 x 12)

UNIT = "GB/s"
HEADLINE_MAX_BYTES = 2000                # the driver keeps a tail of stdout: the line must survive it whole
DEFAULT_EXTRAS = os.path.join("gpurun_out", "bench_extras.json")


def lattice_name(dims) -> str:
    d = tuple(dims)
    return f"{d[0]}^4" if len(set(d)) == 1 else "x".join(map(str, d))


def metric_name(dims, prec: int = 64) -> str:
    return (f"staggered CG-iteration effective GB/s (two half-Dslash at {198 * prec // 8} B/site + CG vector kernels), "
            f"{lattice_name(dims)} fp{prec}")


def workload_name(dims, m, prec: int = 64) -> str:
    return f"{'x'.join(map(str, dims))} staggered CG iteration, Haar links, m={m}, fp{prec}, full 18-real links"


def log(msg: str) -> None:
    print(f"[bench {time.strftime('%H:%M:%S')}] {msg}", file=sys.stderr, flush=True)


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--lattice", default=None, help="override dims, e.g. 16,16,16,16 (testing only)")
    ap.add_argument("--quick", action="store_true", help="headline only: no sidecar reports, no full solves, no cpu_baseline")
    ap.add_argument("--extras", default=None, help=f"path of the sidecar JSON (default {DEFAULT_EXTRAS})")
    ap.add_argument("--variants-only", action="store_true",
                    help="run only the Dslash variant sweep (two-row / temporal gauge / NMULTI) and print it; used for ncu captures")
    ap.add_argument("--dslash-only", action="store_true",
                    help="run only `--reps` D_oe and D_eo launches of BASELINE.json configs[--config] in --prec; used for ncu captures")
    ap.add_argument("--cg-only", action="store_true",
                    help="run only `--reps` full CG solves of BASELINE.json configs[--config] in --prec with the solver loop the "
                         "library picks; used for ncu captures of the small-lattice loops")
    ap.add_argument("--cg-multi-only", action="store_true",
                    help="run only `--reps` lock-step CG iterations over the first value of --nmulti right-hand sides at 64^4 (or --lattice), on "
                         "full links and on two-row temporal-gauge links; used for ncu captures of the reducing multi-vector kernels")
    ap.add_argument("--config", type=int, default=4, choices=(0, 1, 2, 3, 4), help="BASELINE.json config of --dslash-only / --cg-only")
    ap.add_argument("--prec", type=int, default=64, choices=(64, 32),
                    help="precision of --variants-only / --dslash-only, and of the timed CG iterations (32: the fp32 path of "
                         "the same workload, reported with dtype f32 and without the extra reports; the default line is fp64)")
    ap.add_argument("--nmulti", default="1,2,3,4,6,8", help="NMULTI values of --variants-only")
    ap.add_argument("--reps", type=int, default=10, help="timed launches per variant of --variants-only / --dslash-only")
    ap.add_argument("--kernel", type=int, default=0,
                    help="qcd_set_dslash_variant (A/B runs; 0 the library's choice, 1-3 block shapes of the one-vector kernel, 4 staged, "
                         "5 register, 6/7 pair, 8 tile, 9 rolled, 10 bulk-copy kernel)")
    ap.add_argument("--stream-bulk", action="store_true",
                    help="run only the qcd_stream_bulk sweep (requested bytes per second through the TMA copy engine, 64^4 gauge field) and print it")
    return ap.parse_args(argv)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (torch copy)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_traffic(prec: int):
    """ncu-measured DRAM bytes of one D_oe launch at 64^4 and where they come from: profiles/dslash_traffic.csv
    (text, committed; a constant from the capture named there, NOT a measurement of this run).  (None, None) if absent."""
    p = os.path.join(ROOT, "profiles", "dslash_traffic.csv")
    if not os.path.exists(p):
        return None, None
    with open(p) as f:
        rows = dict(line.strip().split(",", 1) for line in f if "," in line and not line.startswith("#"))
    v = rows.get(f"fp{prec}_64x64x64x64_bytes_per_launch")
    src = "profiles/dslash_traffic.csv (ncu --set full capture" + (f" at {rows['captured_at_commit']}" if "captured_at_commit" in rows else "") + ")"
    return (int(v), src) if v is not None else (None, None)


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


def free_port() -> int:
    with socket.socket(socket.AF_INET, socket.SOCK_STREAM) as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def respawn_under_torchrun(args, argv) -> int | None:
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: launch N ranks (one per GPU) of this very
    command under torch.distributed.run and return its exit code; None when no re-launch is needed."""
    if args.gpus <= 1 or "WORLD_SIZE" in os.environ or args.variants_only or args.dslash_only or args.cg_only or args.cg_multi_only or args.stream_bulk:
        return None
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + list(argv)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    log(f"--gpus {args.gpus} without a torchrun environment: launching {args.gpus} ranks")
    return subprocess.call(cmd, env=env, cwd=ROOT)


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


# ---- the one stdout line ---------------------------------------------------------------------
HEADLINE_KEYS = ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                 "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline",
                 "dslash_gbs_fp64", "dslash_frac_hbm_fp64", "dslash_gbs_fp32", "cg_s_per_solve_fp64", "cg_s_per_solve_fp32",
                 "cg_iters_fp64", "extras")
# dropped, in this order, if a line ever exceeds HEADLINE_MAX_BYTES (never the contract keys)
HEADLINE_OPTIONAL = ("cg_iters_fp64", "data", "dslash_frac_hbm_fp64", "cg_s_per_solve_fp32", "dslash_gbs_fp32")


def headline_line(out: dict) -> str:
    """The compact JSON line: the bench contract's keys, the four numbers BASELINE.json's metric names and the
    path of the sidecar.  Anything else in `out` stays in the sidecar."""
    d = {k: out[k] for k in HEADLINE_KEYS if k in out}
    line = json.dumps(d, separators=(",", ":"))
    for k in HEADLINE_OPTIONAL:
        if len(line) <= HEADLINE_MAX_BYTES:
            break
        d.pop(k, None)
        line = json.dumps(d, separators=(",", ":"))
    if len(line) > HEADLINE_MAX_BYTES:
        raise RuntimeError(f"headline JSON is {len(line)} bytes (> {HEADLINE_MAX_BYTES}): trim a contract key's text")
    return line


def write_sidecar(path: str, data: dict) -> str | None:
    try:
        full = path if os.path.isabs(path) else os.path.join(ROOT, path)
        os.makedirs(os.path.dirname(full), exist_ok=True)
        tmp = full + f".tmp{os.getpid()}"
        with open(tmp, "w") as f:
            json.dump(data, f, indent=1)
        os.replace(tmp, full)
        return path
    except OSError as e:  # a read-only checkout must not cost the headline
        log(f"sidecar not written: {e!r}")
        return None


# ---- our arm ---------------------------------------------------------------------------------
def make_inputs(dims, cfg_index=4):
    import qcd_inputs
    cfg = dict(qcd_inputs.CONFIGS[cfg_index])
    cfg["dims"] = tuple(dims)
    U = qcd_inputs.gauge_field(cfg["dims"], cfg["links"], seed=0, eps=cfg["eps"])
    b = qcd_inputs.gaussian_source(cfg["dims"], seed=1, parity=0)
    return cfg, U, b


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
    ctx.qcd_set_dslash_variant(args.kernel)                # 0 unless an A/B run asks for another block shape
    fU = ctx.field(q.QCD_GAUGE)
    fb = ctx.field(q.QCD_SPINOR_EVEN)
    fx = ctx.field(q.QCD_SPINOR_EVEN)
    fo = ctx.field(q.QCD_SPINOR_ODD)
    if rank == 0:
        log(f"generating {lattice_name(dims)} inputs")
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
    m = cfg["m"]
    t_setup = time.time() - t_setup

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()

    # ---------------- timed region: K CG iterations, inputs resident --------------------------
    log(f"timed region: {W} + {K} CG iterations")
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
    for _ in range(K):
        ctx.qcd_cg_iterate(1)
        ctx.qcd_cg_poll()                                  # D2H read of the step's result (residual)
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
           "what": "upload(b, pinned) + K x [qcd_cg_iterate(1) + qcd_cg_poll D2H] + download(x); source/solution copies "
                   "amortised over K; the 9.7 GB link upload (the operator, resident) is outside"}

    # ---------------- roofline of the dominant kernel ------------------------------------------
    n_ds, ms_ds = prof[q.QCD_K_DSLASH]
    ds_ms = ms_ds / max(n_ds, 1)
    achieved = REALS_DSLASH_COMPULSORY * rsize * Vh / ds_ms / 1e6
    # read-only streaming ceiling over the gauge field's own bytes (qcd_stream_read: the Dslash's link-load
    # instruction and nothing else), measured after the timed region; the third denominator beside the
    # copy peak and the theoretical peak
    ctx.qcd_stream_read(fU, 3)
    stream_gbs = fU.nbytes / ctx.qcd_stream_read(fU, 10) / 1e6
    traffic, traffic_src = load_traffic(prec) if dims == (64, 64, 64, 64) else (None, None)
    roofline = {"bound": "hbm", "kernel": f"dslash_kernel<{'double' if prec == 64 else 'float'},MODE0> (D_oe inside the CG iteration)",
                "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s", "frac": round(achieved / peak, 4),
                "peak_source": peak_src, "traffic": traffic, "traffic_source": traffic_src,
                "algorithmic_bytes_per_launch": REALS_DSLASH_COMPULSORY * rsize * Vh,
                "avg_launch_ms": round(ds_ms, 5), "launches_timed": n_ds,
                "frac_of_theoretical_8184": round(achieved / THEORETICAL_HBM_GBS, 4),
                "read_stream_gbs": round(stream_gbs, 1), "frac_of_read_stream": round(achieved / stream_gbs, 4)}
    kernel_ms = {name: round(prof[k][1] / max(prof[k][0], 1), 5) for name, k in
                 (("dslash_oe", q.QCD_K_DSLASH), ("dslash_eo_epilogue_dot", q.QCD_K_DSLASH_EPI),
                  ("update_xr_norm", q.QCD_K_UPDATE_XR), ("update_p", q.QCD_K_UPDATE_P))}

    out = {
        "metric": metric_name(dims, prec),
        "value": round(value, 2), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": round(ms_max / K, 5), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": f"f{prec}", "data": "synthetic: seeded Haar SU(3) links, Gaussian source (BASELINE.json configs[4])",
        "config": {"workload": workload_name(dims, m, prec),
                   "l2": "inputs (9.7 GB links) >> 126 MB L2, no flush needed" if V >= 1 << 22 else "small lattice: L2-resident",
                   "parallelism": "replicas only (no data-path collective)" if world > 1 else "single GPU"},
        "clocks": clocks.summary(), "e2e": e2e, "gpu_launches": int(launches),
        "roofline": roofline,
    }
    side = dict(out)
    side.update({"kernel_ms": kernel_ms, "setup_seconds": round(t_setup, 1), "lattice": list(dims), "sites": V,
                 "bytes_per_even_site_per_step": REALS_ITER_NOMINAL * rsize})

    ran_reports = rank == 0 and not args.quick and prec == 64
    if ran_reports:
        import bench_reports
        bench_reports.run_all(args, q, torch, ctx, out, side, cfg, dims, U, b, hb, hx, fU, fb, fx, fo, peak, stream_gbs)
    del hb, hx
    if rank == 0:
        if ran_reports or args.extras:                    # --quick has nothing beyond the headline and must not overwrite a sidecar
            path = write_sidecar(args.extras or DEFAULT_EXTRAS, side)
            if path:
                out["extras"] = path
        print(headline_line(out), flush=True)
    try:
        ctx.close()
    except Exception:
        pass
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


# ---- reference arm: the CPU oracle -------------------------------------------------------------
def run_reference(args):
    """The oracle as it stands, on the host cores, on OUR arm's workload (64^4 unless --lattice says otherwise):
    W untimed + K timed CG iterations of the same solve (a bounded sample of it: iterations, not sites)."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    import oracle
    K, W = args.steps, args.warmup
    dims = tuple(int(v) for v in args.lattice.split(",")) if args.lattice else (64, 64, 64, 64)
    log(f"reference arm: generating {lattice_name(dims)} inputs")
    cfg, U, b = make_inputs(dims)
    Vh = int(np.prod(dims)) // 2
    if W > 0:
        oracle.cg(dims, U, b, cfg["m"], 1e-300, W)
    t0 = time.perf_counter()
    _, info = oracle.cg(dims, U, b, cfg["m"], 1e-300, K)
    dt = time.perf_counter() - t0
    value = REALS_ITER_NOMINAL * 8 * Vh * info["iters"] / dt / 1e9
    sample = (f"{K} CG iterations (after {W} untimed) of the CPU oracle on the same {'x'.join(map(str, dims))} solve, "
              f"oracle set-up included; {dt:.1f} s")
    out = {"impl": "reference", "metric": metric_name(dims), "value": round(value, 4), "unit": UNIT,
           "n_gpus": max(world, args.gpus), "steps": K,
           "warmup": W, "ms_per_step": round(1e3 * dt / max(info["iters"], 1), 3), "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded)",
           "config": {"workload": workload_name(dims, cfg["m"]), "sample": sample},
           "cpu_baseline": {"value": round(value, 4), "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
           "e2e": {"value": round(value, 4), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(headline_line(out), flush=True)


def run_variants_only(args):
    """Dslash variant sweep alone (rank 0, one GPU): `--lattice`, `--prec`, `--nmulti`, `--reps`."""
    import torch
    import bench_reports
    import paper_2502_03249_b200 as q
    dims = tuple(int(v) for v in args.lattice.split(",")) if args.lattice else (64, 64, 64, 64)
    peak, _ = load_peaks()
    _, U, _ = make_inputs(dims)
    ctx = q.Context(dims, args.prec)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    ctx.qcd_set_dslash_variant(args.kernel)
    rows = bench_reports.variants_sweep(q, torch, ctx, fU, dims, peak, tuple(int(v) for v in args.nmulti.split(",")), args.reps)
    print(json.dumps({"variants": rows, "lattice": list(dims), "prec": args.prec, "gpu_launches": ctx.qcd_launch_count()}), flush=True)
    ctx.close()


def run_dslash_only(args):
    """`--reps` launches each of D_oe and D_eo (and one qcd_apply_M) at BASELINE.json configs[--config]: the command the
    per-config ncu captures under profiles/ are taken with."""
    import torch
    import qcd_inputs
    import paper_2502_03249_b200 as q
    cfg, U, b = qcd_inputs.config_inputs(args.config)
    if args.lattice:
        cfg, U, b = qcd_inputs.config_inputs(args.config, tuple(int(v) for v in args.lattice.split(",")))
    dims = cfg["dims"]
    ctx = q.Context(dims, args.prec)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    fb = ctx.field(q.QCD_SPINOR_EVEN).upload(b)
    fo, fe = ctx.field(q.QCD_SPINOR_ODD), ctx.field(q.QCD_SPINOR_EVEN)
    ctx.qcd_set_dslash_variant(args.kernel)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ctx.qcd_dslash_oe(fU, fo, fb)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.reps):
        ctx.qcd_dslash_oe(fU, fo, fb)
        ctx.qcd_dslash_eo(fU, fe, fo)
    e1.record()
    torch.cuda.synchronize()
    ctx.qcd_apply_M(fU, fe, fb, cfg["m"])
    torch.cuda.synchronize()
    print(json.dumps({"dslash_only": True, "config": args.config, "lattice": list(dims), "prec": args.prec,
                      "ms_per_half_dslash": round(e0.elapsed_time(e1) / (2 * args.reps), 5),
                      "gpu_launches": ctx.qcd_launch_count()}), flush=True)
    ctx.close()


def run_cg_only(args):
    """`--reps` full solves at BASELINE.json configs[--config] (tolerance of that config and precision): the command the
    captures of the solver-loop kernels under profiles/ are taken with."""
    import torch
    import qcd_inputs
    import paper_2502_03249_b200 as q
    cfg, U, b = qcd_inputs.config_inputs(args.config)
    dims = cfg["dims"]
    tol = cfg["tol64"] if args.prec == 64 else (cfg["tol32"] or 1e-5)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ctx = q.Context(dims, args.prec, stream=stream)
        fU = ctx.field(q.QCD_GAUGE).upload(U)
        fb, fx = ctx.field(q.QCD_SPINOR_EVEN).upload(b), ctx.field(q.QCD_SPINOR_EVEN)
        infos = [ctx.qcd_cg_solve(fU, fb, fx, cfg["m"], tol, cfg["maxiter"]) for _ in range(max(args.reps, 1))]
        best = min(infos, key=lambda i: i["seconds"])
        print(json.dumps({"cg_only": True, "config": args.config, "lattice": list(dims), "prec": args.prec, "tol": tol,
                          "loop": ctx.qcd_last_cg_loop(), "cluster_ctas": ctx.qcd_last_cg_cluster(), "iters": best["iters"],
                          "converged": best["converged"], "s_per_solve": best["seconds"],
                          "us_per_iter": round(1e6 * best["seconds"] / max(best["iters"], 1), 3),
                          "gpu_launches": ctx.qcd_launch_count()}), flush=True)
        ctx.close()


def run_cg_multi_only(args):
    """Lock-step CG iterations alone (bench_reports.cg_multi_report for one n): the command the captures of the multi-vector
    reducing kernels under profiles/ are taken with."""
    import torch
    import bench_reports
    import paper_2502_03249_b200 as q
    dims = tuple(int(v) for v in args.lattice.split(",")) if args.lattice else (64, 64, 64, 64)
    cfg, U, _ = make_inputs(dims)
    n = int(args.nmulti.split(",")[0])
    ctx = q.Context(dims, args.prec)
    fU = ctx.field(q.QCD_GAUGE).upload(U)
    rows = bench_reports.cg_multi_report(q, torch, ctx.device, dims, args.prec, fU, cfg["m"], ns=(n,), iters=max(args.reps, 1))
    print(json.dumps({"cg_multi_only": True, "lattice": list(dims), "prec": args.prec, "rows": rows}), flush=True)
    ctx.close()


def run_stream_bulk(args):
    """qcd_stream_bulk sweep alone (rank 0, one GPU): the rate at which the SMs take in requested bytes through the TMA copy engine, for
    the box shapes and ring depths of the multi-vector Dslash, beside the LSU read stream over the same field."""
    import torch
    import paper_2502_03249_b200 as q
    dims = tuple(int(v) for v in args.lattice.split(",")) if args.lattice else (64, 64, 64, 64)
    ctx = q.Context(dims, 64, workspace=False)
    fU = ctx.field(q.QCD_GAUGE)
    fU.buf.view(torch.float64).normal_()
    groups = int(np.prod(dims)) // 2 // 128
    rows_out = []
    ctx.qcd_stream_read(fU, 2)
    lsu = fU.nbytes / ctx.qcd_stream_read(fU, args.reps) / 1e6
    # (rows per copy, copies per stage, stages, producer warps): one link box = 9 rows; a vector box = 3 rows
    for rows, copies, stages, producers in ((9, 1, 4, 1), (9, 3, 3, 3), (3, 3, 4, 1), (3, 7, 4, 1), (3, 7, 4, 4), (21, 1, 4, 1), (3, 11, 3, 1), (3, 11, 3, 2),
                                            (3, 11, 3, 4), (11, 3, 3, 1), (11, 3, 3, 3), (33, 1, 3, 1), (1, 33, 3, 4), (1, 9, 8, 4)):
        ctx.qcd_stream_bulk(fU, rows, copies, 8, stages, producers, 1)
        ms = ctx.qcd_stream_bulk(fU, rows, copies, 8, stages, producers, args.reps)
        req = groups * 8 * copies * rows * 2048
        hbm = groups * min(72, 8 * copies * rows) * 2048
        rows_out.append({"rows_per_copy": rows, "copies_per_stage": copies, "stage_kb": rows * copies * 2, "stages": stages, "producer_warps": producers,
                         "ms": round(ms, 4), "requested_tbs": round(req / ms / 1e9, 2), "of_which_hbm_tbs": round(hbm / ms / 1e9, 2),
                         "us_per_stage_and_sm": round(ms * 1e3 / (groups * 8 / 148), 3)})
    print(json.dumps({"stream_bulk": rows_out, "lsu_read_stream_gbs": round(lsu, 1), "lattice": list(dims), "gpu_launches": ctx.qcd_launch_count()}), flush=True)
    ctx.close()


def main(argv=None):
    argv = sys.argv[1:] if argv is None else argv
    args = parse_args(argv)
    rc = respawn_under_torchrun(args, argv)
    if rc is not None:
        sys.exit(rc)
    if args.variants_only:
        run_variants_only(args)
    elif args.dslash_only:
        run_dslash_only(args)
    elif args.cg_only:
        run_cg_only(args)
    elif args.cg_multi_only:
        run_cg_multi_only(args)
    elif args.stream_bulk:
        run_stream_bulk(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

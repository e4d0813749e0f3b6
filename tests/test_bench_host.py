"""CPU-side checks of bench.py's host logic: the byte model, the only multi-rank communication
(MAX time / SUM units over ranks, gloo, world_size 2), and the reference arm under torchrun
semantics (rank 0 prints one JSON line, other ranks exit 0 silently)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_byte_and_flop_model():
    import bench
    assert bench.FLOP_PER_SITE == 8 * 66 + 7 * 6 == 570
    assert bench.REALS_DSLASH_NOMINAL * 8 == 1584 and bench.REALS_DSLASH_NOMINAL * 4 == 792   # north_star
    assert bench.REALS_DSLASH_COMPULSORY * 8 == 1248
    assert bench.REALS_ITER_COMPULSORY * 8 == 2976 and bench.REALS_ITER_NOMINAL * 8 == 3648
    # the paper's own model: 6 links x 12 + 9 vectors x 6 = 126 reals -> AI 0.57 / 1.13
    assert abs(570 / (126 * 8) - 0.57) < 0.01 and abs(570 / (126 * 4) - 1.13) < 0.01


def test_variant_byte_model_matches_the_papers_formula():
    """two rows + temporal gauge, n vectors: AI(n) = n 570 / (8 (6 12 + n 9 6)) in fp64."""
    import bench
    import bench_reports
    for n in (1, 2, 3, 4, 6, 8, 16):
        comp, nom = bench_reports.variant_reals(2, 1, n, 10 ** 9)           # N3 -> infinity: exactly 6 links per site
        assert abs(nom - (6 * 12 + n * 9 * 6)) < 1e-6
        assert abs(570 * n / (nom * 8) - n * 570 / (8 * (6 * 12 + n * 9 * 6))) < 1e-8
        assert abs(comp - (72 + 12 * n)) < 1e-6
    assert bench_reports.variant_reals(2, 1, 1, 10 ** 9)[1] == pytest.approx(126)            # "a total float count of 126 per site"
    assert bench_reports.variant_reals(3, 0, 1, 64) == (bench.REALS_DSLASH_COMPULSORY, bench.REALS_DSLASH_NOMINAL)
    assert bench_reports.variant_reals(2, 0, 1, 64) == (108, 150)
    # the slices x3 = 0 / 1 still read their time links: 2 / N3 links per site on average
    assert bench_reports.variant_reals(2, 1, 1, 64)[0] == pytest.approx((6 + 2 / 64) * 12 + 12)


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank = dist.get_rank()
ms, units = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 100.0 * (rank + 1))
assert ms == 15.0 and units == 300.0, (ms, units)
dist.barrier()
dist.destroy_process_group()
sys.stdout.write("rank %d ok\n" % rank)      # ONE write per rank: the two ranks share the pipe
"""


def _torchrun(args, timeout=300):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(29500 + os.getpid() % 400)] + args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, env=env, cwd=ROOT)


def test_aggregate_over_ranks_gloo_world2(tmp_path):
    script = tmp_path / "agg_worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    r = _torchrun([str(script)])
    assert r.returncode == 0, r.stderr[-2000:]
    assert "rank 0 ok" in r.stdout and "rank 1 ok" in r.stdout


def test_reference_arm_world2_prints_one_line():
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2",
                   "--warmup", "1", "--lattice", "8,8,8,8"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1 and len(lines[0]) < 4096
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["steps"] == 2 and d["value"] > 0 and d["n_gpus"] == 2
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["unit"] == "GB/s" and d["higher_is_better"] is True


def test_reference_arm_spawns_its_own_ranks_and_labels_its_lattice():
    """`python bench.py --gpus 2` WITHOUT torchrun (the form the driver uses at N = 1) must launch the ranks itself:
    one JSON line, n_gpus 2; the workload label is the lattice that was actually timed."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_PORT")}
    env["OMP_NUM_THREADS"] = "2"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2",
                        "--warmup", "1", "--lattice", "8,8,8,8"], capture_output=True, text=True, cwd=ROOT, timeout=300, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1 and lines[0].startswith("{"), r.stdout
    assert len(lines[0]) < 4096
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["config"]["workload"].startswith("8x8x8x8 ") and "8^4" in d["metric"] and "64x64" not in d["config"]["workload"]
    assert "8x8x8x8" in d["cpu_baseline"]["sample"]


def test_headline_line_is_compact_and_complete():
    """BENCH_r01 was unparseable because the one stdout line carried 27 KB of sweeps.  The headline must stay far
    below the driver's tail window whatever the sidecar holds, and keep every contract key."""
    import bench
    out = {
        "metric": bench.metric_name((64, 64, 64, 64)), "value": 8459.87, "unit": "GB/s", "n_gpus": 1, "steps": 200, "warmup": 5,
        "ms_per_step": 3.61727, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic: seeded Haar SU(3) links, Gaussian source (BASELINE.json configs[4])",
        "config": {"workload": bench.workload_name((64, 64, 64, 64), 0.01), "l2": "inputs (9.7 GB links) >> 126 MB L2, no flush needed",
                   "parallelism": "replicas only (no data-path collective)"},
        "clocks": {"sm_mhz": 1567.0, "sm_max_mhz": 1965, "reasons": ["hw_power_brake", "sw_power_cap", "sw_thermal_slowdown"],
                   "samples": 72, "power_w": 561.3},
        "e2e": {"value": 8101.72, "unit": "GB/s", "h2d_bytes_per_step": 4026531, "d2h_bytes_per_step": 4026603, "ms_total": 755.436,
                "what": "upload(b, pinned) + K x [qcd_cg_iterate(1) + qcd_cg_poll D2H] + download(x); source/solution copies "
                        "amortised over K; the 9.7 GB link upload (the operator, resident) is outside"},
        "gpu_launches": 800,
        "roofline": {"bound": "hbm", "kernel": "dslash_kernel<double,MODE0> (D_oe inside the CG iteration)", "achieved": 7007.6,
                     "peak": 6532.5, "unit": "GB/s", "frac": 1.0727, "peak_source": "MEASURED_PEAKS.json hbm_gbs (torch copy)",
                     "traffic": 10462276352, "traffic_source": "profiles/dslash_traffic.csv (ncu --set full capture at 0123456789ab)",
                     "algorithmic_bytes_per_launch": 10468982784, "avg_launch_ms": 1.49395, "launches_timed": 200,
                     "frac_of_theoretical_8184": 0.8563, "read_stream_gbs": 7310.1, "frac_of_read_stream": 0.9586},
        "cpu_baseline": {"value": 58.822, "unit": "GB/s", "cores": 16, "kind": "oracle",
                         "sample": "12 CG iterations of the same 64x64x64x64 fp64 solve, oracle set-up included; 6.2 s"},
        "dslash_gbs_fp64": 7056.2, "dslash_frac_hbm_fp64": 1.0802, "dslash_gbs_fp32": 7002.3, "cg_s_per_solve_fp64": 18.3147,
        "cg_s_per_solve_fp32": 6.0803, "cg_iters_fp64": 5060, "extras": "gpurun_out/bench_extras.json",
        "variants_fp64": {"dslash": [{"x": i} for i in range(2000)]},          # sidecar material: must NOT reach the line
    }
    line = bench.headline_line(out)
    assert len(line) < bench.HEADLINE_MAX_BYTES < 4096 and "\n" not in line
    d = json.loads(line)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in d["roofline"], k
    for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"):
        assert k in d["e2e"], k
    assert "variants_fp64" not in d and d["extras"].endswith(".json")
    # an over-long optional key is dropped before a contract key is touched
    out2 = dict(out, data="x" * 3000)
    d2 = json.loads(bench.headline_line(out2))
    assert "data" not in d2 and "roofline" in d2 and "cpu_baseline" in d2


def test_our_arm_refuses_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "1",
                        "--lattice", "4,4,4,4"], capture_output=True, text=True, cwd=ROOT, timeout=300)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)

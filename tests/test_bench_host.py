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
    for n in (1, 2, 3, 4, 6, 8, 16):
        comp, nom = bench.variant_reals(2, 1, n, 10 ** 9)           # N3 -> infinity: exactly 6 links per site
        assert abs(nom - (6 * 12 + n * 9 * 6)) < 1e-6
        assert abs(570 * n / (nom * 8) - n * 570 / (8 * (6 * 12 + n * 9 * 6))) < 1e-8
        assert abs(comp - (72 + 12 * n)) < 1e-6
    assert bench.variant_reals(2, 1, 1, 10 ** 9)[1] == pytest.approx(126)            # "a total float count of 126 per site"
    assert bench.variant_reals(3, 0, 1, 64) == (bench.REALS_DSLASH_COMPULSORY, bench.REALS_DSLASH_NOMINAL)
    assert bench.variant_reals(2, 0, 1, 64) == (108, 150)
    # the slices x3 = 0 / 1 still read their time links: 2 / N3 links per site on average
    assert bench.variant_reals(2, 1, 1, 64)[0] == pytest.approx((6 + 2 / 64) * 12 + 12)


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
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["steps"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["unit"] == "GB/s" and d["higher_is_better"] is True


def test_our_arm_refuses_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "1",
                        "--lattice", "4,4,4,4"], capture_output=True, text=True, cwd=ROOT, timeout=300)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)

"""Writes tests/golden/cg_config<i>_fp<prec>.json: the CPU oracle's CG result for one of
BASELINE.json's configs (iteration count, recurrence and true residual), so that GPU tests and
bench.py need not repeat an oracle solve that takes minutes (32^4) to hours (64^4).

    python tests/golden/make_cg_golden.py --config 4 --prec 64

Calls ONLY oracle/ and qcd_inputs/ (never the CUDA path).  The stored numbers are the
oracle's; the input fingerprint lets a test verify that it regenerated the same inputs.
"""
import argparse
import hashlib
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import qcd_inputs  # noqa: E402


def fingerprint(U: np.ndarray, b: np.ndarray) -> str:
    """sha256 over the first / last 256 links, every 4099th link and every 1031st source site (fp64 bytes)."""
    h = hashlib.sha256()
    Uf = U.reshape(-1, 3, 3)
    h.update(np.ascontiguousarray(Uf[:256]).tobytes())
    h.update(np.ascontiguousarray(Uf[-256:]).tobytes())
    h.update(np.ascontiguousarray(Uf[::4099]).tobytes())
    h.update(np.ascontiguousarray(b[::1031]).tobytes())
    return h.hexdigest()


def golden_path(config: int, prec: int) -> str:
    return os.path.join(HERE, f"cg_config{config}_fp{prec}.json")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--prec", type=int, default=64, choices=(64, 32))
    ap.add_argument("--threads", type=int, default=0)
    a = ap.parse_args()
    if a.threads:
        oracle.set_num_threads(a.threads)
    cfg, U, b = qcd_inputs.config_inputs(a.config)
    tol = cfg["tol64"] if a.prec == 64 else cfg["tol32"]
    if tol is None:
        raise SystemExit(f"config {a.config} has no fp{a.prec} solve")
    fp = fingerprint(U, b)
    cd = np.complex128 if a.prec == 64 else np.complex64
    Ur, br = U.astype(cd), b.astype(cd)
    if a.prec == 32:
        del U, b
    t0 = time.time()
    x, info = oracle.cg(cfg["dims"], Ur, br, cfg["m"], tol, cfg["maxiter"])
    secs = time.time() - t0
    true = oracle.true_residual(cfg["dims"], Ur, br, x, cfg["m"])
    out = dict(config=a.config, name=cfg["name"], dims=list(cfg["dims"]), links=cfg["links"], eps=cfg["eps"],
               m=cfg["m"], tol=tol, maxiter=cfg["maxiter"], prec=a.prec,
               iters=info["iters"], status=info["status"], rel_resid=info["rel_resid"], true_resid=true,
               bnorm2=info["bnorm2"], oracle_seconds=secs, oracle_threads=oracle.num_threads(),
               input_fingerprint=fp, written_by="tests/golden/make_cg_golden.py (oracle only)")
    with open(golden_path(a.config, a.prec), "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")
    print(json.dumps(out))


if __name__ == "__main__":
    main()

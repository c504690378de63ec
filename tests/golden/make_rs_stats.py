#!/usr/bin/env python
"""Stationary rho_C(r) of config 2 under classic RANDOM SEQUENTIAL update, by the
CPU oracle only (oracle.rs_sweep) -> tests/golden/C2_rs_stats.json.

    python tests/golden/make_rs_stats.py [--seeds 201 202] [--mcs 20000] [--procs 8]

BASELINE.json configs[1]: L=400, K=0.5, Bernoulli(0.5) start, 20000 MCS, mean of the last 10000
(time average after discarding the relaxation).  For every r and seed the file holds
the mean, and the standard error from 10 batch means of the averaging window.  The GPU test
(tests/test_gpu_physics.py) compares the sublattice schedule against these numbers; nothing here
touches the CUDA path.  About 8 core-minutes per (r, seed).
"""
from __future__ import annotations

import argparse
import json
import multiprocessing as mp
import sys
import time
from pathlib import Path

import numpy as np

HERE = Path(__file__).resolve().parent
sys.path.insert(0, str(HERE.parents[1]))

import oracle as orc  # noqa: E402
import workloads as wl  # noqa: E402


def window_stats(counts: np.ndarray, sites: int, n_batches: int = 10):
    """Mean of rho_C over the second half and its standard error from batch means."""
    w = counts[len(counts) // 2:].astype(np.float64) / sites
    b = w[: len(w) // n_batches * n_batches].reshape(n_batches, -1).mean(axis=1)
    return float(w.mean()), float(b.std(ddof=1) / np.sqrt(n_batches))


def run(job):
    L, r, K, rho0, seed, n_mcs = job
    lat = orc.init(L, rho0, seed)
    counts = orc.rs_sweep(lat, r, K, seed, 0, n_mcs)
    mean, err = window_stats(counts, L * L)
    return {"r": r, "seed": seed, "mean": mean, "stderr": err, "final": int(counts[-1])}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--seeds", type=int, nargs="+", default=[201, 202])
    ap.add_argument("--mcs", type=int, default=20000)
    ap.add_argument("--procs", type=int, default=8)
    args = ap.parse_args()
    cfg = wl.config2(n_mcs=args.mcs)
    jobs = [(cfg.L, r, cfg.K, cfg.rho0, s, cfg.n_mcs) for r in wl.config2_rs() for s in args.seeds]
    t0 = time.time()
    with mp.Pool(args.procs) as pool:
        rows = pool.map(run, jobs, chunksize=1)
    out = {"config": cfg.name, "schedule": "random sequential (oracle.rs_sweep, D8)",
           "generator": "python tests/golden/make_rs_stats.py " + " ".join(sys.argv[1:]),
           "L": cfg.L, "K": cfg.K, "rho0": cfg.rho0, "n_mcs": cfg.n_mcs, "window": "last half, 10 batch means",
           "oracle_seconds": round(time.time() - t0, 1), "rows": rows}
    (HERE / "C2_rs_stats.json").write_text(json.dumps(out, indent=1) + "\n")
    print(f"{time.time() - t0:.0f} s")


if __name__ == "__main__":
    main()

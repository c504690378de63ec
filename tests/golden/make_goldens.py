#!/usr/bin/env python
"""Write the stored expected values of the full-length parity runs (tests/golden/*.json).

    python tests/golden/make_goldens.py c2|c3|c4|c5 [--mcs N] [--procs P]

Calls ONLY ``oracle/`` (the plain C CPU oracle) and ``workloads.py`` (config names and
sizes); nothing here touches the CUDA path.  For every lattice of the config it runs the
16-sublattice Philox schedule (IID order) from the
Bernoulli(rho0) start and stores

  * ``count0`` and the SHA-256 of the whole cooperator-count trace (little-endian uint64,
    one entry per MCS: the numerator of Eq. 4),
  * the counts at log-spaced MCS (readable; they localise a mismatch in time),
  * the SHA-256 of the lattice (row-major uint8, C = 1 / D = 0) at the snapshot times.

``tests/test_gpu_goldens.py`` runs the same configs through libpgg on the GPU and compares.
The runs take minutes to an hour of CPU time each (that is why they are stored).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import multiprocessing as mp
import sys
import time
from pathlib import Path

import numpy as np

HERE = Path(__file__).resolve().parent
ROOT = HERE.parents[1]
sys.path.insert(0, str(ROOT))

import oracle as orc  # noqa: E402
import workloads as wl  # noqa: E402


def sample_times(n_mcs: int):
    """1, 2, 3, 5, 8, ... roughly 8 per decade, and the last MCS."""
    ts, t = set(), 1.0
    while t <= n_mcs:
        ts.add(int(t))
        t *= 10 ** 0.125
    ts.add(n_mcs)
    return sorted(ts)


def run_member(job):
    L, r, K, rho0, seed, n_mcs, snaps, n_threads = job
    lat = orc.init(L, rho0, seed)
    count0 = orc.count(lat)
    parts, snap_sha, t = [], {}, 0
    for stop in sorted(set(list(snaps) + [n_mcs])):
        if stop > t:
            c, _ = orc.sweep(lat, r, K, seed, orc.ORDER_IID, t, stop - t, n_threads=n_threads)
            parts.append(c)
            t = stop
        if stop in snaps:
            snap_sha[str(stop)] = hashlib.sha256(lat.tobytes()).hexdigest()
    trace = np.concatenate(parts).astype("<u8")
    return {
        "r_hex": float(r).hex(), "r": float(r), "seed": int(seed), "count0": int(count0),
        "trace_sha256": hashlib.sha256(trace.tobytes()).hexdigest(),
        "samples": {str(s): int(trace[s - 1]) for s in sample_times(n_mcs)},
        "snap_sha256": snap_sha,
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config", choices=["c2", "c3", "c4", "c5"])
    ap.add_argument("--mcs", type=int, default=0, help="MCS per lattice (default: see below)")
    ap.add_argument("--procs", type=int, default=0)
    ap.add_argument("--members", type=int, default=0, help="only the first M lattices")
    args = ap.parse_args()
    procs = args.procs or orc.max_threads()

    if args.config == "c2":      # BASELINE.json configs[1], one seed, full length
        cfg = wl.config2(seed=101, n_mcs=args.mcs or 20000)
        snaps = [cfg.n_mcs // 2, cfg.n_mcs]
    elif args.config == "c3":    # configs[2]: a prefix for all 16 seeds, or the full 10^5 MCS for a few
        cfg = wl.config3(n_mcs=args.mcs or 1000)   # (--mcs 100000 --members 2: ~6 core hours per seed)
        snaps = [cfg.n_mcs] if cfg.n_mcs < 10000 else [cfg.n_mcs // 10, cfg.n_mcs // 2, cfg.n_mcs]
    elif args.config == "c4":    # configs[3], full length
        cfg = wl.config4(n_mcs=args.mcs or 10000)
        snaps = [cfg.n_mcs // 10, cfg.n_mcs]
    else:                        # configs[4]: prefix of the 1000 MCS (full: ~12 core hours)
        cfg = wl.config5(n_mcs=args.mcs or 300)
        snaps = sorted({2, cfg.n_mcs // 10, cfg.n_mcs // 3, cfg.n_mcs})
    B = args.members or cfg.batch
    solo = B == 1
    # threads per lattice: all of them for one lattice, else what is left per pool process
    per_member = procs if solo else max(1, procs // B)
    jobs = [(cfg.L, cfg.rs[b], cfg.K, cfg.rho0, cfg.seeds[b], cfg.n_mcs, snaps, per_member)
            for b in range(B)]
    t0 = time.time()
    if solo:
        members = [run_member(jobs[0])]
    else:
        with mp.Pool(min(procs, B)) as pool:
            members = pool.map(run_member, jobs, chunksize=1)
    out = {
        "config": cfg.name, "generator": "python tests/golden/make_goldens.py " + " ".join(sys.argv[1:]),
        "source": "oracle/pgg_oracle.c only (orc_init, orc_sweep ORDER_IID)",
        "L": cfg.L, "K": cfg.K, "rho0": cfg.rho0, "order": "iid", "n_mcs": cfg.n_mcs,
        "snapshots": snaps, "oracle_seconds": round(time.time() - t0, 1), "members": members,
    }
    path = HERE / f"{cfg.name}_mcs{cfg.n_mcs}.json"
    path.write_text(json.dumps(out, indent=1) + "\n")
    print(path, f"{time.time() - t0:.0f} s")


if __name__ == "__main__":
    main()

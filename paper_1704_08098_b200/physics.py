"""Observables of the paper measured with libpgg (GPU only; thin drivers around pgg_run_ensemble).

    python -m paper_1704_08098_b200.physics stationary [--L 400] [--mcs 20000] [--seeds 101 102 103 104]
                                                       [--order iid|perm] [--rs 3.6 3.65 ...]
    python -m paper_1704_08098_b200.physics decay --r 3.7443 [--L 2048] [--mcs 100000] [--seeds 1..16] [--fmt bits]
    python -m paper_1704_08098_b200.physics fig5 [--order dtile|iid] [--mcs 2000]

``stationary``: rho_C(r) of BASELINE.json configs[1] -- the time average of Eq. (4) over
the second half of the run, with the standard error from 10 batch means, per (r, seed) and pooled.
``decay``: rho_C(t) of configs[2] averaged over seeds on log-spaced t, and the local decay exponent
delta_eff(t) = -ln[rho(t)/rho(t/8)] / ln 8 (directed percolation: delta = 0.4505; PAPER.md:97,111 place
the transition in that class).  Every number comes from the integer count traces the kernels produce;
the arithmetic here is averaging only.
``fig5``: the timing experiment of the paper's Fig. 5: L = 32 ... 4096 at K = 0.5,
r = 3.98, wall time per 10^6 full MCS, extrapolated from --mcs MCS timed with CUDA events after a
warm-up of the same length (the paper ran 10^6 MCS; its GTX 1080 / Xeon times are context only).
"""
from __future__ import annotations

import argparse
import json
import math

import numpy as np

from . import (FMT_BITS, FMT_U8, ORDER_DTILE, ORDER_IID, ORDER_PERM, pgg_init_lattice, pgg_run_ensemble, pgg_sweep)


def run_traces(L, rs, seeds, K, rho0, n_mcs, order=ORDER_IID, fmt=FMT_U8, chunk=None):
    """One lattice per (r, seed) pair in one ensemble launch -> counts [B, n_mcs] (numpy int64)."""
    import torch
    B = len(rs)
    shape = (B, L, L) if fmt == FMT_U8 else (B, L, L // 32)
    d = torch.empty(shape, dtype=torch.uint8 if fmt == FMT_U8 else torch.int32, device="cuda")
    cnt = torch.zeros((B, n_mcs), dtype=torch.int64, device="cuda")
    pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, order, rho0, 0, n_mcs, cnt)
    torch.cuda.synchronize()
    return cnt.cpu().numpy()


def window_stats(counts, sites, n_batches=10):
    w = counts[len(counts) // 2:].astype(np.float64) / sites
    b = w[: len(w) // n_batches * n_batches].reshape(n_batches, -1).mean(axis=1)
    return float(w.mean()), float(b.std(ddof=1) / math.sqrt(n_batches))


def stationary(rs, seeds, L=400, n_mcs=20000, K=0.5, rho0=0.5, order=ORDER_IID, fmt=FMT_U8):
    """-> {r: {"per_seed": [(mean, stderr)...], "mean": m, "stderr": e}}; e combines the batch-mean
    errors with the scatter between seeds (whichever is larger)."""
    pairs = [(r, s) for r in rs for s in seeds]
    tr = run_traces(L, [p[0] for p in pairs], [p[1] for p in pairs], K, rho0, n_mcs, order, fmt)
    out = {}
    for a, r in enumerate(rs):
        st = [window_stats(tr[a * len(seeds) + b], L * L) for b in range(len(seeds))]
        means = np.array([m for m, _ in st])
        within = math.sqrt(sum(e * e for _, e in st)) / len(st)
        between = float(means.std(ddof=1) / math.sqrt(len(st))) if len(st) > 1 else 0.0
        out[r] = {"per_seed": st, "mean": float(means.mean()), "stderr": max(within, between)}
    return out


def log_times(n_mcs, per_decade=8):
    ts, t = set(), 1.0
    while t <= n_mcs:
        ts.add(int(t))
        t *= 10 ** (1.0 / per_decade)
    ts.add(n_mcs)
    return sorted(ts)


def decay(r, seeds, L=2048, n_mcs=100000, K=0.5, rho0=0.5, order=ORDER_IID, fmt=FMT_U8):
    """-> list of rows {t, rho, rho_err, delta_eff, delta_err}: seed average of rho_C(t), error from the
    scatter between seeds; delta_eff(t) between t/8 and t with a seed-jackknife error."""
    tr = run_traces(L, [r] * len(seeds), seeds, K, rho0, n_mcs, order, fmt).astype(np.float64) / (L * L)
    decay.last_fit = decay_fit(tr, n_mcs)      # read by main(): the last-decade fit of the same traces
    rows = []
    n = len(seeds)
    for t in log_times(n_mcs):
        col = tr[:, t - 1]
        row = {"t": t, "alive": int((col > 0).sum()), "rho": float(col.mean()), "rho_err": float(col.std(ddof=1) / math.sqrt(n)) if n > 1 else 0.0}
        t8 = t // 8
        if t8 >= 1 and col.mean() > 0 and tr[:, t8 - 1].mean() > 0:
            def d_eff(sel):
                a, b = tr[sel, t - 1].mean(), tr[sel, t8 - 1].mean()
                return -math.log(a / b) / math.log(t / t8) if a > 0 and b > 0 else float("nan")
            full = d_eff(slice(None))
            if n > 1:
                jk = np.array([d_eff([i for i in range(n) if i != j]) for j in range(n)])
                err = float(math.sqrt((n - 1) / n * ((jk - jk.mean()) ** 2).sum()))
            else:
                err = 0.0
            row.update(delta_eff=full, delta_err=err)
        rows.append(row)
    return rows


def decay_fit(tr, n_mcs, t_lo=None):
    """Least-squares slope of ln rho(t) against ln t over the log-spaced times in [t_lo, n_mcs] (default: the
    last decade), rho = seed mean; error from a jackknife over the seeds.  tr: [n_seeds, n_mcs] densities."""
    t_lo = t_lo or max(1, n_mcs // 10)
    ts = np.array([t for t in log_times(n_mcs) if t >= t_lo])
    x = np.log(ts.astype(np.float64))

    def slope(sel):
        y = tr[sel][:, ts - 1].mean(axis=0)
        if (y <= 0).any():
            return float("nan")
        return -float(np.polyfit(x, np.log(y), 1)[0])
    n = tr.shape[0]
    full = slope(slice(None))
    if n > 1:
        jk = np.array([slope([i for i in range(n) if i != j]) for j in range(n)])
        err = float(math.sqrt((n - 1) / n * ((jk - jk.mean()) ** 2).sum()))
    else:
        err = 0.0
    return {"t_lo": int(ts[0]), "t_hi": int(ts[-1]), "points": int(len(ts)), "delta": full, "delta_err": err}


def fig5(order=ORDER_DTILE, n_mcs=2000, Ls=(32, 64, 128, 256, 512, 1024, 2048, 4096), r=3.98, K=0.5, seed=1):
    """-> rows {L, ms_per_mcs, updates_per_s, hours_per_1e6_mcs, rho_C}."""
    import torch
    rows = []
    stream = torch.cuda.current_stream()
    for L in Ls:
        d = torch.empty((L, L), dtype=torch.uint8, device="cuda")
        cnt = torch.zeros(n_mcs, dtype=torch.int64, device="cuda")
        pgg_init_lattice(d, FMT_U8, L, 0.5, seed, stream)
        pgg_sweep(d, FMT_U8, L, r, K, seed, order, 0, n_mcs, None, stream)       # warm-up, reaches rho_C ~ 0.5
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        pgg_sweep(d, FMT_U8, L, r, K, seed, order, n_mcs, n_mcs, cnt, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / n_mcs
        rows.append({"L": L, "ms_per_mcs": ms, "updates_per_s": L * L / (ms * 1e-3),
                     "hours_per_1e6_mcs": ms * 1e3 / 3600.0, "rho_C": float(cnt[-1]) / (L * L)})
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("what", choices=["stationary", "decay", "fig5"])
    ap.add_argument("--L", type=int, default=0)
    ap.add_argument("--mcs", type=int, default=0)
    ap.add_argument("--seeds", type=int, nargs="+", default=None)
    ap.add_argument("--order", default="iid", choices=["iid", "perm", "dtile"])
    ap.add_argument("--rs", type=float, nargs="+", default=None)
    ap.add_argument("--r", type=float, default=3.7443)
    ap.add_argument("--fmt", default="u8", choices=["u8", "bits"], help="lattice layout (same trajectories; bits is the fast path for L >= 1024)")
    args = ap.parse_args()
    order = {"iid": ORDER_IID, "perm": ORDER_PERM, "dtile": ORDER_DTILE}[args.order]
    if args.what == "fig5":
        print(json.dumps({"what": "fig5", "order": args.order, "r": 3.98, "mcs_timed": args.mcs or 2000,
                          "rows": fig5(order, args.mcs or 2000)}))
    elif args.what == "stationary":
        rs = args.rs or [round(3.60 + 0.05 * a, 2) for a in range(9)] + [5.3, 5.4, 5.5, 5.6]
        seeds = args.seeds or [101, 102, 103, 104]
        res = stationary(rs, seeds, args.L or 400, args.mcs or 20000, order=order,
                         fmt=FMT_BITS if args.fmt == "bits" else FMT_U8)
        print(json.dumps({"what": "stationary", "order": args.order, "L": args.L or 400, "mcs": args.mcs or 20000,
                          "fmt": args.fmt, "seeds": seeds, "rows": [{"r": r, **v} for r, v in res.items()]}))
    else:
        seeds = args.seeds or list(range(1, 17))
        rows = decay(args.r, seeds, args.L or 2048, args.mcs or 100000, order=order,
                     fmt=FMT_BITS if args.fmt == "bits" else FMT_U8)
        print(json.dumps({"what": "decay", "order": args.order, "r": args.r, "L": args.L or 2048, "fmt": args.fmt,
                          "mcs": args.mcs or 100000, "seeds": seeds, "last_decade_fit": decay.last_fit, "rows": rows}))


if __name__ == "__main__":
    main()

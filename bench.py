#!/usr/bin/env python
"""bench.py -- throughput of the PGG Monte Carlo sweep on BASELINE.json configs[4].

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--fmt u8|bits] [--L 16384] [--mcs 1000] [--variant auto|v0|tile]

One *step* is one whole pass of the hot path over the throughput workload: Bernoulli(0.5)
initial condition from seed 1 (K0) followed by `--mcs` full Monte Carlo steps (16 phase
launches each: class draw, staging, Philox draws, payoff differences, acceptance,
in-place writes, fused density) on a single L x L lattice, r = 3.8, K = 0.5.
Metric: elementary strategy updates per second (BASELINE.json `metric`), plus the
fraction of the HBM roofline for the sweep's contract bytes (17 B/update for uint8,
SURVEY.md section 8(d)).

N > 1 (torchrun): the path has no exchange step on one GPU, so ranks run independent
replicas (rank q uses seed 1+q) -- weak scaling, no data-path collective.

`--impl reference` times the CPU oracle (oracle/, plain C, as it stands) on the host
cores, one MCS of the same workload per step.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

R, K_NOISE, RHO0, SEED = 3.8, 0.5, 0.5, 1           # BASELINE.json configs[4]; --rho0 overrides RHO0 (profiling aid)
METRIC = "elementary strategy updates/sec at L=16384"


def load_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-i", str(self.index), "-lms", "200"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown",
                                "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


ORC_ORDER = 0  # oracle order mode of the cpu_baseline / reference legs (set from --order)


def oracle_sample(L: int, max_mcs: int, min_seconds: float, threads: int = 0):
    """Time the oracle (as it stands) on the first MCS of the workload (MCS 0 .. done-1 from the
    Bernoulli start), on `threads` host threads (0 = all)."""
    import numpy as np
    import oracle as orc
    threads = threads or orc.max_threads()
    lat = orc.init(L, RHO0, SEED)
    done, t0 = 0, time.perf_counter()
    while done < max_mcs:
        orc.sweep(lat, R, K_NOISE, SEED, ORC_ORDER, done, 1, n_threads=threads)
        done += 1
        if time.perf_counter() - t0 >= min_seconds:
            break
    dt = time.perf_counter() - t0
    return done * L * L / dt, threads, done, dt


def max_over_ranks(vals, world, device="cpu"):
    """Timings are reported as the MAX over ranks (the job is as slow as its slowest replica)."""
    if world == 1:
        return list(vals)
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(vals), device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def job_value(world, steps, updates_per_step, ms):
    """Whole-job throughput: the updates all ranks processed / the slowest rank's time."""
    return world * steps * updates_per_step / (ms * 1e-3)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle as orc
    L = args.L
    threads = orc.max_threads()
    lat = orc.init(L, RHO0, SEED)
    t = 0
    for _ in range(args.warmup):
        orc.sweep(lat, R, K_NOISE, SEED, ORC_ORDER, t, 1, n_threads=threads); t += 1
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.sweep(lat, R, K_NOISE, SEED, ORC_ORDER, t, 1, n_threads=threads); t += 1
    dt = time.perf_counter() - t0
    value = args.steps * L * L / dt
    sample = (f"each step = 1 MCS; timed window = MCS {args.warmup}..{t - 1} of the L={L} workload from the "
              f"Bernoulli(0.5) seed-1 start (after {args.warmup} warm-up MCS the state is sparser than at MCS 0, so the "
              f"rate differs from cpu_baseline's window MCS 0..7); oracle/pgg_oracle.c -O2, rows of a class split over threads")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": "updates/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8",
        "data": "synthetic", "config": {"workload": f"C5 L={L} r={R} K={K_NOISE} rho0={RHO0} seed={SEED}",
                                        "fmt": "u8", "mcs_per_step": 1},
        "cpu_baseline": {"value": value, "unit": "updates/s", "cores": threads, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": "updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_1704_08098_b200 as pgg

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    pgg.lib()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    L, n_mcs = args.L, args.mcs
    ORDER = {"iid": pgg.ORDER_IID, "perm": pgg.ORDER_PERM, "dtile": pgg.ORDER_DTILE}[args.order]
    dtile = args.order == "dtile"
    fmt = pgg.FMT_U8 if args.fmt == "u8" else pgg.FMT_BITS
    variant = {"auto": pgg.VARIANT_AUTO, "v0": pgg.VARIANT_V0, "tile": pgg.VARIANT_TILE,
               "pipe": pgg.VARIANT_PIPE, "band": pgg.VARIANT_BAND,
               "ring": pgg.VARIANT_RING, "split": pgg.VARIANT_SPLIT, "dyn": pgg.VARIANT_DYN, "resident": pgg.VARIANT_RESIDENT, "lean": pgg.VARIANT_LEAN, "persist": pgg.VARIANT_PERSIST, "cluster": pgg.VARIANT_CLUSTER, "packed": pgg.VARIANT_PACKED}[args.variant]
    pgg.pgg_set_variant(variant)
    seed = SEED + rank
    shape = (L, L) if fmt == pgg.FMT_U8 else (L, L // 32)
    tdtype = torch.uint8 if fmt == pgg.FMT_U8 else torch.int32
    d_lat = torch.empty(shape, dtype=tdtype, device="cuda")
    d_counts = torch.zeros(n_mcs, dtype=torch.int64, device="cuda")
    stream = torch.cuda.current_stream()
    lat_bytes = d_lat.numel() * d_lat.element_size()

    ev_a = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ev_b = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ev_c = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]

    def step(i=None):
        if i is not None:
            ev_a[i].record(stream)
        pgg.pgg_init_lattice(d_lat, fmt, L, RHO0, seed, stream)
        if i is not None:
            ev_b[i].record(stream)
        if args.profile_mcs >= 0:
            # for `ncu --profile-from-start off`: only MCS `profile_mcs` lies in the profiled range
            pm = min(args.profile_mcs, n_mcs - 1)
            pgg.pgg_sweep(d_lat, fmt, L, R, K_NOISE, seed, ORDER, 0, pm, None, stream)
            torch.cuda.synchronize()
            torch.cuda.profiler.start()
            pgg.pgg_sweep(d_lat, fmt, L, R, K_NOISE, seed, ORDER, pm, 1, None, stream)
            torch.cuda.synchronize()
            torch.cuda.profiler.stop()
            pgg.pgg_sweep(d_lat, fmt, L, R, K_NOISE, seed, ORDER, pm + 1, n_mcs - pm - 1, None, stream)
            pgg.pgg_init_lattice(d_lat, fmt, L, RHO0, seed, stream)
        pgg.pgg_sweep(d_lat, fmt, L, R, K_NOISE, seed, ORDER, 0, n_mcs, d_counts, stream)
        if i is not None:
            ev_c[i].record(stream)

    # ---- device-resident timing: W warm-up steps, then exactly K steps
    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = pgg.pgg_launch_count()
    for i in range(args.steps):
        step(i)
    barrier()
    launches = pgg.pgg_launch_count() - launches0
    variant_used = pgg.pgg_get_variant_used()
    # PACKED: the uint8 lattice is the caller's layout only; the kernels run on a bit-packed working copy
    packed = variant_used == pgg.VARIANT_PACKED
    clocks = sampler.stop() if rank == 0 else None
    total_ms = ev_a[0].elapsed_time(ev_c[-1])
    sweep_ms = sum(ev_b[i].elapsed_time(ev_c[i]) for i in range(args.steps))
    last_counts = d_counts.cpu()
    total_ms, sweep_ms = max_over_ranks([total_ms, sweep_ms], world, "cuda")
    updates_per_step = float(n_mcs) * L * L
    value = job_value(world, args.steps, updates_per_step, total_ms)

    # ---- end to end through the C ABI with HOST buffers (pinned): per step copy the initial
    # lattice host->device, sweep, copy the final lattice and the count trace device->host.
    h_lat0 = torch.empty(shape, dtype=tdtype).pin_memory()
    pgg.pgg_init_lattice(d_lat, fmt, L, RHO0, seed, stream)
    h_lat0.copy_(d_lat)
    h_out = torch.empty(shape, dtype=tdtype).pin_memory()
    h_counts = torch.empty(n_mcs, dtype=torch.int64).pin_memory()

    def e2e_step():
        d_lat.copy_(h_lat0, non_blocking=True)
        pgg.pgg_sweep(d_lat, fmt, L, R, K_NOISE, seed, ORDER, 0, n_mcs, d_counts, stream)
        h_out.copy_(d_lat, non_blocking=True)
        h_counts.copy_(d_counts, non_blocking=True)
        stream.synchronize()

    e2e_steps = max(1, min(args.steps, 3))
    e2e_step()
    barrier()
    t0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(e2e_steps):
        e2e_step()
    e1.record(stream)
    barrier()
    e2e_ms = max(e0.elapsed_time(e1), 0.0)
    e2e_wall_ms = (time.perf_counter() - t0) * 1e3
    (e2e_ms,) = max_over_ranks([e2e_ms], world, "cuda")
    e2e_value = job_value(world, e2e_steps, updates_per_step, e2e_ms)
    assert torch.equal(h_counts, last_counts), "e2e run and device-resident run disagree"

    # ---- context for a PACKED run: the same step on the in-place streaming kernel (RING reads the uint8 rows
    # from HBM every phase), one warm-up + one timed step, so that its HBM fraction stays on record
    streaming = None
    if packed and not args.no_streaming_context and pgg.pgg_variant_supported(pgg.VARIANT_RING, fmt, L):
        pgg.pgg_set_variant(pgg.VARIANT_RING)
        step()
        s0, s1, s2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        s0.record(stream)
        pgg.pgg_init_lattice(d_lat, fmt, L, RHO0, seed, stream)
        s1.record(stream)
        pgg.pgg_sweep(d_lat, fmt, L, R, K_NOISE, seed, ORDER, 0, n_mcs, d_counts, stream)
        s2.record(stream)
        barrier()
        assert torch.equal(d_counts.cpu(), last_counts), "RING and PACKED disagree"
        pgg.pgg_set_variant(variant)
        us = s1.elapsed_time(s2) * 1e3 / (16 * n_mcs)
        gbs = (L * L * 17.0 / 16.0) / (us * 1e-6) / 1e9
        pk, _ = load_peaks()
        streaming = {"variant": pgg.VARIANT_RING, "kernel": "phase_ring_kernel, in place on the uint8 rows",
                     "updates_per_s": updates_per_step / (s0.elapsed_time(s2) * 1e-3), "avg_launch_us": us,
                     "bound": "hbm", "achieved": gbs, "peak": pk, "unit": "GB/s", "frac": gbs / pk,
                     "algorithmic_bytes_per_launch": L * L * 17.0 / 16.0, "steps": 1}
        try:
            streaming["traffic"] = json.loads((ROOT / "profiles" / "traffic.json").read_text()).get(f"u8_L{L}_bytes_per_launch")
        except (ValueError, OSError):
            streaming["traffic"] = None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- the ALU ceiling: STEP draws per second of a Philox-only kernel
    n_draws = pgg.pgg_probe_draw_rate(64, seed, stream)          # warm-up launch
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record(stream)
    n_draws = sum(pgg.pgg_probe_draw_rate(2048, seed, stream) for _ in range(4))
    p1.record(stream)
    stream.synchronize()
    draws_per_s = n_draws / (p0.elapsed_time(p1) * 1e-3)
    # the draw fraction of the workload: sites with a neighbour of the other strategy (S9), sampled
    # at log-spaced MCS of the same deterministic run (untimed) and averaged over time
    d_if = torch.zeros(1, dtype=torch.int64, device="cuda")
    stops = sorted({0, n_mcs} | {min(n_mcs, int(round(10 ** (a / 4.0)))) for a in range(0, 4 * 8)})
    pgg.pgg_init_lattice(d_lat, fmt, L, RHO0, seed, stream)
    f_t, t_prev = [], 0
    for t_stop in stops:
        if t_stop > t_prev:
            pgg.pgg_sweep(d_lat, fmt, L, R, K_NOISE, seed, ORDER, t_prev, t_stop - t_prev, None, stream)
            t_prev = t_stop
        pgg.pgg_count_interface(d_lat, fmt, L, d_if, stream)
        stream.synchronize()
        f_t.append((t_stop, d_if.item() / float(L * L)))
    draw_fraction = (sum(0.5 * (f_t[a][1] + f_t[a + 1][1]) * (f_t[a + 1][0] - f_t[a][0]) for a in range(len(f_t) - 1))
                     / max(1, n_mcs)) if n_mcs else f_t[0][1]

    # ---- roofline of the dominant kernel (the phase kernel; 16 launches per MCS)
    peak, peak_src = load_peaks()
    # (the paper's double-tiling schedule, --order dtile: 4 parts per MCS, each reads N and writes N/4)
    per_mcs = 4 if dtile else 16
    n_phase = per_mcs * n_mcs * args.steps
    phase_us = sweep_ms * 1e3 / n_phase            # includes the per-call order/density/finalize kernels
    b_site = 1.0 if (fmt == pgg.FMT_U8 and not packed) else 0.125   # of the layout the phase kernel reads
    bytes_per_launch = (L * L + L * L / float(per_mcs)) * b_site   # read the lattice, write the active class
    achieved = bytes_per_launch / (phase_us * 1e-6) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                "kernel": ("dtile_part_kernel" if dtile else
                           "phase_lean_kernel on the bit-packed working copy" if packed else "phase kernel") + " (variant %d)" % variant_used,
                "avg_launch_us": phase_us, "algorithmic_bytes_per_launch": bytes_per_launch,
                "note": ("5 B/update (4 parts x (read N + write N/4)); 16 full Philox draws per domain make this "
                         "schedule ALU-bound, the HBM fraction is context" if dtile else
                         "17 B/update contract bytes (16 phases x (read N + write N/16)), SURVEY 8(d)")
                        + ("; the 32 MiB packed lattice is L2-resident, so this is not a DRAM fraction"
                           if (fmt == pgg.FMT_BITS or packed) else "")}
    tr = ROOT / "profiles" / "traffic.json"
    if tr.exists():
        try:
            roofline["traffic"] = json.loads(tr.read_text()).get(
                f"{'bits' if packed else args.fmt}_L{L}_bytes_per_launch" + ("_dtile" if dtile else ""))
        except (ValueError, OSError):
            pass
    # the ALU view: STEP draws per second against the Philox-only ceiling
    sweep_rate = args.steps * updates_per_step / (sweep_ms * 1e-3)
    alu = {"bound": "alu", "achieved": sweep_rate * draw_fraction / 1e9, "peak": draws_per_s / 1e9,
           "unit": "Gdraw/s", "frac": sweep_rate * draw_fraction / draws_per_s,
           "draw_fraction": draw_fraction,
           "note": "achieved = updates/s x the time-averaged fraction of sites that need a draw "
                   "(pgg_count_interface at log-spaced MCS of the same run); peak = pgg_probe_draw_rate, "
                   "a kernel that makes STEP draws only (DESIGN.md section 5)"}
    # instruction-issue view: warp instructions of one launch (ncu, profiles/traffic.json) over the measured launch time
    # against what the SMs can issue (one warp instruction per cycle and scheduler, 4 schedulers per SM)
    issue = None
    try:
        n_inst = json.loads(tr.read_text()).get(f"{'bits' if (packed or fmt == pgg.FMT_BITS) else 'u8'}_L{L}_warp_instructions_per_launch")
        if n_inst and not dtile and clocks and clocks.get("sm_mhz"):
            sms = torch.cuda.get_device_properties(local).multi_processor_count
            peak_issue = sms * 4 * clocks["sm_mhz"] * 1e6
            issue = {"warp_instructions_per_launch": n_inst, "achieved": n_inst / (phase_us * 1e-6) / 1e9,
                     "peak": peak_issue / 1e9, "unit": "Gwarp-inst/s", "frac": n_inst / (phase_us * 1e-6) / peak_issue,
                     "note": "ncu smsp__inst_executed.sum of one launch at MCS 600 / this run's average launch time; "
                             "peak = SMs x 4 schedulers x the SM clock sampled during the timed region"}
    except (ValueError, OSError):
        pass
    if (fmt == pgg.FMT_BITS or packed) and not dtile:
        # the packed lattice is L2-resident: its bound is integer instruction issue, not HBM
        alu.update({"traffic": roofline["traffic"], "kernel": roofline["kernel"], "avg_launch_us": phase_us,
                    "hbm_context": {k: roofline[k] for k in ("achieved", "peak", "frac", "algorithmic_bytes_per_launch")}})
        if packed:
            # SURVEY 8(d)'s contract figure for a uint8 lattice, 17 B per update, over the same time: what the
            # north_star's "% of the HBM roofline" formula gives.  NOT bytes this path moves (see hbm_context).
            contract = (L * L + L * L / 16.0) / (phase_us * 1e-6) / 1e9
            alu["hbm_contract_u8"] = {"achieved": contract, "peak": peak, "unit": "GB/s", "frac": contract / peak,
                                      "note": "updates/s x 17 B / peak (SURVEY 8(d)); the phase kernel reads the 1/8-size "
                                              "working copy instead of the uint8 rows, so this is not DRAM traffic"}
            if streaming is not None:
                alu["streaming_kernel_u8"] = streaming
        roofline = alu
    else:
        roofline["alu_context"] = {k: alu[k] for k in ("achieved", "peak", "unit", "frac", "draw_fraction")}

    if issue is not None:
        roofline["issue_context"] = issue
    out = {
        "metric": METRIC, "value": value, "unit": "updates/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": ("u8 (lattice in HBM) / u1 (bit-packed u32 working copy the phases run on)" if packed
                  else "u8" if fmt == pgg.FMT_U8 else "u1 (bit-packed u32)"),
        "data": "synthetic",
        "config": {"workload": f"C5 throughput: single L={L} lattice, Bernoulli(0.5) init seed 1, r={R}, "
                               f"K={K_NOISE}, {n_mcs} MCS per step (init + sweep + fused rho_C trace)",
                   "fmt": args.fmt, "L": L, "mcs_per_step": n_mcs, "order_mode": args.order,
                   "variant": variant_used,
                   "l2": ("the call packs the uint8 lattice into a working copy of 1/8 its size, which fits L2; "
                          "no flush between phases (there is none in the workload)" if packed and lat_bytes / 8 < 120e6
                          else "inputs larger than L2 (256 MiB lattice re-read every phase)" if lat_bytes > 130e6
                          else "lattice fits L2 by nature of the workload; no flush"),
                   "parallelism": f"replicas x{world}" if world > 1 else "single GPU"},
        "mcs_per_s": world * args.steps * n_mcs / (total_ms * 1e-3),
        "sweep_only_updates_per_s": args.steps * updates_per_step / (sweep_ms * 1e-3),
        "final_rho_C": float(last_counts[-1]) / (L * L),
        "gpu_launches": int(launches),
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "updates/s", "h2d_bytes_per_step": lat_bytes,
                "d2h_bytes_per_step": lat_bytes + 8 * n_mcs, "steps": e2e_steps,
                "ms_per_step": e2e_ms / e2e_steps, "wall_ms_per_step": e2e_wall_ms / e2e_steps},
        "roofline": roofline,
        "ceilings": {"philox_step_draws_per_s": draws_per_s,
                     "note": "pgg_probe_draw_rate: every thread of a full grid makes STEP draws only "
                             "(Philox4x32-10, words x0/x1, two chains per thread); the rate no phase kernel "
                             "can exceed for the sites that need a draw (SURVEY 8(d)(ii))"},
    }
    if world == 1 and not args.no_cpu_baseline:
        v, threads, n_done, dt = oracle_sample(L, max_mcs=8, min_seconds=10.0)
        v1, _, n1, dt1 = oracle_sample(L, max_mcs=1, min_seconds=0.0, threads=1)
        # the like-for-like analogue of the paper's CPU rows: classic random sequential update
        import oracle as orc
        L_rs = min(L, 4096)
        lat_rs = orc.init(L_rs, RHO0, SEED)
        t_rs = time.perf_counter()
        orc.rs_sweep(lat_rs, R, K_NOISE, SEED, 0, 2)
        dt_rs = time.perf_counter() - t_rs
        out["cpu_baseline"] = {"value": v, "unit": "updates/s", "cores": threads, "kind": "oracle",
                               "sample": f"MCS 0..{n_done - 1} (the dense start: rho_C 0.5 -> 0.04) of the same L={L} "
                                         f"workload ({dt:.1f} s wall), oracle/pgg_oracle.c as it stands, class rows "
                                         f"split over {threads} OpenMP threads",
                               "one_thread": {"value": v1, "unit": "updates/s", "cores": 1,
                                              "sample": f"MCS 0 of the same workload ({dt1:.1f} s wall)"},
                               "random_sequential": {"value": 2.0 * L_rs * L_rs / dt_rs, "unit": "updates/s", "cores": 1,
                                                     "sample": f"oracle's random sequential mode (PAPER.md:58,65), "
                                                               f"L={L_rs}, MCS 0..1 ({dt_rs:.1f} s wall); the paper's Xeon: "
                                                               f"~6.5e6 updates/s at L=4096 (PAPER.md:115)"}}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--fmt", default="u8", choices=["u8", "bits"])
    ap.add_argument("--L", type=int, default=16384)
    ap.add_argument("--mcs", type=int, default=1000)
    ap.add_argument("--variant", default="auto", choices=["auto", "v0", "tile", "pipe", "band", "ring", "split", "dyn", "resident", "lean", "persist", "cluster", "packed"])
    ap.add_argument("--order", default="iid", choices=["iid", "perm", "dtile"],
                    help="schedule: the 16-sublattice schedule with i.i.d. (bench default) or permuted classes, or "
                         "the paper's own double-tiling schedule (PAPER.md:75-93); anything but iid is not the bench workload")
    ap.add_argument("--r", type=float, default=R, help="synergy factor; anything but 3.8 is not the bench workload")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-streaming-context", action="store_true",
                    help="skip the extra RING step a PACKED run adds for context (roofline.streaming_kernel_u8)")
    ap.add_argument("--profile-mcs", type=int, default=-1,
                    help="profiling aid: bracket this MCS with cudaProfilerStart/Stop (ncu --profile-from-start off); "
                         "the run's numbers are then not bench values")
    ap.add_argument("--rho0", type=float, default=RHO0,
                    help="initial cooperator fraction; 0 gives an all-D lattice (no site ever needs a draw): the "
                         "pure streaming rate of the phase kernel.  Anything but 0.5 is not the bench workload")
    args = ap.parse_args()
    globals()["RHO0"] = args.rho0
    globals()["R"] = args.r
    globals()["ORC_ORDER"] = {"iid": 0, "perm": 1, "dtile": 2}[args.order]
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

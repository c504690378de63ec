"""Which kernel variant for which workload: the timing loops behind PGG_VARIANT_AUTO (GPU only).

    python -m paper_1704_08098_b200.tune small      # L = 128 .. 2048, B = 1, 4, 13, 52, both layouts
    python -m paper_1704_08098_b200.tune ensembles  # config-3-like ensembles and single large lattices
    python -m paper_1704_08098_b200.tune cluster    # L = 1024 .. 4096: streaming kernels against the cluster-resident one

Every entry is the time of ``pgg_run_ensemble`` under ``pgg_set_variant(v)`` measured with CUDA
events after a warm-up, divided by 16 x MCS: microseconds per phase (for RESIDENT, which runs a whole
call in one launch, the per-phase share of that launch).  Marshalling and timing only; the variants
are bit-identical (tests/test_gpu_parity.py), so this is a pure speed comparison.
"""
from __future__ import annotations

import sys

from . import (FMT_BITS, FMT_U8, ORDER_IID, VARIANT_AUTO, VARIANT_BAND, VARIANT_CLUSTER, VARIANT_LEAN, VARIANT_PACKED, VARIANT_RESIDENT, VARIANT_RING,
               VARIANT_V0, pgg_density, pgg_run_ensemble, pgg_set_variant, pgg_variant_supported)

K = 0.5
NAMES = {VARIANT_V0: "V0", VARIANT_RESIDENT: "RESIDENT", VARIANT_RING: "RING", VARIANT_BAND: "BAND", VARIANT_LEAN: "LEAN",
         VARIANT_CLUSTER: "CLUSTER", VARIANT_PACKED: "PACKED"}


def time_variant(variant, fmt, B, L, r, warm, n):
    """-> (us per phase, rho_C of lattice 0 at the end) or None if the variant does not run (fmt, L)."""
    import torch
    if not pgg_variant_supported(variant, fmt, L):
        return None
    shape = (B, L, L) if fmt == FMT_U8 else (B, L, L // 32)
    d = torch.empty(shape, dtype=torch.uint8 if fmt == FMT_U8 else torch.int32, device="cuda")
    seeds, rs = list(range(1, B + 1)), [r] * B
    pgg_set_variant(VARIANT_AUTO)
    pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, ORDER_IID, 0.5, 0, warm, None)
    pgg_set_variant(variant)
    pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, ORDER_IID, -1.0, warm, 10, None)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, ORDER_IID, -1.0, warm + 10, n, None)
    e1.record()
    torch.cuda.synchronize()
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    pgg_density(d[0], fmt, L, cnt)
    torch.cuda.synchronize()
    pgg_set_variant(VARIANT_AUTO)
    return e0.elapsed_time(e1) * 1e3 / (16 * n), cnt.item() / float(L * L)


def table(cases, variants):
    print("| layout | B | L | r | rho_C | " + " | ".join(NAMES[v] for v in variants) + " |")
    print("|---|---|---|---|---|" + "---|" * len(variants))
    for fmt, B, L, r, warm, n in cases:
        if fmt == FMT_BITS and L % 32:
            continue
        cells, rho = [], None
        for v in variants:
            res = time_variant(v, fmt, B, L, r, warm, n)
            cells.append("-" if res is None else f"{res[0]:.2f}")
            rho = res[1] if res is not None else rho
        print(f"| {'u8' if fmt == FMT_U8 else 'bits'} | {B} | {L} | {r} | {rho:.3f} | " + " | ".join(cells) + " |", flush=True)


def main():
    what = sys.argv[1] if len(sys.argv) > 1 else "small"
    variants = [VARIANT_V0, VARIANT_RESIDENT, VARIANT_RING, VARIANT_BAND, VARIANT_LEAN, VARIANT_CLUSTER]
    if what == "small":
        cases = [(fmt, B, L, 3.8, 60, 300 if L <= 512 else 100)
                 for fmt in (FMT_U8, FMT_BITS) for L in (128, 256, 320, 400, 448, 512, 1024, 2048) for B in (1, 4, 13, 52)]
    elif what == "ensembles":
        shapes = [(16, 2048, 3.7446, 2000, 200), (16, 2048, 3.8, 500, 200), (1, 4096, 3.7446, 1000, 200),
                  (16, 4096, 3.7446, 1000, 100), (1, 8192, 3.8, 300, 100), (64, 1024, 3.75, 500, 200)]
        cases = [(fmt, B, L, r, warm, n) for (B, L, r, warm, n) in shapes for fmt in (FMT_U8, FMT_BITS)]
        variants = [VARIANT_RING, VARIANT_BAND, VARIANT_LEAN, VARIANT_CLUSTER, VARIANT_PACKED]
    elif what == "cluster":   # where the lattice fits a cluster's shared memory: L = 1024, 2048, 4096
        shapes = [(1, 1024, 3.8, 100, 300), (1, 2048, 3.8, 100, 300), (1, 4096, 3.8, 100, 200), (1, 4096, 3.7446, 1000, 200),
                  (16, 2048, 3.7446, 2000, 200), (16, 2048, 3.8, 500, 200), (64, 1024, 3.75, 500, 200),
                  (9, 4096, 3.7446, 1000, 100), (16, 4096, 3.7446, 1000, 100), (64, 2048, 3.7446, 500, 100)]
        cases = [(fmt, B, L, r, warm, n) for (B, L, r, warm, n) in shapes for fmt in (FMT_U8, FMT_BITS)]
        variants = [VARIANT_RING, VARIANT_LEAN, VARIANT_CLUSTER, VARIANT_PACKED]
    else:
        raise SystemExit(__doc__)
    table(cases, variants)


if __name__ == "__main__":
    main()

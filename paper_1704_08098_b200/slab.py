"""Row-slab sharding of ONE lattice over several GPUs -- the host side of ``pgg_slab_sweep`` (include/pgg.h;
SURVEY.md section 8(e): "1-D row slabs, after each phase exchange the 3 boundary rows each way").

What is here is layout arithmetic and wiring only: which rows a rank owns, how a slab buffer (own rows plus
three halo rows on either side, the periodic images of PAPER.md:45) is cut out of a lattice and put back,
which pointers of which neighbour a slab pushes its boundary rows to.  Every step of the method runs in the
library's kernels; the halo push is fused into the phase kernel and the order between phases is kept by
flags in device memory, so there is no collective on the data path -- ``run_distributed`` uses
``torch.distributed`` to exchange 64-byte IPC handles once and to sum the per-MCS flip counts at the end.

``LocalSlabs`` holds S slabs of one lattice on ONE device and drives them phase by phase on one stream
(launch order = dependency order, so the flags are always found set): the single-GPU test of the kernel,
the push and the flag protocol (tests/test_gpu_slab.py).  ``run_distributed`` is the one-process-per-GPU
driver; its wiring is covered on CPU with gloo (tests/test_slab_host.py).
"""
from __future__ import annotations

from . import (FMT_BITS, FMT_U8, SLAB_MAX_MCS, pgg_pd_slab_sweep, pgg_slab_alloc, pgg_slab_bytes, pgg_slab_free, pgg_slab_ipc_close,
               pgg_slab_ipc_export, pgg_slab_ipc_open, pgg_slab_step_rows, pgg_slab_sweep)

HALO = 3          # rows: the read stencil of an elementary step has radius 3
FLAG_BYTES = 256  # the three flag words of a slab, in a block of their own behind the rows


def slab_rows(L: int, world: int, rank: int, align: int = 4) -> tuple[int, int]:
    """-> (row0, n_rows) of rank's slab: the L/align row groups split as evenly as possible, in rank order.
    align = 4 (a class row every four rows) or a multiple the fast kernel wants (pgg_slab_step_rows); an align
    the lattice is too small for (fewer groups than ranks) falls back to 4."""
    if align % 4 or align < 4 or L % align or L // align < world:
        align = 4
    groups = L // align
    if L % 4 or not 1 <= world <= groups or not 0 <= rank < world:
        raise ValueError(f"L = {L}, world = {world}, rank = {rank}: need L % 4 == 0 and 1 <= world <= L / 4")
    base, rem = divmod(groups, world)
    g0 = rank * base + min(rank, rem)
    return align * g0, align * (base + (1 if rank < rem else 0))


def neighbours(world: int, rank: int) -> tuple[int, int]:
    """-> (upper, lower) neighbour ranks: the slabs form a ring (rows are periodic)."""
    return (rank - 1) % world, (rank + 1) % world


def row_bytes(fmt: int, L: int) -> int:
    return L if fmt == FMT_U8 else L // 8


def scatter(full, row0: int, n_rows: int):
    """Slab buffer of lattice rows [row0, row0 + n_rows) with its halo rows, cut out of a whole lattice
    (a [L, W] tensor, W = L for uint8 and L/32 for bit rows): buffer row q = lattice row (row0 - 3 + q) mod L."""
    import torch
    L = full.shape[0]
    idx = (torch.arange(row0 - HALO, row0 + n_rows + HALO, device=full.device) % L)
    return full.index_select(0, idx).contiguous()


def own_rows(slab):
    return slab[HALO:slab.shape[0] - HALO]


def gather(slabs):
    """Whole lattice from the slabs' own rows, in rank order."""
    import torch
    return torch.cat([own_rows(s) for s in slabs], dim=0)


class _RawCuda:
    """A device allocation as something torch.as_tensor understands (CUDA array interface, bytes)."""

    def __init__(self, ptr: int, n_bytes: int):
        self.__cuda_array_interface__ = {"shape": (n_bytes,), "typestr": "|u1", "data": (ptr, False), "version": 2}


def as_byte_tensor(ptr: int, n_bytes: int, device):
    import torch
    return torch.as_tensor(_RawCuda(ptr, n_bytes), device=device)


def halo_offsets(fmt: int, L: int, n_rows: int) -> tuple[int, int, int]:
    """Byte offsets inside a slab allocation: (top halo rows 0..2, bottom halo rows n_rows+3.., flag block)."""
    rb = row_bytes(fmt, L)
    return 0, (n_rows + HALO) * rb, (pgg_slab_bytes(fmt, L, n_rows) + 255) // 256 * 256


class SlabBuffer:
    """One slab in an allocation of its own (rows, then the flag block): what pgg_slab_ipc_export can export."""

    def __init__(self, fmt: int, L: int, row0: int, n_rows: int, device):
        self.fmt, self.L, self.row0, self.n_rows = fmt, L, row0, n_rows
        self.top_off, self.bottom_off, self.flag_off = halo_offsets(fmt, L, n_rows)
        self.n_bytes = self.flag_off + FLAG_BYTES
        self.ptr = pgg_slab_alloc(self.n_bytes)
        self.bytes = as_byte_tensor(self.ptr, self.n_bytes, device)

    def rows(self):
        """The (n_rows + 6) rows as a [rows, W] view: uint8 sites or int32 bit words."""
        import torch
        v = self.bytes[:self.flag_off][:pgg_slab_bytes(self.fmt, self.L, self.n_rows)]
        if self.fmt == FMT_BITS:
            return v.view(torch.int32).view(self.n_rows + 2 * HALO, self.L // 32)
        return v.view(self.n_rows + 2 * HALO, self.L)

    def free(self):
        if self.ptr:
            self.bytes = None
            pgg_slab_free(self.ptr)
            self.ptr = 0


def wire(ptr_self: int, n_rows_self: int, ptr_up: int, n_rows_up: int, ptr_dn: int, n_rows_dn: int, fmt: int, L: int):
    """Addresses a slab hands to pgg_slab_sweep, from the base addresses (local or peer) of the three allocations:
    -> dict(d_up_halo, d_dn_halo, d_flags, d_up_flag, d_dn_flag).  My first three own rows are the upper neighbour's
    BOTTOM halo; my last three are the lower neighbour's TOP halo; I post my progress to the upper neighbour's
    flags[2] (I am its lower neighbour) and to the lower neighbour's flags[1]."""
    _, bottom_up, flag_up = halo_offsets(fmt, L, n_rows_up)
    top_dn, _, flag_dn = halo_offsets(fmt, L, n_rows_dn)
    _, _, flag_self = halo_offsets(fmt, L, n_rows_self)
    return dict(d_up_halo=ptr_up + bottom_up, d_dn_halo=ptr_dn + top_dn, d_flags=ptr_self + flag_self,
                d_up_flag=ptr_up + flag_up + 8, d_dn_flag=ptr_dn + flag_dn + 4)


def phase_chunks(t_begin: int, n_mcs: int):
    """(t, n) pieces of at most SLAB_MAX_MCS MCS."""
    t, left = t_begin, n_mcs
    while left > 0:
        n = min(left, SLAB_MAX_MCS)
        yield t, n
        t, left = t + n, left - n


class LocalSlabs:
    """S slabs of one lattice on ONE device, launched phase by phase over the slabs on one stream (every slab runs
    phase p before any runs p + 1, so no kernel ever waits for a later one), with or without the flag protocol;
    the result equals pgg_sweep on the whole lattice bit for bit.  ``align``: row granularity of the split
    (None: pgg_slab_step_rows, what the fast kernel wants; 4: any split, general kernels where needed)."""

    def __init__(self, full, fmt: int, L: int, n_slabs: int, use_flags: bool = True, align: int | None = None):
        self.fmt, self.L, self.S, self.use_flags = fmt, L, n_slabs, use_flags
        self.align = pgg_slab_step_rows(fmt, L) if align is None else align  # None: what the fast kernel wants
        self.slabs = []
        for rank in range(n_slabs):
            row0, n_rows = slab_rows(L, n_slabs, rank, self.align)
            sb = SlabBuffer(fmt, L, row0, n_rows, full.device)
            sb.rows().copy_(scatter(full, row0, n_rows))
            self.slabs.append(sb)
        self.wiring = []
        for rank, sb in enumerate(self.slabs):
            up, dn = (self.slabs[q] for q in neighbours(n_slabs, rank))
            self.wiring.append(wire(sb.ptr, sb.n_rows, up.ptr, up.n_rows, dn.ptr, dn.n_rows, fmt, L))
        self.epoch = 0

    def sweep(self, r, K: float, seed: int, order_mode: int, t_begin: int, n_mcs: int, stream=None):
        """-> int64 tensor [n_mcs]: flips per MCS summed over the slabs (add the running sum to the initial count).
        r: the synergy factor, or a 4-tuple (R, S, T, P) for the prisoner's dilemma (pgg_pd_slab_sweep)."""
        import torch
        dev = self.slabs[0].bytes.device
        deltas = torch.zeros((self.S, max(n_mcs, 1)), dtype=torch.int64, device=dev)
        for t in range(t_begin, t_begin + n_mcs):
            for k in range(16):
                for rank, (sb, w) in enumerate(zip(self.slabs, self.wiring)):
                    flags = dict(d_flags=w["d_flags"], d_up_flag=w["d_up_flag"], d_dn_flag=w["d_dn_flag"]) if self.use_flags else {}
                    if isinstance(r, (tuple, list)):
                        pgg_pd_slab_sweep(sb.ptr, self.fmt, self.L, sb.row0, sb.n_rows, *r, K, seed, order_mode, t, k, 1,
                                          w["d_up_halo"], w["d_dn_halo"], epoch0=self.epoch,
                                          d_deltas=deltas[rank, t - t_begin:], stream=stream, **flags)
                    else:
                        pgg_slab_sweep(sb.ptr, self.fmt, self.L, sb.row0, sb.n_rows, r, K, seed, order_mode, t, k, 1,
                                       w["d_up_halo"], w["d_dn_halo"], epoch0=self.epoch,
                                       d_deltas=deltas[rank, t - t_begin:], stream=stream, **flags)
                self.epoch += 1
        return deltas[:, :n_mcs].sum(dim=0)

    def lattice(self):
        return gather([sb.rows() for sb in self.slabs])

    def halos_consistent(self) -> bool:
        """Every halo row equals the own row of the neighbour it mirrors."""
        import torch
        full = self.lattice()
        return all(torch.equal(sb.rows(), scatter(full, sb.row0, sb.n_rows)) for sb in self.slabs)

    def free(self):
        for sb in self.slabs:
            sb.free()


def exchange(payload, group=None):
    """All ranks' payloads (any picklable object), in rank order; -> (list, rank, world)."""
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    out = [None] * world
    dist.all_gather_object(out, payload, group=group)
    return out, rank, world


def run_distributed(full, fmt: int, L: int, r: float, K: float, seed: int, order_mode: int, t_begin: int, n_mcs: int,
                    group=None, stream=None):
    """One process per GPU (torch.distributed initialised, the CUDA device of the rank current).  Every rank passes
    the same whole initial lattice ``full`` (a CUDA tensor [L, W]; seeded initial conditions are cheap to make on
    every rank) and keeps its own rows from then on.  -> (own rows tensor [n_rows, W], deltas int64 [n_mcs] summed
    over all ranks).  The phases of all ranks run without the host: halo rows travel by stores into the
    neighbours' buffers from inside the phase kernel, order is kept by flags in device memory."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    row0, n_rows = slab_rows(L, world, rank, pgg_slab_step_rows(fmt, L))  # the same on every rank
    sb = SlabBuffer(fmt, L, row0, n_rows, full.device)
    sb.rows().copy_(scatter(full, row0, n_rows))
    torch.cuda.synchronize()
    infos, _, _ = exchange((pgg_slab_ipc_export(sb.ptr), torch.cuda.current_device(), n_rows), group)
    up, dn = neighbours(world, rank)
    opened = {}

    def base(q):
        if q == rank:
            return sb.ptr
        if q not in opened:
            opened[q] = pgg_slab_ipc_open(infos[q][0], infos[q][1])
        return opened[q]

    w = wire(sb.ptr, n_rows, base(up), infos[up][2], base(dn), infos[dn][2], fmt, L)
    dist.barrier(group)  # every slab is filled and every flag block zero before the first push
    deltas = torch.zeros(max(n_mcs, 1), dtype=torch.int64, device=full.device)
    epoch = 0
    for t, n in phase_chunks(t_begin, n_mcs):
        pgg_slab_sweep(sb.ptr, fmt, L, row0, n_rows, r, K, seed, order_mode, t, 0, 16 * n, w["d_up_halo"], w["d_dn_halo"],
                       w["d_flags"], w["d_up_flag"], w["d_dn_flag"], epoch, deltas[t - t_begin:], stream)
        epoch += 16 * n
    torch.cuda.synchronize()
    dist.all_reduce(deltas, group=group)  # the one collective: per-MCS flip counts, once per call
    mine = own_rows(sb.rows()).clone()
    dist.barrier(group)  # nobody unmaps a buffer a neighbour may still push into
    for p in opened.values():
        pgg_slab_ipc_close(p)
    sb.free()
    return mine, deltas[:n_mcs]


def _time_table(n_mcs: int = 20) -> None:
    """``python -m paper_1704_08098_b200.slab``: microseconds per phase of the slab kernel on ONE device -- a slab
    of L / S rows that is its own neighbour (the work and the flag traffic one of S GPUs has; only the timing is
    meaningful for S > 1) -- beside pgg_sweep on the whole lattice (V0 and AUTO), from the state after 50 MCS."""
    import torch
    import paper_1704_08098_b200 as pgg

    def timed(fn, reps=3):
        best = float("inf")
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        return best * 1e3 / (16 * n_mcs)

    print("| layout | L | pgg_sweep V0 | pgg_sweep AUTO | slab S=1 | S=2 | S=4 | S=8 |")
    print("|---|---|---|---|---|---|---|---|")
    for fmt, name in ((FMT_U8, "uint8"), (FMT_BITS, "bits")):
        for L in (2048, 4096, 16384):
            shape = (L, L) if fmt == FMT_U8 else (L, L // 32)
            d = torch.empty(shape, dtype=torch.uint8 if fmt == FMT_U8 else torch.int32, device="cuda")
            pgg.pgg_init_lattice(d, fmt, L, 0.5, 1)
            pgg.pgg_sweep(d, fmt, L, 3.8, 0.5, 1, pgg.ORDER_IID, 0, 50)
            cells = []
            for variant in (pgg.VARIANT_V0, pgg.VARIANT_AUTO):
                pgg.pgg_set_variant(variant)
                c = d.clone()
                cells.append(timed(lambda: pgg.pgg_sweep(c, fmt, L, 3.8, 0.5, 1, pgg.ORDER_IID, 50, n_mcs)))
            pgg.pgg_set_variant(pgg.VARIANT_AUTO)
            for S in (1, 2, 4, 8):
                n_rows = L // S
                sb = SlabBuffer(fmt, L, 0, n_rows, d.device)
                sb.rows().copy_(scatter(d, 0, n_rows))
                w = wire(sb.ptr, n_rows, sb.ptr, n_rows, sb.ptr, n_rows, fmt, L)
                epoch = [0]

                def run():
                    pgg_slab_sweep(sb.ptr, fmt, L, 0, n_rows, 3.8, 0.5, 1, pgg.ORDER_IID, 50, 0, 16 * n_mcs, w["d_up_halo"],
                                   w["d_dn_halo"], w["d_flags"], w["d_up_flag"], w["d_dn_flag"], epoch[0], None)
                    epoch[0] += 16 * n_mcs

                cells.append(timed(run))
                sb.free()
            print(f"| {name} | {L} | " + " | ".join(f"{x:.1f}" for x in cells) + " |", flush=True)


def _run_sharded(args) -> None:
    """One process per GPU (torchrun): ONE lattice of size L in row slabs, ``--mcs`` MCS from a Bernoulli(0.5) start;
    rank 0 prints one JSON line (updates/s of the whole lattice, device time as the max over ranks).  ``--check``
    also runs the unsharded pgg_sweep on every rank and compares its rows and the count trace with the slabs'."""
    import json
    import os

    import torch
    import torch.distributed as dist

    import paper_1704_08098_b200 as pgg

    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", 0)))
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29531")
        dist.init_process_group("nccl" if world > 1 else "gloo", rank=rank, world_size=world)
    fmt = FMT_BITS if args.fmt == "bits" else FMT_U8
    L, n, r, K, seed = args.L, args.mcs, args.r, 0.5, args.seed
    full = torch.empty((L, L) if fmt == FMT_U8 else (L, L // 32), dtype=torch.uint8 if fmt == FMT_U8 else torch.int32,
                       device="cuda")
    pgg.pgg_init_lattice(full, fmt, L, 0.5, seed)   # every rank makes the same seeded start; it keeps only its slab
    count0 = torch.zeros(1, dtype=torch.int64, device="cuda")
    pgg.pgg_density(full, fmt, L, count0)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    dist.barrier()
    e0.record()
    mine, deltas = run_distributed(full, fmt, L, r, K, seed, pgg.ORDER_IID, 0, n)
    e1.record()
    torch.cuda.synchronize()
    ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device="cuda" if world > 1 else "cpu")
    dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    counts = count0 + torch.cumsum(deltas, 0)
    ok = None
    if args.check:
        cnt = torch.zeros(n, dtype=torch.int64, device="cuda")
        pgg.pgg_sweep(full, fmt, L, r, K, seed, pgg.ORDER_IID, 0, n, cnt)
        torch.cuda.synchronize()
        row0, n_rows = slab_rows(L, world, rank, pgg_slab_step_rows(fmt, L))
        good = torch.tensor([int(torch.equal(mine, full[row0:row0 + n_rows]) and torch.equal(counts, cnt))],
                            device="cuda" if world > 1 else "cpu")
        dist.all_reduce(good, op=dist.ReduceOp.MIN)
        ok = bool(good.item())
    if rank == 0:
        print(json.dumps({"metric": "elementary strategy updates/sec, one lattice in row slabs", "value": L * L * n / (ms.item() * 1e-3),
                          "unit": "updates/s", "n_gpus": world, "L": L, "fmt": args.fmt, "mcs": n, "ms": ms.item(),
                          "us_per_phase": ms.item() * 1e3 / (16 * n), "scaling": "strong", "final_rho_C": counts[-1].item() / L**2,
                          "equals_unsharded_pgg_sweep": ok, "note": "includes slab set-up, the handle exchange and the final all-reduce"}))
    dist.barrier()
    dist.destroy_process_group()
    if ok is False:
        raise SystemExit("slabs differ from the unsharded sweep")


def main(argv=None) -> None:
    import argparse
    ap = argparse.ArgumentParser(description="row slabs of one lattice (DESIGN.md section 10): with no arguments the timing "
                                 "table of the slab kernel on one device; --sharded under torchrun: one lattice over all ranks")
    ap.add_argument("--sharded", action="store_true")
    ap.add_argument("--L", type=int, default=16384)
    ap.add_argument("--fmt", choices=("bits", "u8"), default="bits")
    ap.add_argument("--mcs", type=int, default=100)
    ap.add_argument("--r", type=float, default=3.8)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--check", action="store_true")
    args = ap.parse_args(argv)
    if args.sharded:
        _run_sharded(args)
    else:
        _time_table()


if __name__ == "__main__":
    main()

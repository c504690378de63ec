"""Host logic of the row-slab path (paper_1704_08098_b200/slab.py) on CPU: the row partition, scatter / gather
with periodic halo rows, the neighbour wiring, and -- with gloo, world_size 3 -- the handle exchange that
``run_distributed`` does before its first phase.  No kernel runs here."""
import json
import os
from pathlib import Path

import numpy as np
import pytest

torch = pytest.importorskip("torch")
from paper_1704_08098_b200 import FMT_BITS, FMT_U8, slab  # noqa: E402


@pytest.mark.parametrize("L,world", [(64, 1), (64, 2), (64, 3), (96, 5), (16384, 8), (400, 7), (8, 2)])
def test_slab_rows_partition_the_lattice(L, world):
    rows = [slab.slab_rows(L, world, q) for q in range(world)]
    assert rows[0][0] == 0 and sum(n for _, n in rows) == L
    for (r0, n), (r1, _) in zip(rows, rows[1:]):
        assert r0 + n == r1
    assert all(r0 % 4 == 0 and n % 4 == 0 and n >= 4 for r0, n in rows)
    assert max(n for _, n in rows) - min(n for _, n in rows) <= 4
    with pytest.raises(ValueError):
        slab.slab_rows(L, L // 4 + 1, 0)


def test_slab_rows_with_the_fast_kernels_alignment():
    """align = 4 R rows (pgg_slab_step_rows): every slab a whole number of LEAN steps; too few groups -> align 4."""
    rows = [slab.slab_rows(1024, 3, q, 64) for q in range(3)]
    assert rows == [(0, 384), (384, 320), (704, 320)]
    rows = [slab.slab_rows(16384, 3, q, 8) for q in range(3)]
    assert sum(n for _, n in rows) == 16384 and all(r0 % 8 == 0 and n % 8 == 0 for r0, n in rows)
    assert [slab.slab_rows(1024, 32, q, 64)[1] for q in range(32)] == [32] * 32       # 16 groups < 32 ranks: align 4
    assert slab.slab_rows(96, 5, 0, 64) == slab.slab_rows(96, 5, 0)                    # L % align != 0: align 4


def test_scatter_has_periodic_halos_and_gather_inverts():
    L, world = 32, 3
    full = torch.arange(L * L, dtype=torch.int64).reshape(L, L)
    slabs = []
    for q in range(world):
        row0, n = slab.slab_rows(L, world, q)
        s = slab.scatter(full, row0, n)
        assert s.shape == (n + 6, L)
        want = np.take(full.numpy(), np.arange(row0 - 3, row0 + n + 3), axis=0, mode="wrap")
        assert np.array_equal(s.numpy(), want)
        slabs.append(s)
    assert torch.equal(slab.gather(slabs), full)


@pytest.mark.parametrize("fmt", [FMT_U8, FMT_BITS])
def test_wiring_points_at_the_neighbours_halo_rows_and_flags(fmt):
    """Model the three allocations as byte ranges and check where a slab's pushes and posts land."""
    L, world = 64, 3
    rb = slab.row_bytes(fmt, L)
    rows = [slab.slab_rows(L, world, q) for q in range(world)]
    base = [1 << 20, 5 << 20, 9 << 20]
    for q in range(world):
        up, dn = slab.neighbours(world, q)
        w = slab.wire(base[q], rows[q][1], base[up], rows[up][1], base[dn], rows[dn][1], fmt, L)
        # the upper neighbour's bottom halo = its buffer rows n_up + 3 .. n_up + 5; the lower one's top halo = rows 0..2
        assert w["d_up_halo"] == base[up] + (rows[up][1] + 3) * rb
        assert w["d_dn_halo"] == base[dn]
        flag = lambda p, n: p + (rb * (n + 6) + 255) // 256 * 256   # noqa: E731
        assert w["d_flags"] == flag(base[q], rows[q][1])
        assert w["d_up_flag"] == flag(base[up], rows[up][1]) + 8     # its flags[2]: "my lower neighbour has completed"
        assert w["d_dn_flag"] == flag(base[dn], rows[dn][1]) + 4     # its flags[1]: "my upper neighbour has completed"
        assert w["d_flags"] % 256 == 0
    assert slab.neighbours(1, 0) == (0, 0) and slab.neighbours(2, 0) == (1, 1) and slab.neighbours(4, 0) == (3, 1)


def test_phase_chunks_cover_the_run():
    got = list(slab.phase_chunks(10, 9000))
    assert got == [(10, 4096), (4106, 4096), (8202, 808)]
    assert list(slab.phase_chunks(0, 0)) == []


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    L = 64
    row0, n = slab.slab_rows(L, world, rank)
    infos, r, w = slab.exchange((bytes([rank]) * 64, rank, n))   # (handle, device, rows) as run_distributed sends them
    up, dn = slab.neighbours(w, r)
    dist.barrier()
    dist.destroy_process_group()
    Path(out, f"r{rank}.json").write_text(json.dumps({
        "rank": r, "world": w, "up": [infos[up][0][0], infos[up][1], infos[up][2]],
        "dn": [infos[dn][0][0], infos[dn][1], infos[dn][2]]}))


def test_handle_exchange_world3_gloo(tmp_path):
    import torch.multiprocessing as mp
    world = 3
    port = 33500 + os.getpid() % 2000
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    for rank in range(world):
        d = json.loads((tmp_path / f"r{rank}.json").read_text())
        up, dn = (rank - 1) % world, (rank + 1) % world
        assert d["rank"] == rank and d["world"] == world
        assert d["up"] == [up, up, slab.slab_rows(64, world, up)[1]]
        assert d["dn"] == [dn, dn, slab.slab_rows(64, world, dn)[1]]

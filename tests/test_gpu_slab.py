"""Row slabs of one lattice (``pgg_slab_sweep``, include/pgg.h) against the
oracle's UNSHARDED sweep, bit for bit (``-m gpu``).

One GPU is all there is here, so the S slabs of a lattice live on one device and are driven phase by phase on
one stream (paper_1704_08098_b200.slab.LocalSlabs): launch order = dependency order, no kernel ever waits
for a later one.  What the cases pin: the global site index in the Philox counter (any split gives the
unsharded result), the fused halo push (halo rows equal the neighbour's own rows after every run), the flag
protocol (a run with flags equals a run without; the epoch numbers advance), the per-slab flip counts, and
the same through an IPC handle opened by a second process on the same GPU.  Integer work: exact equality."""
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

import oracle as orc
import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1704_08098_b200 as pgg  # noqa: E402
from paper_1704_08098_b200 import slab  # noqa: E402

ROOT = Path(__file__).resolve().parents[1]
K = wl.K_DEFAULT
FMTS = [pgg.FMT_U8, pgg.FMT_BITS]


@pytest.fixture(scope="module", autouse=True)
def _gpu():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    pgg.lib()


def to_device(lat, fmt):
    lat = np.ascontiguousarray(lat, dtype=np.uint8)
    if fmt == pgg.FMT_U8:
        return torch.from_numpy(lat).cuda()
    L = lat.shape[-1]
    bits = lat.reshape(lat.shape[:-1] + (L // 32, 32)).astype(np.uint32)
    words = (bits << np.arange(32, dtype=np.uint32)).sum(axis=-1, dtype=np.uint64).astype(np.uint32)
    return torch.from_numpy(words.view(np.int32)).cuda()


def to_host(d_lat, fmt, L):
    a = d_lat.cpu().numpy()
    if fmt == pgg.FMT_U8:
        return a
    words = a.view(np.uint32)
    bits = (words[..., None] >> np.arange(32, dtype=np.uint32)) & 1
    return bits.reshape(words.shape[:-1] + (L,)).astype(np.uint8)


def run_slabs(lat0, fmt, S, r, seed, order, t_begin, n_mcs, use_flags, align=None):
    L = lat0.shape[0]
    ls = slab.LocalSlabs(to_device(lat0, fmt), fmt, L, S, use_flags=use_flags, align=align)
    try:
        deltas = ls.sweep(r, K, seed, order, t_begin, n_mcs)
        torch.cuda.synchronize()
        assert ls.halos_consistent(), "a halo row differs from the own row it mirrors"
        counts = int(lat0.sum()) + np.cumsum(deltas.cpu().numpy())
        flags = [sb.bytes[sb.flag_off:sb.flag_off + 12].view(torch.int32).cpu().numpy().tolist() for sb in ls.slabs]
        return to_host(ls.lattice(), fmt, L), counts.astype(np.uint64), flags
    finally:
        ls.free()


@pytest.mark.parametrize("fmt", FMTS)
@pytest.mark.parametrize("S", [1, 2, 3, 4, 16])
def test_slabs_equal_the_unsharded_oracle(fmt, S):
    L, n_mcs, seed, r = 64, 12, 21, 3.9
    lat0 = wl.random_lattice(L, 0.5, 3)
    ref = lat0.copy()
    ref_counts, _ = orc.sweep(ref, r, K, seed, orc.ORDER_IID, 5, n_mcs)
    got, counts, flags = run_slabs(lat0, fmt, S, r, seed, pgg.ORDER_IID, 5, n_mcs, use_flags=True)
    assert np.array_equal(got, ref), f"{int((got != ref).sum())} sites differ"
    assert np.array_equal(counts, ref_counts)
    # every slab has been told by both neighbours that all 16 n_mcs phases are complete; the CTA counter is back at 0
    assert flags == [[0, 16 * n_mcs, 16 * n_mcs]] * S


@pytest.mark.parametrize("fmt", FMTS)
def test_uneven_split_perm_order_structured_state_no_flags(fmt):
    """L = 96: 24 row groups over 5 slabs (20, 20, 20, 20, 16 rows); PERM order; blobs; caller-ordered phases."""
    L, n_mcs, seed, r = 96, 8, 2**40 + 9, 4.2
    lat0 = wl.blobs_lattice(L, 4)
    ref = lat0.copy()
    ref_counts, _ = orc.sweep(ref, r, K, seed, orc.ORDER_PERM, 0, n_mcs)
    got, counts, flags = run_slabs(lat0, fmt, 5, r, seed, pgg.ORDER_PERM, 0, n_mcs, use_flags=False)
    assert np.array_equal(got, ref) and np.array_equal(counts, ref_counts)
    assert flags == [[0, 0, 0]] * 5


@pytest.mark.parametrize("fmt", FMTS)
def test_slabs_equal_pgg_sweep_on_a_larger_lattice(fmt):
    """L = 512 in 4 slabs against the library's own unsharded pgg_sweep (itself oracle-checked elsewhere) and,
    for the first MCS, against the oracle; late t_begin (the counter's MCS word)."""
    L, n_mcs, seed, r, t0 = 512, 3, 77, 3.8, 2**32 - 40
    lat0 = wl.random_lattice(L, 0.5, 8)
    d = to_device(lat0, fmt)
    cnt = torch.zeros(n_mcs, dtype=torch.int64, device="cuda")
    pgg.pgg_sweep(d, fmt, L, r, K, seed, pgg.ORDER_IID, t0, n_mcs, cnt)
    got, counts, _ = run_slabs(lat0, fmt, 4, r, seed, pgg.ORDER_IID, t0, n_mcs, use_flags=True)
    assert np.array_equal(got, to_host(d, fmt, L))
    assert np.array_equal(counts, cnt.cpu().numpy().astype(np.uint64))
    ref = lat0.copy()
    ref_counts, _ = orc.sweep(ref, r, K, seed, orc.ORDER_IID, t0, n_mcs, n_threads=orc.max_threads())
    assert np.array_equal(got, ref) and np.array_equal(counts, ref_counts)


@pytest.mark.parametrize("fmt", FMTS)
@pytest.mark.parametrize("L,S", [(1024, 1), (1024, 2), (1024, 3), (1024, 4), (1024, 16), (2048, 8), (4096, 4)])
def test_lean_slabs_equal_the_unsharded_oracle(fmt, L, S):
    """Slabs of whole LEAN steps run LEAN's ring kernel on the slab's buffer (rows never wrap, the virtual lattice
    base, the steps of the whole lattice, the push from the level-2 write; uint8 rows are packed to bits on arrival
    as in the unsharded kernel): same bar, against the oracle."""
    n_mcs, seed, r = 3, 31, 3.8
    lat0 = wl.random_lattice(L, 0.5, 17)
    ref = lat0.copy()
    ref_counts, _ = orc.sweep(ref, r, K, seed, orc.ORDER_IID, 7, n_mcs, n_threads=orc.max_threads())
    got, counts, flags = run_slabs(lat0, fmt, S, r, seed, pgg.ORDER_IID, 7, n_mcs, use_flags=True)
    assert pgg.pgg_get_variant_used() == pgg.VARIANT_LEAN
    assert np.array_equal(got, ref), f"{int((got != ref).sum())} sites differ"
    assert np.array_equal(counts, ref_counts)
    assert flags == [[0, 16 * n_mcs, 16 * n_mcs]] * S


def test_lean_slab_structured_state_and_ragged_split_falls_back():
    """Blobs and stripes (long quiet stretches, busy boundaries) on LEAN slabs; a split into slabs that are not whole
    LEAN steps (align = 4; 3 slabs of L = 1024: 344, 340, 340 rows) takes the general word kernel and gives the same
    lattice.  (By default the split follows pgg_slab_step_rows: 384, 320, 320 rows, all on LEAN.)"""
    L, n_mcs, seed, r = 1024, 2, 5, 4.4
    for lat0 in (wl.blobs_lattice(L, 9), wl.stripes_lattice(L, 5)):
        ref = lat0.copy()
        ref_counts, _ = orc.sweep(ref, r, K, seed, orc.ORDER_PERM, 0, n_mcs, n_threads=orc.max_threads())
        for S, align, want in ((4, None, pgg.VARIANT_LEAN), (3, 4, pgg.VARIANT_V0)):
            got, counts, _ = run_slabs(lat0, pgg.FMT_BITS, S, r, seed, pgg.ORDER_PERM, 0, n_mcs, use_flags=True, align=align)
            assert pgg.pgg_get_variant_used() == want
            assert np.array_equal(got, ref) and np.array_equal(counts, ref_counts)


@pytest.mark.parametrize("case", range(10))
def test_random_splits(case):
    """Seeded random (L, layout, number of slabs, split granularity, order, start MCS, state): whatever the split and
    whichever kernel each slab gets, the slabs together are the unsharded oracle."""
    rng = np.random.default_rng(1000 + case)
    L = int(rng.choice([32, 64, 128, 160, 256, 1024, 2048]))
    fmt = int(rng.choice(FMTS)) if L % 32 == 0 else pgg.FMT_U8
    S = int(rng.integers(1, min(9, L // 4) + 1))
    align = [None, 4][int(rng.integers(0, 2))]
    order = [pgg.ORDER_IID, pgg.ORDER_PERM][int(rng.integers(0, 2))]
    t0 = int(rng.choice([0, 3, 4095, 99_990, 2**32 - 8]))
    r = float(rng.choice([3.6, 3.8, 4.0, 4.6, 5.5]))
    seed = int(rng.integers(1, 2**63))
    lat0 = wl.random_lattice(L, float(rng.choice([0.1, 0.5, 0.9])), case) if rng.integers(0, 3) else wl.blobs_lattice(L, case)
    n_mcs = 2
    ref = lat0.copy()
    ref_counts, _ = orc.sweep(ref, r, K, seed, order, t0, n_mcs, n_threads=orc.max_threads())
    got, counts, _ = run_slabs(lat0, fmt, S, r, seed, order, t0, n_mcs, use_flags=bool(rng.integers(0, 2)), align=align)
    assert np.array_equal(got, ref), (L, fmt, S, align, order, t0, r)
    assert np.array_equal(counts, ref_counts)


@pytest.mark.parametrize("fmt", FMTS)
@pytest.mark.parametrize("L,S,align", [(64, 3, None), (96, 2, None), (1024, 4, None), (1024, 3, 4), (2048, 2, None)])
def test_prisoners_dilemma_on_slabs(fmt, L, S, align):
    """The second game (pgg_pd_sweep) on row slabs: general kernels (L = 64, 96, the ragged split of
    1024) and LEAN on the slab (1024, 2048), against the unsharded prisoner's-dilemma oracle."""
    if fmt == pgg.FMT_BITS and L % 32:
        pytest.skip("bit rows need L % 32 == 0")
    pay, n_mcs, seed = (1.0, 0.0, 1.3, 0.1), 4, 77
    lat0 = wl.random_lattice(L, 0.5, 23)
    ref = lat0.copy()
    ref_counts = orc.pd_sweep(ref, *pay, K, seed, orc.ORDER_IID, 3, n_mcs)
    got, counts, _ = run_slabs(lat0, fmt, S, pay, seed, pgg.ORDER_IID, 3, n_mcs, use_flags=True, align=align)
    assert pgg.pgg_get_variant_used() == (pgg.VARIANT_LEAN if L >= 1024 and align is None else pgg.VARIANT_V0)
    assert np.array_equal(got, ref), f"{int((got != ref).sum())} sites differ"
    assert np.array_equal(counts, ref_counts)


def test_one_call_for_many_phases_on_a_single_slab():
    """A single slab is its own neighbour both ways, so ONE call may run all phases of several MCS (the way
    run_distributed calls it): mid-MCS start, flags on, against the oracle."""
    L, seed, r = 64, 5, 3.8
    lat0 = wl.random_lattice(L, 0.5, 11)
    ref = lat0.copy()
    ref_counts, _ = orc.sweep(ref, r, K, seed, orc.ORDER_IID, 0, 6)
    d = to_device(lat0, pgg.FMT_U8)
    ls = slab.LocalSlabs(d, pgg.FMT_U8, L, 1)
    try:
        sb, w = ls.slabs[0], ls.wiring[0]
        deltas = torch.zeros(6, dtype=torch.int64, device="cuda")
        # phases 0 .. 39 (MCS 0, 1 and half of 2), then the remaining 56: the second call starts at phase 8 of MCS 2
        pgg.pgg_slab_sweep(sb.ptr, pgg.FMT_U8, L, 0, L, r, K, seed, pgg.ORDER_IID, 0, 0, 40, w["d_up_halo"], w["d_dn_halo"],
                           w["d_flags"], w["d_up_flag"], w["d_dn_flag"], 0, deltas)
        pgg.pgg_slab_sweep(sb.ptr, pgg.FMT_U8, L, 0, L, r, K, seed, pgg.ORDER_IID, 2, 8, 56, w["d_up_halo"], w["d_dn_halo"],
                           w["d_flags"], w["d_up_flag"], w["d_dn_flag"], 40, deltas[2:])
        torch.cuda.synchronize()
        assert ls.halos_consistent()
        assert np.array_equal(ls.lattice().cpu().numpy(), ref)
        counts = int(lat0.sum()) + np.cumsum(deltas.cpu().numpy())
        assert np.array_equal(counts.astype(np.uint64), ref_counts)
    finally:
        ls.free()


def test_argument_validation():
    L = 64
    d = torch.zeros(pgg.pgg_slab_bytes(pgg.FMT_U8, L, 16), dtype=torch.uint8, device="cuda")
    ok = dict(d_up_halo=d, d_dn_halo=d)

    def code(**kw):
        a = dict(d_slab=d, fmt=pgg.FMT_U8, L=L, row0=0, n_rows=16, r=3.8, K=K, seed=1, order_mode=pgg.ORDER_IID,
                 t_begin=0, k_begin=0, n_phases=1, **ok)
        a.update(kw)
        try:
            pgg.pgg_slab_sweep(**a)
        except pgg.PggError as e:
            return e.code
        return pgg.OK

    assert code() == pgg.OK
    assert code(n_phases=0) == pgg.OK
    assert code(row0=2) == pgg.ERR_BAD_PARAM and code(n_rows=10) == pgg.ERR_BAD_PARAM
    assert code(row0=56, n_rows=16) == pgg.ERR_BAD_PARAM and code(n_rows=0) == pgg.ERR_BAD_PARAM
    assert code(k_begin=16) == pgg.ERR_BAD_PARAM and code(K=0.0) == pgg.ERR_BAD_PARAM
    assert code(n_phases=16 * pgg.SLAB_MAX_MCS + 1) == pgg.ERR_BAD_PARAM
    assert code(order_mode=pgg.ORDER_DTILE) == pgg.ERR_UNSUPPORTED
    assert code(d_up_halo=None) == pgg.ERR_NULL and code(d_slab=None) == pgg.ERR_NULL
    assert code(d_flags=d) == pgg.ERR_NULL           # flags without the neighbours' flag addresses
    assert code(L=66) == pgg.ERR_BAD_L
    torch.cuda.synchronize()


_CHILD = r"""
import sys, torch
import paper_1704_08098_b200 as pgg
handle = bytes.fromhex(sys.argv[1]); L = int(sys.argv[2])
torch.cuda.init()
p = pgg.pgg_slab_ipc_open(handle, -1)
pgg.pgg_init_lattice(p, pgg.FMT_U8, L, 0.5, 4242)   # the other process's allocation, written from here
torch.cuda.synchronize()
pgg.pgg_slab_ipc_close(p)
print("child ok")
"""


def test_ipc_handle_opens_in_a_second_process():
    """pgg_slab_alloc -> pgg_slab_ipc_export here, pgg_slab_ipc_open in a child process on the same GPU, which
    writes a seeded lattice into the allocation; this process then finds exactly that lattice in it.  (The two
    processes never run kernels that wait for each other.)"""
    L = 64
    p = pgg.pgg_slab_alloc(L * L)
    try:
        handle = pgg.pgg_slab_ipc_export(p)
        assert len(handle) == pgg.SLAB_IPC_HANDLE_BYTES
        out = subprocess.run([sys.executable, "-c", _CHILD, handle.hex(), str(L)], capture_output=True, text=True,
                             timeout=300, cwd=ROOT)
        assert out.returncode == 0 and "child ok" in out.stdout, out.stderr[-2000:]
        mine = torch.empty((L, L), dtype=torch.uint8, device="cuda")
        pgg.pgg_init_lattice(mine, pgg.FMT_U8, L, 0.5, 4242)
        theirs = slab.as_byte_tensor(p, L * L, mine.device).view(L, L)
        torch.cuda.synchronize()
        assert torch.equal(mine, theirs)
        assert np.array_equal(mine.cpu().numpy(), orc.init(L, 0.5, 4242))
    finally:
        pgg.pgg_slab_free(p)


def test_sharded_driver_world_size_one():
    """The one-process-per-GPU driver (slab.run_distributed behind ``python -m paper_1704_08098_b200.slab --sharded``)
    with the one rank there is: its slab is the whole lattice and its own neighbour, so the handle exchange, the
    wiring, the chunked calls with running epochs and the final all-reduce all run -- only the IPC mapping does not
    (test_ipc_handle_opens_in_a_second_process).  --check compares with the unsharded pgg_sweep; the rho_C it prints
    is compared with the oracle here."""
    import json
    L, n = 1024, 5
    out = subprocess.run([sys.executable, "-m", "paper_1704_08098_b200.slab", "--sharded", "--L", str(L), "--mcs", str(n),
                          "--fmt", "bits", "--seed", "3", "--check"], capture_output=True, text=True, timeout=600, cwd=ROOT,
                         env={**__import__("os").environ, "MASTER_PORT": str(36500 + __import__("os").getpid() % 2000)})
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads([ln for ln in out.stdout.splitlines() if ln.startswith("{")][-1])
    assert d["equals_unsharded_pgg_sweep"] is True and d["n_gpus"] == 1 and d["value"] > 0
    ref = orc.init(L, 0.5, 3)
    ref_counts, _ = orc.sweep(ref, 3.8, K, 3, orc.ORDER_IID, 0, n, n_threads=orc.max_threads())
    assert d["final_rho_C"] == int(ref_counts[-1]) / L**2


def test_sharded_driver_long_run_crosses_the_call_limit():
    """4200 MCS = 67 200 phases through run_distributed at world size 1: two calls (4096 + 104 MCS, PGG_SLAB_MAX_MCS),
    epochs running on from the first into the second, against the unsharded pgg_sweep (--check; that path's own
    run across the 4096-MCS boundary is checked against the oracle in test_gpu_parity.py)."""
    import json
    out = subprocess.run([sys.executable, "-m", "paper_1704_08098_b200.slab", "--sharded", "--L", "1024", "--mcs", "4200",
                          "--fmt", "bits", "--seed", "9", "--r", "3.9", "--check"], capture_output=True, text=True, timeout=900,
                         cwd=ROOT, env={**__import__("os").environ, "MASTER_PORT": str(38500 + __import__("os").getpid() % 2000)})
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads([ln for ln in out.stdout.splitlines() if ln.startswith("{")][-1])
    assert d["equals_unsharded_pgg_sweep"] is True and d["mcs"] == 4200

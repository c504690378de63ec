"""GPU <-> oracle parity for the paper's double-tiling schedule (PGG_ORDER_DTILE),
bit for bit through the C ABI (``-m gpu``): every lattice site and every cooperator count."""
import hashlib

import numpy as np
import pytest

import oracle as orc
import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1704_08098_b200 as pgg  # noqa: E402
from test_gpu_parity import FMTS, K, assert_same, empty_lattice, gpu_sweep, to_device, to_host  # noqa: E402


@pytest.fixture(scope="module", autouse=True)
def _gpu():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    pgg.lib()
    yield


def _skip_bits(fmt, L):
    if fmt == pgg.FMT_BITS and L % 32:
        pytest.skip("bits layout needs L % 32 == 0")


@pytest.mark.parametrize("fmt", FMTS)
@pytest.mark.parametrize("L,r,seed,n_mcs", [(8, 4.0, 3, 40), (16, 3.9, 99, 30), (32, 4.0, 5, 50), (64, 4.0, 1, 200),
                                            (96, 3.8, 2**40 + 7, 40), (200, 5.4, 12, 30), (416, 3.76, 8, 25),
                                            (1024, 3.98, 21, 12)])
def test_dtile_sweep_parity(fmt, L, r, seed, n_mcs):
    """Small lattices (L = 8: every patch wraps onto itself), ragged grids (L/8 not a multiple of
    the CTA size), word-straddling patches in the bit-packed layout, 64-bit seeds."""
    _skip_bits(fmt, L)
    lat0 = orc.init(L, 0.5, seed)
    ref = lat0.copy()
    ref_counts, _ = orc.sweep(ref, r, K, seed, order_mode=orc.ORDER_DTILE, t_begin=7, n_mcs=n_mcs,
                              n_threads=4 if L >= 416 else 1)
    got, counts = gpu_sweep(lat0, fmt, r, seed, pgg.ORDER_DTILE, 7, n_mcs)
    assert_same(got, ref, "lattice")
    assert_same(counts, ref_counts, "counts")
    assert pgg.pgg_get_variant_used() == 10
    assert not np.array_equal(ref, lat0)


@pytest.mark.parametrize("fmt", FMTS)
def test_dtile_config1_trace_and_snapshots(fmt):
    """Config 1 (L=64, r=4, 1000 MCS) under the paper's schedule: lattice every 100 MCS + all counts."""
    cfg = wl.config1()
    L, seed, r = cfg.L, cfg.seeds[0], cfg.rs[0]
    lat = orc.init(L, 0.5, seed)
    ref_counts, snaps = orc.sweep(lat, r, K, seed, order_mode=orc.ORDER_DTILE, n_mcs=1000, snap_every=100)
    d = to_device(orc.init(L, 0.5, seed), fmt)
    cnt = torch.zeros(100, dtype=torch.int64, device="cuda")
    for s in range(10):
        pgg.pgg_sweep(d, fmt, L, r, K, seed, pgg.ORDER_DTILE, 100 * s, 100, cnt)
        torch.cuda.synchronize()
        assert_same(to_host(d, fmt, L), snaps[s], f"snapshot {s}")
        assert_same(cnt.cpu().numpy().astype(np.uint64), ref_counts[100 * s:100 * s + 100], f"counts {s}")


@pytest.mark.parametrize("fmt", FMTS)
def test_dtile_structured_and_absorbing_states(fmt):
    L = 128
    for name, lat0 in (("blobs", wl.blobs_lattice(L, 4)), ("stripes", wl.stripes_lattice(L, 5)),
                       ("checker", wl.checkerboard_lattice(L)), ("sparse", wl.random_lattice(L, 0.02, 9)),
                       ("dense", wl.random_lattice(L, 0.98, 9)), ("allD", np.zeros((L, L), np.uint8)),
                       ("allC", np.ones((L, L), np.uint8))):
        ref = lat0.copy()
        ref_counts, _ = orc.sweep(ref, 3.9, K, 31, order_mode=orc.ORDER_DTILE, n_mcs=20)
        got, counts = gpu_sweep(lat0, fmt, 3.9, 31, pgg.ORDER_DTILE, 0, 20)
        assert_same(got, ref, name)
        assert_same(counts, ref_counts, name + " counts")


@pytest.mark.parametrize("fmt", FMTS)
def test_dtile_ensemble_equals_solo_and_oracle(fmt):
    """a9 under the paper's schedule: B lattices in one grid, each with its own r and seed."""
    L, B, n = 64, 5, 60
    rs = [3.7 + 0.1 * k for k in range(B)]
    seeds = [1000 + k for k in range(B)]
    d = empty_lattice(fmt, L, B)
    cnt = torch.zeros((B, n), dtype=torch.int64, device="cuda")
    pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_DTILE, 0.5, 0, n, cnt)
    torch.cuda.synchronize()
    got = to_host(d, fmt, L)
    for k in range(B):
        ref = orc.init(L, 0.5, seeds[k])
        ref_counts, _ = orc.sweep(ref, rs[k], K, seeds[k], order_mode=orc.ORDER_DTILE, n_mcs=n)
        assert_same(got[k], ref, f"member {k}")
        assert_same(cnt[k].cpu().numpy().astype(np.uint64), ref_counts, f"member {k} counts")


def test_dtile_clamped_tables_and_late_time():
    """K = 1e-3 (thresholds clamp to 0 / 2^32-1), r = 25, t_begin near 2^32, NULL counts."""
    L = 48
    for r, k_noise, t0 in ((3.8, 1e-3, 0), (25.0, 0.5, 2**32 - 6)):
        lat0 = orc.init(L, 0.5, 77)
        ref = lat0.copy()
        lib_counts, _ = orc.sweep(ref, r, k_noise, 77, order_mode=orc.ORDER_DTILE, t_begin=t0, n_mcs=5)
        d = to_device(lat0, pgg.FMT_U8)
        pgg.pgg_sweep(d, pgg.FMT_U8, L, r, k_noise, 77, pgg.ORDER_DTILE, t0, 5, None)
        torch.cuda.synchronize()
        assert_same(to_host(d, pgg.FMT_U8, L), ref, f"r={r}")


def test_dtile_rejects_L_not_divisible_by_8():
    d = empty_lattice(pgg.FMT_U8, 12)
    with pytest.raises(Exception):
        pgg.pgg_sweep(d, pgg.FMT_U8, 12, 4.0, K, 1, pgg.ORDER_DTILE, 0, 1, None)


@pytest.mark.parametrize("fmt", FMTS)
def test_dtile_config5_size_two_mcs(fmt):
    """L = 16384 in the launch configuration bench.py --order dtile times: 2 MCS against a live
    oracle run (all host threads), whole lattice compared by hash + counts."""
    L, seed, r = 16384, 1, 3.8
    ref = orc.init(L, 0.5, seed)
    ref_counts, _ = orc.sweep(ref, r, K, seed, order_mode=orc.ORDER_DTILE, n_mcs=2, n_threads=orc.max_threads())
    d = empty_lattice(fmt, L)
    pgg.pgg_init_lattice(d, fmt, L, 0.5, seed)
    cnt = torch.zeros(2, dtype=torch.int64, device="cuda")
    pgg.pgg_sweep(d, fmt, L, r, K, seed, pgg.ORDER_DTILE, 0, 2, cnt)
    torch.cuda.synchronize()
    assert_same(cnt.cpu().numpy().astype(np.uint64), ref_counts, "counts")
    got = to_host(d, fmt, L)
    assert hashlib.sha256(got.tobytes()).hexdigest() == hashlib.sha256(ref.tobytes()).hexdigest()

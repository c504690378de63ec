"""``pgg_sweep_static`` -- the sweep for callers that may not allocate -- against ``pgg_sweep`` (``-m gpu``).

The entry point keeps the temporaries of a sweep (seed, acceptance table, initial count, class order) in
one file-scope device array instead of the stream-ordered pool (include/pgg.h).  Every call on a device
shares that array and finds the previous call's contents in it, so each case makes TWO calls in a row,
with different r and seed, WITHOUT a synchronisation between them, and compares both with the existing
path.  Integer work: the bar is exact equality of every site and every count (as in test_gpu_parity.py).

The file sorts last on purpose (the suite runs with ``pytest -x``); it must pass alone in a fresh
process and after the other tests, so it sets the variant it wants and restores AUTO."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1704_08098_b200 as pgg  # noqa: E402

K = wl.K_DEFAULT


@pytest.fixture(autouse=True)
def _gpu():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    pgg.lib()
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)
    yield
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)


def to_device(lat, fmt):
    lat = np.ascontiguousarray(lat, dtype=np.uint8)
    if fmt == pgg.FMT_U8:
        return torch.from_numpy(lat).cuda()
    L = lat.shape[-1]
    bits = lat.reshape(lat.shape[:-1] + (L // 32, 32)).astype(np.uint32)
    words = (bits << np.arange(32, dtype=np.uint32)).sum(axis=-1, dtype=np.uint64).astype(np.uint32)
    return torch.from_numpy(words.view(np.int32)).cuda()


def run_pair(sweep, fmt, L, n1, n2, with_counts=True):
    """Two calls in a row on the current stream, no synchronisation in between: lattice A (r = 3.8, seed 11,
    MCS 0 .. n1-1, IID order), then lattice B (r = 4.3, seed 12, MCS 7 .. 7+n2-1, PERM order)."""
    a = to_device(wl.random_lattice(L, 0.5, 5), fmt)
    b = to_device(wl.blobs_lattice(L, 6), fmt)
    ca = torch.full((n1,), -1, dtype=torch.int64, device="cuda") if with_counts else None
    cb = torch.full((n2,), -1, dtype=torch.int64, device="cuda") if with_counts else None
    sweep(a, fmt, L, 3.8, K, 11, pgg.ORDER_IID, 0, n1, ca)
    used_a = pgg.lib().pgg_get_variant_used()
    sweep(b, fmt, L, 4.3, K, 12, pgg.ORDER_PERM, 7, n2, cb)
    torch.cuda.synchronize()
    out = [a.cpu().numpy(), b.cpu().numpy()]
    if with_counts:
        out += [ca.cpu().numpy(), cb.cpu().numpy()]
    return out, used_a


# (fmt, L, kernel pgg_sweep_static picks, MCS of the two calls)
CASES = [
    (pgg.FMT_U8, 128, pgg.VARIANT_RESIDENT, 12, 9),
    (pgg.FMT_BITS, 128, pgg.VARIANT_RESIDENT, 12, 9),
    (pgg.FMT_U8, 512, pgg.VARIANT_CLUSTER, 10, 6),
    (pgg.FMT_BITS, 1024, pgg.VARIANT_CLUSTER, 6, 5),
    (pgg.FMT_U8, 2048, pgg.VARIANT_RING, 4, 3),
    (pgg.FMT_BITS, 2048, pgg.VARIANT_LEAN, 4, 3),
    (pgg.FMT_U8, 400, pgg.VARIANT_V0, 8, 5),
    (pgg.FMT_BITS, 384, pgg.VARIANT_V0, 8, 5),
]


@pytest.mark.parametrize("fmt,L,kernel,n1,n2", CASES)
def test_static_sweep_equals_sweep_on_two_calls_in_a_row(fmt, L, kernel, n1, n2):
    ref, _ = run_pair(pgg.pgg_sweep, fmt, L, n1, n2)  # (its AUTO choice may differ: PACKED needs a working copy)
    got, used = run_pair(pgg.pgg_sweep_static, fmt, L, n1, n2)
    assert used == kernel, (used, kernel)
    for what, x, y in zip(("lattice A", "lattice B", "counts A", "counts B"), got, ref):
        assert np.array_equal(x, y), f"{what}: {int((x != y).sum())} mismatches"
    assert got[2].min() >= 0 and got[3].min() >= 0  # every count written


def test_static_sweep_without_counts_and_with_a_chosen_variant():
    # d_counts = NULL; pgg_set_variant is honoured for the five kernels the entry point carries
    fmt, L = pgg.FMT_U8, 1024
    for v in (pgg.VARIANT_V0, pgg.VARIANT_RING, pgg.VARIANT_LEAN, pgg.VARIANT_CLUSTER):
        pgg.pgg_set_variant(v)
        ref, _ = run_pair(pgg.pgg_sweep, fmt, L, 3, 2, with_counts=False)
        got, used = run_pair(pgg.pgg_sweep_static, fmt, L, 3, 2, with_counts=False)
        assert used == v
        assert np.array_equal(got[0], ref[0]) and np.array_equal(got[1], ref[1]), f"variant {v}"


def test_static_sweep_continues_a_run_bit_for_bit():
    # the stated way around the limit: (t_begin = a, n = b) then (a + b, c) equals (a, b + c)
    fmt, L = pgg.FMT_BITS, 512
    lat0 = wl.random_lattice(L, 0.5, 21)
    whole, parts = to_device(lat0, fmt), to_device(lat0, fmt)
    pgg.pgg_sweep(whole, fmt, L, 3.8, K, 3, pgg.ORDER_IID, 100, 9)
    pgg.pgg_sweep_static(parts, fmt, L, 3.8, K, 3, pgg.ORDER_IID, 100, 4)
    pgg.pgg_sweep_static(parts, fmt, L, 3.8, K, 3, pgg.ORDER_IID, 104, 5)
    torch.cuda.synchronize()
    assert torch.equal(whole, parts)


def test_static_sweep_rejects_what_it_cannot_hold():
    fmt, L = pgg.FMT_U8, 128
    d = to_device(wl.random_lattice(L, 0.5, 1), fmt)
    before = d.clone()
    with pytest.raises(pgg.PggError) as e:
        pgg.pgg_sweep_static(d, fmt, L, 3.8, K, 1, pgg.ORDER_IID, 0, pgg.STATIC_MAX_MCS + 1)
    assert e.value.code == pgg.ERR_BAD_PARAM and "PGG_STATIC_MAX_MCS" in str(e.value)
    with pytest.raises(pgg.PggError) as e:
        pgg.pgg_sweep_static(d, fmt, L, 3.8, K, 1, pgg.ORDER_DTILE, 0, 1)
    assert e.value.code == pgg.ERR_UNSUPPORTED
    pgg.pgg_set_variant(pgg.VARIANT_BAND)  # not one of the five
    with pytest.raises(pgg.PggError) as e:
        pgg.pgg_sweep_static(d, fmt, L, 3.8, K, 1, pgg.ORDER_IID, 0, 1)
    assert e.value.code == pgg.ERR_UNSUPPORTED
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)
    torch.cuda.synchronize()
    assert torch.equal(d, before)  # a rejected call touches nothing
    pgg.pgg_sweep_static(d, fmt, L, 3.8, K, 1, pgg.ORDER_IID, 0, 0)  # n_mcs == 0: a no-op
    torch.cuda.synchronize()
    assert torch.equal(d, before)


def test_static_sweep_at_the_limit():
    # PGG_STATIC_MAX_MCS MCS in one call fill the whole order array (small lattice: RESIDENT, one launch)
    fmt, L, n = pgg.FMT_BITS, 64, pgg.STATIC_MAX_MCS
    lat0 = wl.random_lattice(L, 0.5, 2)
    x, y = to_device(lat0, fmt), to_device(lat0, fmt)
    cx = torch.zeros(n, dtype=torch.int64, device="cuda")
    cy = torch.zeros(n, dtype=torch.int64, device="cuda")
    pgg.pgg_sweep(x, fmt, L, 3.8, K, 9, pgg.ORDER_IID, 0, n, cx)
    pgg.pgg_sweep_static(y, fmt, L, 3.8, K, 9, pgg.ORDER_IID, 0, n, cy)
    torch.cuda.synchronize()
    assert torch.equal(x, y) and torch.equal(cx, cy)


@pytest.mark.parametrize("fmt,L,kernel", [(f, L, k) for f, L, k, _, _ in CASES])
def test_static_sweep_is_capturable_into_a_cuda_graph(fmt, L, kernel):
    """What the entry point is for: the whole call (memsets, the upload / order / density / phase / finalize kernels,
    cluster and programmatic-dependent launches) is captured into a CUDA graph -- an allocation would fail the
    capture -- and two replays equal two eager pgg_sweep calls bit for bit.  One warm-up call outside the capture
    resolves the scratch address and the function attributes."""
    n = 3
    a = to_device(wl.random_lattice(L, 0.5, 31), fmt)
    b = a.clone()
    ca = torch.zeros(n, dtype=torch.int64, device="cuda")
    cb = torch.zeros(n, dtype=torch.int64, device="cuda")
    for _ in range(2):
        pgg.pgg_sweep(a, fmt, L, 3.8, K, 3, pgg.ORDER_IID, 0, n, ca)
    warm = b.clone()
    pgg.pgg_sweep_static(warm, fmt, L, 3.8, K, 3, pgg.ORDER_IID, 0, 1)
    assert pgg.pgg_get_variant_used() == kernel
    torch.cuda.synchronize()
    graph, side = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            pgg.pgg_sweep_static(b, fmt, L, 3.8, K, 3, pgg.ORDER_IID, 0, n, cb, stream=side)
    graph.replay()
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(a, b) and torch.equal(ca, cb)

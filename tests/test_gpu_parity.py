"""GPU <-> oracle parity, bit for bit, through the C ABI (``-m gpu``).

Every case runs the same seeded input through ``libpgg`` (CUDA, sm_100a) and
through ``oracle/`` (plain C on the CPU) and compares every lattice site and
every cooperator count.  Integer work: the bar is exact equality."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1704_08098_b200 as pgg  # noqa: E402

K = wl.K_DEFAULT
FMTS = [pgg.FMT_U8, pgg.FMT_BITS]
VARIANTS = [pgg.VARIANT_V0, pgg.VARIANT_TILE, pgg.VARIANT_PIPE, pgg.VARIANT_BAND, pgg.VARIANT_RING, pgg.VARIANT_SPLIT, pgg.VARIANT_DYN,
            pgg.VARIANT_RESIDENT, pgg.VARIANT_LEAN, pgg.VARIANT_PACKED]


@pytest.fixture(scope="module", autouse=True)
def _gpu():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    pgg.lib()
    yield
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)


def use_variant(v, fmt, L):
    """Select kernel variant v; skip if it does not support (fmt, L)."""
    if not pgg.pgg_variant_supported(v, fmt, L):
        pytest.skip("this variant does not support this (fmt, L)")
    pgg.pgg_set_variant(v)


# ---------------------------------------------------------------- marshalling helpers
def to_device(lat, fmt):
    """numpy uint8 [.., L, L] -> device tensor in layout fmt (packing is pure layout)."""
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


def empty_lattice(fmt, L, B=None):
    shape = (L, L) if fmt == pgg.FMT_U8 else (L, L // 32)
    if B is not None:
        shape = (B,) + shape
    return torch.empty(shape, dtype=torch.uint8 if fmt == pgg.FMT_U8 else torch.int32, device="cuda")


def gpu_sweep(lat0, fmt, r, seed, order, t_begin, n_mcs, want_counts=True):
    L = lat0.shape[0]
    d = to_device(lat0, fmt)
    cnt = torch.zeros(max(n_mcs, 1), dtype=torch.int64, device="cuda") if want_counts else None
    pgg.pgg_sweep(d, fmt, L, r, K, seed, order, t_begin, n_mcs, cnt)
    torch.cuda.synchronize()
    counts = cnt.cpu().numpy().astype(np.uint64)[:n_mcs] if want_counts else None
    return to_host(d, fmt, L), counts


def assert_same(a, b, what=""):
    if not np.array_equal(a, b):
        bad = np.argwhere(a != b)
        raise AssertionError(f"{what}: {len(bad)} mismatches, first at {bad[:5].tolist()}")


# ---------------------------------------------------------------- K0 init (D4)
@pytest.mark.parametrize("fmt", FMTS)
@pytest.mark.parametrize("L,rho0,seed", [(64, 0.5, 1), (32, 0.0, 3), (32, 1.0, 3), (96, 0.2, 2**40 + 7),
                                         (416, 0.77, 12), (4, 0.5, 9), (20, 0.5, 5), (2048, 0.5, 16)])
def test_init_parity(fmt, L, rho0, seed):
    if fmt == pgg.FMT_BITS and L % 32:
        pytest.skip("bits layout needs L % 32 == 0")
    d = empty_lattice(fmt, L)
    pgg.pgg_init_lattice(d, fmt, L, rho0, seed)
    torch.cuda.synchronize()
    assert_same(to_host(d, fmt, L), orc.init(L, rho0, seed), "init")


# ---------------------------------------------------------------- a1 phase classes (D5)
@pytest.mark.parametrize("order", [pgg.ORDER_IID, pgg.ORDER_PERM])
def test_phase_classes_parity(order):
    for seed in (1, 2**33 + 5):
        for t in (0, 1, 17, 99999, 2**32 - 1):
            got = pgg.pgg_phase_classes(seed, t, order)
            assert got == orc.phase_classes(seed, t, order).tolist(), (seed, t)
            if order == pgg.ORDER_PERM:
                assert sorted(got) == list(range(16))


# ---------------------------------------------------------------- K3 density (Eq. 4)
@pytest.mark.parametrize("fmt", FMTS)
def test_density_parity(fmt):
    for L, p in ((64, 0.5), (416, 0.3), (32, 0.0), (32, 1.0), (1024, 0.9)):
        lat = wl.random_lattice(L, p, seed=L)
        out = torch.full((1,), -1, dtype=torch.int64, device="cuda")
        pgg.pgg_density(to_device(lat, fmt), fmt, L, out)
        torch.cuda.synchronize()
        assert int(out.item()) == orc.count(lat) == int(lat.sum())


@pytest.mark.parametrize("fmt", FMTS)
def test_interface_count(fmt):
    """pgg_count_interface = sites with a nearest neighbour of the other strategy (the sites an
    elementary step needs its draw for, S9); numpy rolls are the plain definition."""
    for L, p in ((64, 0.5), (416, 0.3), (32, 0.0), (1024, 0.05)):
        lat = wl.random_lattice(L, p, seed=3 * L)
        want = 0
        diff = np.zeros_like(lat, dtype=bool)
        for ax, sh in ((0, 1), (0, -1), (1, 1), (1, -1)):
            diff |= np.roll(lat, sh, axis=ax) != lat
        want = int(diff.sum())
        out = torch.full((1,), -1, dtype=torch.int64, device="cuda")
        pgg.pgg_count_interface(to_device(lat, fmt), fmt, L, out)
        torch.cuda.synchronize()
        assert int(out.item()) == want


# ---------------------------------------------------------------- config 1 in full
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("fmt", FMTS)
@pytest.mark.parametrize("order", [pgg.ORDER_IID, pgg.ORDER_PERM])
def test_config1_full_trace_and_snapshots(variant, fmt, order):
    """BASELINE.json configs[0]: L=64, r=4, K=.5, seed 1, 1000 MCS; the lattice every 100 MCS
    and the whole rho_C trace."""
    cfg = wl.config1()
    L, r, seed = cfg.L, cfg.rs[0], cfg.seeds[0]
    use_variant(variant, fmt, L)
    lat = orc.init(L, cfg.rho0, seed)
    ref_counts, ref_snaps = orc.sweep(lat.copy(), r, K, seed, order, 0, cfg.n_mcs, snap_every=cfg.snap_every)
    d = empty_lattice(fmt, L)
    pgg.pgg_init_lattice(d, fmt, L, cfg.rho0, seed)
    counts = []
    for a in range(cfg.n_mcs // cfg.snap_every):
        cnt = torch.zeros(cfg.snap_every, dtype=torch.int64, device="cuda")
        pgg.pgg_sweep(d, fmt, L, r, K, seed, order, a * cfg.snap_every, cfg.snap_every, cnt)
        torch.cuda.synchronize()
        assert_same(to_host(d, fmt, L), ref_snaps[a], f"snapshot after {(a + 1) * cfg.snap_every} MCS")
        counts.append(cnt.cpu().numpy().astype(np.uint64))
    assert_same(np.concatenate(counts), ref_counts, "rho_C trace")


# ---------------------------------------------------------------- sizes, tails, wrap
SIZES = [4, 8, 12, 16, 20, 32, 36, 48, 64, 100, 128, 144, 256, 400, 512, 640]


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("fmt", FMTS)
@pytest.mark.parametrize("L", SIZES)
def test_sweep_parity_sizes(variant, fmt, L):
    """Several tiles plus ragged tails; L = 4 and 8 exercise coinciding wrap neighbours."""
    if fmt == pgg.FMT_BITS and L % 32:
        pytest.skip("bits layout needs L % 32 == 0")
    use_variant(variant, fmt, L)
    n_mcs = 12 if L <= 256 else 5
    for seed, r, order in ((L + 1, 3.8, pgg.ORDER_IID), (2**35 + L, 4.6, pgg.ORDER_PERM)):
        lat0 = orc.init(L, 0.5, seed)
        ref = lat0.copy()
        ref_counts, _ = orc.sweep(ref, r, K, seed, order, 3, n_mcs)
        got, counts = gpu_sweep(lat0, fmt, r, seed, order, 3, n_mcs)
        assert_same(got, ref, f"lattice L={L}")
        assert_same(counts, ref_counts, f"counts L={L}")


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("fmt", FMTS)
def test_sweep_parity_structured_states(variant, fmt):
    """Interfaces, compact clusters and the checkerboard: states where most
    sites are bulk (skipped) or where every site is active."""
    L = 256
    use_variant(variant, fmt, L)
    states = [wl.blobs_lattice(L, 3), wl.stripes_lattice(L, 5, True), wl.stripes_lattice(L, 7, False),
              wl.checkerboard_lattice(L), wl.random_lattice(L, 0.03, 8), wl.random_lattice(L, 0.97, 9)]
    for n, lat0 in enumerate(states):
        for r in (3.8, 5.4):
            ref = lat0.copy()
            ref_counts, _ = orc.sweep(ref, r, K, 77 + n, pgg.ORDER_IID, 0, 8)
            got, counts = gpu_sweep(lat0, fmt, r, 77 + n, pgg.ORDER_IID, 0, 8)
            assert_same(got, ref, f"state {n}")
            assert_same(counts, ref_counts, f"counts state {n}")


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("fmt", FMTS)
def test_absorbing_states_stay_absorbing(variant, fmt):
    L = 128
    use_variant(variant, fmt, L)
    for v in (0, 1):
        lat0 = np.full((L, L), v, dtype=np.uint8)
        got, counts = gpu_sweep(lat0, fmt, 3.8, 5, pgg.ORDER_IID, 0, 6)
        assert_same(got, lat0)
        assert (counts == v * L * L).all()


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("fmt", FMTS)
def test_extreme_parameters(variant, fmt):
    """Clamped table entries (S7): tiny K (step function) and huge r."""
    L = 128
    use_variant(variant, fmt, L)
    for r, Kx in ((4.0, 1e-3), (25.0, 0.5), (1.0, 50.0)):
        lat0 = orc.init(L, 0.5, 21)
        ref = lat0.copy()
        tab = orc.accept_table(r, Kx)
        assert np.array_equal(tab, np.array(pgg.pgg_build_accept_table(r, Kx), dtype=np.uint32))
        ref_counts, _ = orc.sweep(ref, r, Kx, 21, pgg.ORDER_IID, 0, 6)
        d = to_device(lat0, fmt)
        cnt = torch.zeros(6, dtype=torch.int64, device="cuda")
        pgg.pgg_sweep(d, fmt, L, r, Kx, 21, pgg.ORDER_IID, 0, 6, cnt)
        torch.cuda.synchronize()
        assert_same(to_host(d, fmt, L), ref)
        assert_same(cnt.cpu().numpy().astype(np.uint64), ref_counts)


# ---------------------------------------------------------------- composition (P7)
@pytest.mark.parametrize("fmt", FMTS)
def test_composition_and_late_window(fmt):
    """(a,b) then (a+b,c) == (a,b+c); t_begin near 2^32 exercises the counter width."""
    L = 128
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)
    lat0 = orc.init(L, 0.5, 4)
    for t0 in (0, 2**32 - 40):
        one, c_one = gpu_sweep(lat0, fmt, 3.9, 4, pgg.ORDER_IID, t0, 30)
        d = to_device(lat0, fmt)
        c1 = torch.zeros(12, dtype=torch.int64, device="cuda")
        c2 = torch.zeros(18, dtype=torch.int64, device="cuda")
        pgg.pgg_sweep(d, fmt, L, 3.9, K, 4, pgg.ORDER_IID, t0, 12, c1)
        pgg.pgg_sweep(d, fmt, L, 3.9, K, 4, pgg.ORDER_IID, t0 + 12, 18, c2)
        torch.cuda.synchronize()
        assert_same(to_host(d, fmt, L), one)
        assert_same(torch.cat([c1, c2]).cpu().numpy().astype(np.uint64), c_one)
        ref = lat0.copy()
        ref_counts, _ = orc.sweep(ref, 3.9, K, 4, pgg.ORDER_IID, t0, 30)
        assert_same(one, ref)
        assert_same(c_one, ref_counts)


def test_counts_null_and_zero_mcs():
    L = 64
    lat0 = orc.init(L, 0.5, 2)
    got, _ = gpu_sweep(lat0, pgg.FMT_U8, 3.8, 2, pgg.ORDER_IID, 0, 4, want_counts=False)
    ref = lat0.copy()
    orc.sweep(ref, 3.8, K, 2, pgg.ORDER_IID, 0, 4)
    assert_same(got, ref)
    got, _ = gpu_sweep(lat0, pgg.FMT_U8, 3.8, 2, pgg.ORDER_IID, 0, 0, want_counts=False)
    assert_same(got, lat0)


# ---------------------------------------------------------------- a9 ensemble
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("fmt", FMTS)
def test_ensemble_equals_solo_and_oracle(variant, fmt):
    """Config-4 shape at reduced size: B lattices, r_k = 3.70 + (0.1 k)/63, seeds 1000+k."""
    cfg = wl.config4()
    B, L, n_mcs = 8, 128, 20
    use_variant(variant, fmt, L)
    rs, seeds = cfg.rs[::8][:B], cfg.seeds[::8][:B]
    d = empty_lattice(fmt, L, B)
    cnt = torch.zeros((B, n_mcs), dtype=torch.int64, device="cuda")
    pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_IID, 0.5, 0, n_mcs, cnt)
    torch.cuda.synchronize()
    got = to_host(d, fmt, L)
    counts = cnt.cpu().numpy().astype(np.uint64)
    for b in range(B):
        ref = orc.init(L, 0.5, seeds[b])
        solo, solo_counts = gpu_sweep(ref, fmt, rs[b], seeds[b], pgg.ORDER_IID, 0, n_mcs)
        ref_counts, _ = orc.sweep(ref, rs[b], K, seeds[b], pgg.ORDER_IID, 0, n_mcs)
        assert_same(got[b], ref, f"member {b} vs oracle")
        assert_same(got[b], solo, f"member {b} vs solo")
        assert_same(counts[b], ref_counts)
        assert_same(solo_counts, ref_counts)
    # continue (rho0 < 0) from the given states
    pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_PERM, -1.0, n_mcs, 3, None)
    torch.cuda.synchronize()
    got2 = to_host(d, fmt, L)
    for b in range(B):
        ref = got[b].copy()
        orc.sweep(ref, rs[b], K, seeds[b], pgg.ORDER_PERM, n_mcs, 3)
        assert_same(got2[b], ref, f"member {b} continued")


# ---------------------------------------------------------------- full-size configs
@pytest.mark.parametrize("fmt", FMTS)
def test_config3_and_4_shapes_prefix(fmt):
    """Configs 3 and 4 at full lattice size, in the ensemble launch bench-like runs use,
    for a prefix of MCS the oracle finishes in seconds (full-length runs: DESIGN.md)."""
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)
    for cfg, B, n_mcs in ((wl.config3(), 2, 3), (wl.config4(), 4, 6)):
        L = cfg.L
        rs, seeds = cfg.rs[-B:], cfg.seeds[-B:]
        d = empty_lattice(fmt, L, B)
        cnt = torch.zeros((B, n_mcs), dtype=torch.int64, device="cuda")
        pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_IID, cfg.rho0, 0, n_mcs, cnt)
        torch.cuda.synchronize()
        got = to_host(d, fmt, L)
        for b in range(B):
            ref = orc.init(L, cfg.rho0, seeds[b])
            ref_counts, _ = orc.sweep(ref, rs[b], K, seeds[b], pgg.ORDER_IID, 0, n_mcs,
                                      n_threads=orc.max_threads())
            assert_same(got[b], ref, f"{cfg.name} member {b}")
            assert_same(cnt[b].cpu().numpy().astype(np.uint64), ref_counts)


@pytest.mark.parametrize("fmt", FMTS)
def test_config5_full_size(fmt):
    """BASELINE.json configs[4] at its full size (L=16384) in the launch configuration
    bench.py times: whole lattice and counts after 2 MCS against a live oracle run.  Later
    times (lattice hashes and the whole count trace of a stored oracle run) are checked in
    tests/test_gpu_goldens.py; no GPU-produced state is ever handed to the oracle."""
    cfg = wl.config5()
    L, r, seed = cfg.L, cfg.rs[0], cfg.seeds[0]
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)
    d = empty_lattice(fmt, L)
    pgg.pgg_init_lattice(d, fmt, L, cfg.rho0, seed)
    cnt = torch.zeros(2, dtype=torch.int64, device="cuda")
    pgg.pgg_sweep(d, fmt, L, r, K, seed, pgg.ORDER_IID, 0, 2, cnt)
    torch.cuda.synchronize()
    ref = orc.init(L, cfg.rho0, seed)
    ref_counts, _ = orc.sweep(ref, r, K, seed, pgg.ORDER_IID, 0, 2, n_threads=orc.max_threads())
    assert_same(to_host(d, fmt, L), ref, "C5 lattice after 2 MCS")
    assert_same(cnt.cpu().numpy().astype(np.uint64), ref_counts)


@pytest.mark.parametrize("fmt", FMTS)
def test_oversubscribed_ensemble(fmt):
    """More CTAs than SMs (300 lattices of L=1024): the streaming kernels are launched with the
    programmatic-dependent-launch attribute, so a phase may start while CTAs of the previous one are
    still queued.  Sampled members against the oracle, all members across kernel variants."""
    B, L, n_mcs = 300, 1024, 4
    rs = [3.7 + 0.001 * b for b in range(B)]
    seeds = list(range(100, 100 + B))
    variants = [v for v in (pgg.VARIANT_V0, pgg.VARIANT_BAND, pgg.VARIANT_RING, pgg.VARIANT_DYN)
                if pgg.pgg_variant_supported(v, fmt, L)]
    first = None
    for v in variants:
        pgg.pgg_set_variant(v)
        d = empty_lattice(fmt, L, B)
        cnt = torch.zeros((B, n_mcs), dtype=torch.int64, device="cuda")
        pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_IID, 0.5, 0, n_mcs, cnt)
        torch.cuda.synchronize()
        if first is None:
            first = (d, cnt)
            for b in (0, 149, 299):
                ref = orc.init(L, 0.5, seeds[b])
                ref_counts, _ = orc.sweep(ref, rs[b], K, seeds[b], pgg.ORDER_IID, 0, n_mcs,
                                          n_threads=orc.max_threads())
                assert_same(to_host(d[b], fmt, L), ref, f"member {b}")
                assert_same(cnt[b].cpu().numpy().astype(np.uint64), ref_counts)
        else:
            assert torch.equal(d, first[0]) and torch.equal(cnt, first[1]), f"variant {v} differs from variant {variants[0]}"
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)


@pytest.mark.parametrize("L", [4096, 8192])
def test_fullrow_strip_sizes(L):
    """uint8 lattices whose row is one strip (512 B ... 8 KB): staged without halo columns, one bulk copy
    per chunk, column wrap resolved in the sites near a row end (RING full-row mode)."""
    pgg.pgg_set_variant(pgg.VARIANT_RING)
    seed, r, n_mcs = 40 + L, 3.8, 2
    lat0 = orc.init(L, 0.5, seed)
    ref = lat0.copy()
    ref_counts, _ = orc.sweep(ref, r, K, seed, pgg.ORDER_IID, 5, n_mcs, n_threads=orc.max_threads())
    got, counts = gpu_sweep(lat0, pgg.FMT_U8, r, seed, pgg.ORDER_IID, 5, n_mcs)
    assert pgg.pgg_get_variant_used() == pgg.VARIANT_RING
    assert_same(got, ref, f"lattice L={L}")
    assert_same(counts, ref_counts, f"counts L={L}")


def test_large_lattice_L32768():
    """A 1 GiB uint8 lattice (4 strips of 8 KB, site indices up to 2^30): one MCS against the oracle."""
    L, seed, r = 32768, 9, 3.8
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)
    d = empty_lattice(pgg.FMT_U8, L)
    pgg.pgg_init_lattice(d, pgg.FMT_U8, L, 0.5, seed)
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    pgg.pgg_sweep(d, pgg.FMT_U8, L, r, K, seed, pgg.ORDER_IID, 7, 1, cnt)
    torch.cuda.synchronize()
    ref = orc.init(L, 0.5, seed)
    ref_counts, _ = orc.sweep(ref, r, K, seed, pgg.ORDER_IID, 7, 1, n_threads=orc.max_threads())
    got = d.cpu().numpy()
    del d
    assert np.array_equal(got, ref), "L=32768 lattice differs"
    assert int(cnt.item()) == int(ref_counts[0])


# ---------------------------------------------------------------- long calls: order-buffer chunks, late windows
# run_sweeps() holds the phase classes of at most 4096 MCS on the device and rewrites that buffer
# between two dependent-launch chained phases; every 10^5..10^6-MCS physics run crosses it.
LONG_CASES = [
    # (variant, fmt, L, env) -- the kernels AUTO ships for long runs, each forced by name
    ("RING", pgg.FMT_U8, 512, {}),                               # RING, full-row mode (C3's path)
    ("RING", pgg.FMT_U8, 512, {"PGG_RING_FULLROW": "0"}),        # RING, strips with halo columns (C5's path)
    ("BAND", pgg.FMT_BITS, 512, {}),                             # BAND, bit-packed (C5 packed)
    ("LEAN", pgg.FMT_U8, 1024, {}),                              # LEAN, uint8 packed to bits on chip
    ("LEAN", pgg.FMT_BITS, 1024, {}),                            # LEAN, bit-packed source
    ("PERSIST", pgg.FMT_BITS, 1024, {}),                         # LEAN, one cooperative launch per 4096 MCS
    ("CLUSTER", pgg.FMT_U8, 1024, {}),                           # lattice resident in a cluster's shared memory
    ("CLUSTER", pgg.FMT_BITS, 1024, {}),
    ("PACKED", pgg.FMT_U8, 1024, {}),                            # uint8 in HBM, bit-packed working copy + LEAN (C5's path)
]


def _variant_by_name(name):
    return getattr(pgg, "VARIANT_" + name)


@pytest.mark.parametrize("name,fmt,L,env", LONG_CASES,
                         ids=[f"{n}-{'u8' if f == pgg.FMT_U8 else 'bits'}-L{L}{'-strips' if e else ''}"
                              for n, f, L, e in LONG_CASES])
def test_one_call_longer_than_an_order_chunk(name, fmt, L, env, monkeypatch):
    """ONE call of 4200 MCS from t_begin = 4000 (a call that starts mid-way through the run and
    crosses the 4096-MCS order-buffer boundary): lattice and the whole count trace against a live
    oracle run.  PAPER.md:113 (runs of 10^5..3*10^6 MCS near r_c) is what takes this path."""
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    use_variant(_variant_by_name(name), fmt, L)
    seed, r, t0, n_mcs = 900 + L, 3.8, 4000, 4200
    lat0 = orc.init(L, 0.5, seed)
    ref = lat0.copy()
    ref_counts, _ = orc.sweep(ref, r, K, seed, pgg.ORDER_IID, t0, n_mcs, n_threads=orc.max_threads())
    got, counts = gpu_sweep(lat0, fmt, r, seed, pgg.ORDER_IID, t0, n_mcs)
    assert_same(counts, ref_counts, "count trace across the chunk boundary")
    assert_same(got, ref, "lattice after 4200 MCS")
    assert 0 < int(ref_counts[-1]) < L * L, "the run must not have been absorbed (it would test nothing)"


@pytest.mark.parametrize("name,fmt,L,env", LONG_CASES,
                         ids=["RING-fullrow", "RING-strips", "BAND-bits", "LEAN-u8", "LEAN-bits", "PERSIST-bits", "CLUSTER-u8", "CLUSTER-bits", "PACKED-u8"])
@pytest.mark.parametrize("t0", [99900, 2**32 - 40])
def test_streaming_kernels_late_windows(name, fmt, L, env, t0, monkeypatch):
    """SURVEY 8(d) late windows (t = 99 900) and the counter width (t_begin + m up to 2^32 - 1)
    for the streaming kernels by name; the oracle starts from the same given state (legal by P7)."""
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    use_variant(_variant_by_name(name), fmt, L)
    seed, r, n_mcs = 2**34 + 77, 3.9, 40
    lat0 = wl.random_lattice(L, 0.3, 5)
    ref = lat0.copy()
    ref_counts, _ = orc.sweep(ref, r, K, seed, pgg.ORDER_IID, t0, n_mcs, n_threads=orc.max_threads())
    got, counts = gpu_sweep(lat0, fmt, r, seed, pgg.ORDER_IID, t0, n_mcs)
    assert_same(got, ref, f"lattice, window at t = {t0}")
    assert_same(counts, ref_counts, f"counts, window at t = {t0}")


# ---------------------------------------------------------------- LEAN (L = 1024 .. 32768, powers of two)
@pytest.mark.parametrize("fmt", FMTS)
@pytest.mark.parametrize("L,n_mcs", [(1024, 6), (2048, 4), (4096, 3), (8192, 2)])
def test_lean_parity_sizes(fmt, L, n_mcs):
    """One band per SM down to one step per CTA (L = 1024: 16 active rows per step), both orders,
    a 64-bit seed, from the dense random start (every extraction round crowded) and a sparse one."""
    use_variant(pgg.VARIANT_LEAN, fmt, L)
    for seed, r, order, rho0 in ((L + 1, 3.8, pgg.ORDER_IID, 0.5), (2**35 + L, 4.6, pgg.ORDER_PERM, 0.1)):
        lat0 = orc.init(L, rho0, seed)
        ref = lat0.copy()
        ref_counts, _ = orc.sweep(ref, r, K, seed, order, 3, n_mcs, n_threads=orc.max_threads())
        got, counts = gpu_sweep(lat0, fmt, r, seed, order, 3, n_mcs)
        assert pgg.pgg_get_variant_used() == pgg.VARIANT_LEAN
        assert_same(got, ref, f"lattice L={L}")
        assert_same(counts, ref_counts, f"counts L={L}")


@pytest.mark.parametrize("fmt", FMTS)
def test_lean_structured_absorbing_and_clamped(fmt):
    """Checkerboard (all eight active sites of every word survive the S9 test: the split
    extraction round), stripes and blobs (mostly bulk), absorbing states, clamped tables."""
    L = 1024
    use_variant(pgg.VARIANT_LEAN, fmt, L)
    states = [wl.checkerboard_lattice(L), wl.stripes_lattice(L, 5, True), wl.stripes_lattice(L, 7, False),
              wl.blobs_lattice(L, 3), wl.random_lattice(L, 0.03, 8), wl.random_lattice(L, 0.97, 9)]
    for n, lat0 in enumerate(states):
        for r, Kx in ((3.8, K), (5.4, K), (4.0, 1e-3)):
            ref = lat0.copy()
            ref_counts, _ = orc.sweep(ref, r, Kx, 77 + n, pgg.ORDER_IID, 0, 4, n_threads=orc.max_threads())
            d = to_device(lat0, fmt)
            cnt = torch.zeros(4, dtype=torch.int64, device="cuda")
            pgg.pgg_sweep(d, fmt, L, r, Kx, 77 + n, pgg.ORDER_IID, 0, 4, cnt)
            torch.cuda.synchronize()
            assert_same(to_host(d, fmt, L), ref, f"state {n} r={r} K={Kx}")
            assert_same(cnt.cpu().numpy().astype(np.uint64), ref_counts, f"counts state {n}")
    for v in (0, 1):
        lat0 = np.full((L, L), v, dtype=np.uint8)
        got, counts = gpu_sweep(lat0, fmt, 3.8, 5, pgg.ORDER_IID, 0, 3)
        assert_same(got, lat0)
        assert (counts == v * L * L).all()


@pytest.mark.parametrize("fmt", FMTS)
def test_lean_ensemble_equals_solo_and_oracle(fmt):
    """Config-3 shape at reduced length: B lattices of L = 2048 in one grid per phase (bands share
    the SMs), each with its own r and seed; then continued (rho0 < 0) in PERM order."""
    B, L, n_mcs = 5, 2048, 3
    use_variant(pgg.VARIANT_LEAN, fmt, L)
    rs = [3.74 + 0.01 * b for b in range(B)]
    seeds = [2**33 + 11 * b for b in range(B)]
    d = empty_lattice(fmt, L, B)
    cnt = torch.zeros((B, n_mcs), dtype=torch.int64, device="cuda")
    pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_IID, 0.5, 0, n_mcs, cnt)
    torch.cuda.synchronize()
    got = to_host(d, fmt, L)
    for b in range(B):
        ref = orc.init(L, 0.5, seeds[b])
        ref_counts, _ = orc.sweep(ref, rs[b], K, seeds[b], pgg.ORDER_IID, 0, n_mcs, n_threads=orc.max_threads())
        assert_same(got[b], ref, f"member {b}")
        assert_same(cnt[b].cpu().numpy().astype(np.uint64), ref_counts)
    pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_PERM, -1.0, n_mcs, 2, None)
    torch.cuda.synchronize()
    got2 = to_host(d, fmt, L)
    for b in (0, B - 1):
        ref = got[b].copy()
        orc.sweep(ref, rs[b], K, seeds[b], pgg.ORDER_PERM, n_mcs, 2, n_threads=orc.max_threads())
        assert_same(got2[b], ref, f"member {b} continued")


@pytest.mark.parametrize("fmt", FMTS)
def test_lean_config5_full_size(fmt):
    """BASELINE.json configs[4] (L = 16384) through LEAN by name: 2 MCS against a live oracle run."""
    cfg = wl.config5()
    L, r, seed = cfg.L, cfg.rs[0], cfg.seeds[0]
    use_variant(pgg.VARIANT_LEAN, fmt, L)
    d = empty_lattice(fmt, L)
    pgg.pgg_init_lattice(d, fmt, L, cfg.rho0, seed)
    cnt = torch.zeros(2, dtype=torch.int64, device="cuda")
    pgg.pgg_sweep(d, fmt, L, r, K, seed, pgg.ORDER_IID, 0, 2, cnt)
    torch.cuda.synchronize()
    ref = orc.init(L, cfg.rho0, seed)
    ref_counts, _ = orc.sweep(ref, r, K, seed, pgg.ORDER_IID, 0, 2, n_threads=orc.max_threads())
    assert_same(to_host(d, fmt, L), ref, "C5 lattice after 2 MCS")
    assert_same(cnt.cpu().numpy().astype(np.uint64), ref_counts)


# ---------------------------------------------------------------- PERSIST (LEAN in one cooperative launch)
@pytest.mark.parametrize("L,n_mcs", [(1024, 6), (2048, 4), (4096, 3), (16384, 2)])
def test_persist_parity_sizes(L, n_mcs):
    """Every phase of the call in one launch, a barrier in global memory between phases: the same
    lattices and counts as the oracle, from one CTA per lattice row group (L = 1024) to C5's size."""
    fmt = pgg.FMT_BITS
    use_variant(pgg.VARIANT_PERSIST, fmt, L)
    for seed, r, order, rho0 in ((L + 1, 3.8, pgg.ORDER_IID, 0.5), (2**35 + L, 4.6, pgg.ORDER_PERM, 0.1)):
        lat0 = orc.init(L, rho0, seed)
        ref = lat0.copy()
        ref_counts, _ = orc.sweep(ref, r, K, seed, order, 3, n_mcs, n_threads=orc.max_threads())
        before = pgg.pgg_launch_count()
        got, counts = gpu_sweep(lat0, fmt, r, seed, order, 3, n_mcs)
        assert pgg.pgg_get_variant_used() == pgg.VARIANT_PERSIST
        assert pgg.pgg_launch_count() - before == 5       # upload, density, order, ONE sweep launch, finalize
        assert_same(got, ref, f"lattice L={L}")
        assert_same(counts, ref_counts, f"counts L={L}")


def test_persist_ensemble_equals_oracle():
    """16 lattices of L = 2048 (config 3's shape): each lattice's CTAs meet at their own barrier."""
    fmt, B, L, n_mcs = pgg.FMT_BITS, 16, 2048, 3
    use_variant(pgg.VARIANT_PERSIST, fmt, L)
    rs = [3.74 + 0.002 * b for b in range(B)]
    seeds = [2**33 + 7 * b for b in range(B)]
    d = empty_lattice(fmt, L, B)
    cnt = torch.zeros((B, n_mcs), dtype=torch.int64, device="cuda")
    pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_IID, 0.5, 0, n_mcs, cnt)
    torch.cuda.synchronize()
    got = to_host(d, fmt, L)
    for b in (0, 7, 15):
        ref = orc.init(L, 0.5, seeds[b])
        ref_counts, _ = orc.sweep(ref, rs[b], K, seeds[b], pgg.ORDER_IID, 0, n_mcs, n_threads=orc.max_threads())
        assert_same(got[b], ref, f"member {b}")
        assert_same(cnt[b].cpu().numpy().astype(np.uint64), ref_counts)


# ---------------------------------------------------------------- CLUSTER (lattice resident in a CTA cluster)
@pytest.mark.parametrize("fmt", FMTS)
@pytest.mark.parametrize("L,n_mcs", [(1024, 8), (2048, 5), (4096, 3)])
def test_cluster_parity_sizes(fmt, L, n_mcs):
    """The lattice stays in the shared memory of 8 (L = 4096: 16) CTAs for the whole call; halo rows travel
    over distributed shared memory after every phase.  Lattice and counts against the oracle; one sweep
    launch per call; dense and sparse starts, both orders, a 64-bit seed, a late t_begin."""
    use_variant(pgg.VARIANT_CLUSTER, fmt, L)
    for seed, r, order, rho0, t0 in ((L + 1, 3.8, pgg.ORDER_IID, 0.5, 3), (2**35 + L, 4.6, pgg.ORDER_PERM, 0.1, 2**32 - 20)):
        lat0 = orc.init(L, rho0, seed)
        ref = lat0.copy()
        ref_counts, _ = orc.sweep(ref, r, K, seed, order, t0, n_mcs, n_threads=orc.max_threads())
        before = pgg.pgg_launch_count()
        got, counts = gpu_sweep(lat0, fmt, r, seed, order, t0, n_mcs)
        assert pgg.pgg_get_variant_used() == pgg.VARIANT_CLUSTER
        assert pgg.pgg_launch_count() - before == 5       # upload, density, order, ONE sweep launch, finalize
        assert_same(got, ref, f"lattice L={L}")
        assert_same(counts, ref_counts, f"counts L={L}")


def test_packed_ensemble_init_and_continuation():
    """PGG_VARIANT_PACKED (uint8 in HBM, bit-packed working copy for the length of the call): an ensemble that is
    initialised inside the call, then continued by a second call from the uint8 state the first one left
    (the working copy is private to a call), against the oracle; and the caller's buffer is the only output."""
    L, B, fmt = 1024, 3, pgg.FMT_U8
    use_variant(pgg.VARIANT_PACKED, fmt, L)
    rs, seeds = [3.75, 3.9, 5.4], [2**40 + 1, 17, 99]
    d = empty_lattice(fmt, L, B)
    c1 = torch.zeros((B, 3), dtype=torch.int64, device="cuda")
    c2 = torch.zeros((B, 2), dtype=torch.int64, device="cuda")
    before = pgg.pgg_launch_count()
    pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_IID, 0.5, 0, 3, c1)
    # upload, init, density, pack, order, 16 phases per MCS, unpack, finalize
    assert pgg.pgg_launch_count() - before == 1 + 1 + 1 + 1 + 1 + 16 * 3 + 1 + 1
    assert pgg.pgg_get_variant_used() == pgg.VARIANT_PACKED
    pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_PERM, -1.0, 3, 2, c2)
    torch.cuda.synchronize()
    got = to_host(d, fmt, L)
    for b in range(B):
        ref = orc.init(L, 0.5, seeds[b])
        r1, _ = orc.sweep(ref, rs[b], K, seeds[b], pgg.ORDER_IID, 0, 3, n_threads=orc.max_threads())
        r2, _ = orc.sweep(ref, rs[b], K, seeds[b], pgg.ORDER_PERM, 3, 2, n_threads=orc.max_threads())
        assert_same(got[b], ref, f"member {b}")
        assert_same(c1[b].cpu().numpy().astype(np.uint64), r1, f"counts of call 1, member {b}")
        assert_same(c2[b].cpu().numpy().astype(np.uint64), r2, f"counts of call 2, member {b}")
    pgg.pgg_trim_workspace()  # gives the pool's cached working copy back; the next call allocates afresh
    lat0 = got[0].copy()
    ref = lat0.copy()
    orc.sweep(ref, 3.8, K, 5, pgg.ORDER_IID, 5, 1, n_threads=orc.max_threads())
    out, _ = gpu_sweep(lat0, fmt, 3.8, 5, pgg.ORDER_IID, 5, 1)
    assert_same(out, ref, "after pgg_trim_workspace")


@pytest.mark.parametrize("cs", [1, 2, 4, 8, 16])
def test_cluster_every_cluster_size(cs, monkeypatch):
    """The neighbour-only halo exchange (asynchronous stores that complete on the neighbour's mbarrier, no cluster
    barrier) for every cluster size, CS = 1 (the CTA is its own neighbour) and CS = 2 (both neighbours are the same
    CTA) included: five lattices of L = 512 for 50 MCS (800 phases, every class row many times) against the oracle."""
    monkeypatch.setenv("PGG_CLUSTER_SIZE", str(cs))
    L, B, n_mcs, fmt = 512, 5, 50, pgg.FMT_BITS
    use_variant(pgg.VARIANT_CLUSTER, fmt, L)
    rs = [3.74 + 0.02 * b for b in range(B)]
    seeds = [2**36 + 11 * b + cs for b in range(B)]
    d = empty_lattice(fmt, L, B)
    cnt = torch.zeros((B, n_mcs), dtype=torch.int64, device="cuda")
    pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_IID, 0.5, 0, n_mcs, cnt)
    torch.cuda.synchronize()
    got = to_host(d, fmt, L)
    for b in range(B):
        ref = orc.init(L, 0.5, seeds[b])
        ref_counts, _ = orc.sweep(ref, rs[b], K, seeds[b], pgg.ORDER_IID, 0, n_mcs, n_threads=orc.max_threads())
        assert_same(got[b], ref, f"member {b}, cluster size {cs}")
        assert_same(cnt[b].cpu().numpy().astype(np.uint64), ref_counts, f"counts of member {b}, cluster size {cs}")


@pytest.mark.parametrize("fmt", FMTS)
def test_cluster_structured_ensembles_and_waves(fmt):
    """Structured and absorbing states; an ensemble of 40 lattices of L = 1024 (more clusters than the GPU
    holds at once: they run in waves); members against the oracle."""
    L = 1024
    use_variant(pgg.VARIANT_CLUSTER, fmt, L)
    for n, lat0 in enumerate([wl.checkerboard_lattice(L), wl.stripes_lattice(L, 7, False), wl.blobs_lattice(L, 3),
                              np.zeros((L, L), np.uint8), np.ones((L, L), np.uint8)]):
        ref = lat0.copy()
        ref_counts, _ = orc.sweep(ref, 3.8, K, 70 + n, pgg.ORDER_IID, 0, 4, n_threads=orc.max_threads())
        got, counts = gpu_sweep(lat0, fmt, 3.8, 70 + n, pgg.ORDER_IID, 0, 4)
        assert_same(got, ref, f"state {n}")
        assert_same(counts, ref_counts, f"counts state {n}")
    B, n_mcs = 40, 3
    rs = [3.7 + 0.005 * b for b in range(B)]
    seeds = [2**33 + 3 * b for b in range(B)]
    d = empty_lattice(fmt, L, B)
    cnt = torch.zeros((B, n_mcs), dtype=torch.int64, device="cuda")
    pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_IID, 0.5, 0, n_mcs, cnt)
    torch.cuda.synchronize()
    got = to_host(d, fmt, L)
    for b in (0, 17, 39):
        ref = orc.init(L, 0.5, seeds[b])
        ref_counts, _ = orc.sweep(ref, rs[b], K, seeds[b], pgg.ORDER_IID, 0, n_mcs, n_threads=orc.max_threads())
        assert_same(got[b], ref, f"member {b}")
        assert_same(cnt[b].cpu().numpy().astype(np.uint64), ref_counts)

"""The prisoner's dilemma on the GPU against its oracle, bit for bit (``-m gpu``).

Same schedule, same draws as the public goods game; the payoffs are pair games with the four nearest
neighbours (readings G1-G4, include/pgg.h).  Two kernels carry it: V0 (any L % 4 == 0) and LEAN
(L = 1024 .. 32768, powers of two); both layouts."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1704_08098_b200 as pgg  # noqa: E402
from test_gpu_parity import assert_same, to_device, to_host  # noqa: E402

WEAK = (1.0, 0.0, 1.05, 0.0)     # coexistence of C and D at K = 0.1 on this lattice
GEN = (3.0, -0.5, 4.25, 0.75)


@pytest.fixture(scope="module", autouse=True)
def _gpu():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    pgg.lib()
    yield
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)


def gpu_pd(lat0, fmt, pay, K, seed, order, t0, n_mcs):
    L = lat0.shape[0]
    d = to_device(lat0, fmt)
    cnt = torch.zeros(n_mcs, dtype=torch.int64, device="cuda")
    pgg.pgg_pd_sweep(d, fmt, L, *pay, K, seed, order, t0, n_mcs, cnt)
    torch.cuda.synchronize()
    return to_host(d, fmt, L), cnt.cpu().numpy().astype(np.uint64)


@pytest.mark.parametrize("fmt", [pgg.FMT_U8, pgg.FMT_BITS])
@pytest.mark.parametrize("L", [4, 8, 20, 32, 64, 100, 256, 416, 640])
def test_pd_parity_v0_sizes(fmt, L):
    """L = 4 and 8: wrap neighbours coincide (x's neighbour two steps away is y's other neighbour)."""
    if fmt == pgg.FMT_BITS and L % 32:
        pytest.skip("bits layout needs L % 32 == 0")
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)
    for seed, pay, K, order in ((L + 1, WEAK, 0.1, pgg.ORDER_IID), (2**36 + L, GEN, 0.5, pgg.ORDER_PERM)):
        lat0 = orc.init(L, 0.5, seed)
        ref = lat0.copy()
        ref_counts = orc.pd_sweep(ref, *pay, K, seed, order, 2, 10)
        got, counts = gpu_pd(lat0, fmt, pay, K, seed, order, 2, 10)
        assert pgg.pgg_get_variant_used() == pgg.VARIANT_V0
        assert_same(got, ref, f"PD lattice L={L}")
        assert_same(counts, ref_counts, f"PD counts L={L}")


@pytest.mark.parametrize("fmt", [pgg.FMT_U8, pgg.FMT_BITS])
@pytest.mark.parametrize("L,n_mcs", [(1024, 12), (2048, 6), (4096, 3)])
def test_pd_parity_lean(fmt, L, n_mcs):
    pgg.pgg_set_variant(pgg.VARIANT_LEAN)
    for seed, pay, K, order, t0 in ((L + 3, WEAK, 0.1, pgg.ORDER_IID, 0), (2**34 + L, GEN, 0.5, pgg.ORDER_PERM, 2**32 - 20)):
        lat0 = orc.init(L, 0.5, seed)
        ref = lat0.copy()
        ref_counts = orc.pd_sweep(ref, *pay, K, seed, order, t0, n_mcs)
        got, counts = gpu_pd(lat0, fmt, pay, K, seed, order, t0, n_mcs)
        assert pgg.pgg_get_variant_used() == pgg.VARIANT_LEAN
        assert_same(got, ref, f"PD lattice L={L}")
        assert_same(counts, ref_counts, f"PD counts L={L}")
    # the two kernels agree with each other as well (V0 by name at a LEAN size)
    pgg.pgg_set_variant(pgg.VARIANT_V0)
    got_v0, counts_v0 = gpu_pd(lat0, fmt, pay, K, seed, order, t0, n_mcs)
    assert_same(got_v0, ref) and assert_same(counts_v0, ref_counts)


@pytest.mark.parametrize("fmt", [pgg.FMT_U8, pgg.FMT_BITS])
@pytest.mark.parametrize("L,n_mcs", [(512, 12), (1024, 8), (2048, 4)])
def test_pd_parity_cluster(fmt, L, n_mcs):
    """The cluster-resident kernel (AUTO's choice for L = 512 and 1024) with the pair-game payoffs."""
    pgg.pgg_set_variant(pgg.VARIANT_AUTO if L <= 1024 else pgg.VARIANT_CLUSTER)
    for seed, pay, K, order, t0 in ((L + 5, WEAK, 0.1, pgg.ORDER_IID, 0), (2**34 + L, GEN, 0.5, pgg.ORDER_PERM, 2**32 - 20)):
        lat0 = orc.init(L, 0.5, seed)
        ref = lat0.copy()
        ref_counts = orc.pd_sweep(ref, *pay, K, seed, order, t0, n_mcs)
        got, counts = gpu_pd(lat0, fmt, pay, K, seed, order, t0, n_mcs)
        assert pgg.pgg_get_variant_used() == pgg.VARIANT_CLUSTER
        assert_same(got, ref, f"PD lattice L={L}")
        assert_same(counts, ref_counts, f"PD counts L={L}")
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)


@pytest.mark.parametrize("fmt", [pgg.FMT_U8, pgg.FMT_BITS])
def test_pd_structured_and_absorbing_states(fmt):
    L = 1024
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)
    for n, lat0 in enumerate([wl.checkerboard_lattice(L), wl.stripes_lattice(L, 5, True), wl.blobs_lattice(L, 3),
                              wl.random_lattice(L, 0.03, 8)]):
        for pay, K in ((WEAK, 0.1), (GEN, 1e-3)):
            ref = lat0.copy()
            ref_counts = orc.pd_sweep(ref, *pay, K, 50 + n, pgg.ORDER_IID, 0, 4)
            got, counts = gpu_pd(lat0, fmt, pay, K, 50 + n, pgg.ORDER_IID, 0, 4)
            assert_same(got, ref, f"PD state {n}")
            assert_same(counts, ref_counts, f"PD counts state {n}")
    for v in (0, 1):
        lat0 = np.full((L, L), v, dtype=np.uint8)
        got, counts = gpu_pd(lat0, fmt, WEAK, 0.1, 5, pgg.ORDER_IID, 0, 3)
        assert_same(got, lat0) and (counts == v * L * L).all()


def test_pd_rejects_other_variants_and_the_papers_schedule():
    d = torch.zeros((64, 64), dtype=torch.uint8, device="cuda")
    pgg.pgg_set_variant(pgg.VARIANT_RING)
    with pytest.raises(pgg.PggError):
        pgg.pgg_pd_sweep(d, pgg.FMT_U8, 64, *WEAK, 0.1, 1, pgg.ORDER_IID, 0, 1)
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)
    with pytest.raises(pgg.PggError):
        pgg.pgg_pd_sweep(d, pgg.FMT_U8, 64, *WEAK, 0.1, 1, pgg.ORDER_DTILE, 0, 1)

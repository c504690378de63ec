"""CPU-side checks of the product library: it loads, exports every symbol that
include/pgg.h declares, validates its arguments, and its host acceptance-table
builder agrees with the oracle's independently written one (step a6; SURVEY.md
section 8(c) D3, S6).  No kernel is launched here."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

import oracle as orc
import paper_1704_08098_b200 as pgg
from paper_1704_08098_b200 import build as pgg_build

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module", autouse=True)
def _built():
    pgg_build.build()


def test_library_exports_every_declared_symbol():
    header = (ROOT / "include" / "pgg.h").read_text()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(pgg_[a-z0-9_]+)\s*\(", header))
    assert {"pgg_init_lattice", "pgg_build_accept_table", "pgg_sweep", "pgg_density",
            "pgg_run_ensemble"} <= declared
    h = C.CDLL(str(pgg.LIB_PATH))
    for name in declared:
        assert hasattr(h, name), f"{name} declared in pgg.h but not exported"
    assert declared == set(pgg.SIGNATURES), "binding and header disagree on the symbol list"


def test_accept_tables_equal_oracle_tables():
    """North_star: 'the GPU side and the oracle each compute [the table] independently,
    and the two tables are checked equal'."""
    import workloads as wl
    rs = set(wl.config2_rs()) | set(wl.config4().rs) | {3.8, 3.98, 4.0, 3.7443, 1.0, 5.0, 25.0, 0.01}
    for r in sorted(rs):
        for K in (0.5, 0.1, 2.0, 1e-3, 100.0):
            mine = np.array(pgg.pgg_build_accept_table(r, K), dtype=np.uint32)
            assert np.array_equal(mine, orc.accept_table(r, K)), (r, K)


def test_accept_table_paper_limits():
    """equal payoffs -> 1/2; large K -> coin flip; small K -> step."""
    t = pgg.pgg_build_accept_table(4.0, 0.5)
    assert t[51 + 25] == 0x80000000
    t = pgg.pgg_build_accept_table(4.0, 1e9)
    assert all(abs(v - 2**31) < 2**8 for v in t)
    t = pgg.pgg_build_accept_table(4.0, 1e-6)
    assert t[0 * 51 + 25 - 3] == 0 and t[2 * 51 + 25 + 3] == 0xFFFFFFFF  # Pi_x > Pi_y / Pi_x < Pi_y


def test_argument_validation_returns_error_codes():
    h = pgg.lib()
    out = (C.c_uint32 * 153)()
    assert h.pgg_build_accept_table(4.0, 0.0, out) == pgg.ERR_BAD_PARAM
    assert h.pgg_build_accept_table(float("nan"), 0.5, out) == pgg.ERR_BAD_PARAM
    assert h.pgg_build_accept_table(4.0, 0.5, None) == pgg.ERR_NULL
    assert h.pgg_init_lattice(None, 0, 64, 0.5, 1, None) == pgg.ERR_NULL
    fake = 0x1000  # never dereferenced: all of these fail validation first
    assert h.pgg_init_lattice(fake, 0, 6, 0.5, 1, None) == pgg.ERR_BAD_L
    assert h.pgg_init_lattice(fake, 0, 0, 0.5, 1, None) == pgg.ERR_BAD_L
    assert h.pgg_init_lattice(fake, 1, 48, 0.5, 1, None) == pgg.ERR_BAD_L       # bits: L % 32
    assert h.pgg_init_lattice(fake, 7, 64, 0.5, 1, None) == pgg.ERR_UNSUPPORTED
    assert h.pgg_init_lattice(fake + 4, 0, 64, 0.5, 1, None) == pgg.ERR_ALIGN
    assert h.pgg_init_lattice(fake, 0, 64, 1.5, 1, None) == pgg.ERR_BAD_PARAM
    assert h.pgg_sweep(fake, 0, 64, 4.0, -1.0, 1, 0, 0, 1, None, None) == pgg.ERR_BAD_PARAM
    assert h.pgg_sweep(fake, 0, 64, float("inf"), 0.5, 1, 0, 0, 1, None, None) == pgg.ERR_BAD_PARAM
    assert h.pgg_sweep(fake, 0, 64, 4.0, 0.5, 1, 9, 0, 1, None, None) == pgg.ERR_UNSUPPORTED
    assert h.pgg_sweep(fake, 0, 64, 4.0, 0.5, 1, 0, 2**32 - 1, 2, None, None) == pgg.ERR_BAD_PARAM
    assert h.pgg_density(fake, 0, 64, None, None) == pgg.ERR_NULL
    # one rule for the upper end (include/pgg.h): site indices are uint32, so L <= 65532 everywhere
    cnt = C.c_uint64(0)
    for L_bad in (65536, 65540):
        assert h.pgg_init_lattice(fake, 0, L_bad, 0.5, 1, None) == pgg.ERR_BAD_L
        assert h.pgg_sweep(fake, 0, L_bad, 4.0, 0.5, 1, 0, 0, 1, None, None) == pgg.ERR_BAD_L
        assert h.pgg_density(fake, 0, L_bad, C.byref(cnt), None) == pgg.ERR_BAD_L
        assert not pgg.pgg_variant_supported(pgg.VARIANT_V0, pgg.FMT_U8, L_bad)
    assert h.pgg_probe_draw_rate(0, 1, C.byref(cnt), None) == pgg.ERR_BAD_PARAM
    assert h.pgg_probe_draw_rate(4, 1, None, None) == pgg.ERR_NULL
    # the paper's double-tiling schedule needs L % 8 == 0 and has no phase classes
    assert h.pgg_sweep(fake, 0, 12, 4.0, 0.5, 1, pgg.ORDER_DTILE, 0, 1, None, None) == pgg.ERR_BAD_L
    assert h.pgg_sweep(fake, 0, 64, 4.0, 0.0, 1, pgg.ORDER_DTILE, 0, 1, None, None) == pgg.ERR_BAD_PARAM
    assert h.pgg_set_variant(10) == pgg.ERR_UNSUPPORTED  # PGG_VARIANT_DTILE is reported, not selectable
    r = (C.c_double * 1)(4.0)
    s = (C.c_uint64 * 1)(1)
    assert h.pgg_run_ensemble(fake, 0, 0, 64, r, 0.5, s, 0, 0.5, 0, 1, None, None) == pgg.ERR_BAD_PARAM
    assert h.pgg_run_ensemble(fake, 0, 1, 64, None, 0.5, s, 0, 0.5, 0, 1, None, None) == pgg.ERR_NULL
    assert h.pgg_set_variant(99) == pgg.ERR_UNSUPPORTED
    assert b"variant" in h.pgg_last_error()
    # pgg_sweep_static: pgg_sweep's checks, its own limit (PGG_STATIC_MAX_MCS), no double-tiling schedule; all of
    # them before the first CUDA call, and n_mcs == 0 is a no-op that touches nothing
    assert h.pgg_sweep_static(None, 0, 64, 4.0, 0.5, 1, 0, 0, 1, None, None) == pgg.ERR_NULL
    assert h.pgg_sweep_static(fake, 0, 6, 4.0, 0.5, 1, 0, 0, 1, None, None) == pgg.ERR_BAD_L
    assert h.pgg_sweep_static(fake + 4, 0, 64, 4.0, 0.5, 1, 0, 0, 1, None, None) == pgg.ERR_ALIGN
    assert h.pgg_sweep_static(fake, 0, 64, 4.0, 0.0, 1, 0, 0, 1, None, None) == pgg.ERR_BAD_PARAM
    assert h.pgg_sweep_static(fake, 0, 64, float("nan"), 0.5, 1, 0, 0, 1, None, None) == pgg.ERR_BAD_PARAM
    assert h.pgg_sweep_static(fake, 0, 64, 4.0, 0.5, 1, 0, 2**32 - 1, 2, None, None) == pgg.ERR_BAD_PARAM
    assert h.pgg_sweep_static(fake, 0, 64, 4.0, 0.5, 1, pgg.ORDER_DTILE, 0, 1, None, None) == pgg.ERR_UNSUPPORTED
    assert h.pgg_sweep_static(fake, 0, 64, 4.0, 0.5, 1, 9, 0, 1, None, None) == pgg.ERR_UNSUPPORTED
    assert h.pgg_sweep_static(fake, 0, 64, 4.0, 0.5, 1, 0, 0, pgg.STATIC_MAX_MCS + 1, None, None) == pgg.ERR_BAD_PARAM
    assert b"PGG_STATIC_MAX_MCS" in h.pgg_last_error()
    assert h.pgg_sweep_static(fake, 0, 64, 4.0, 0.5, 1, 0, 0, 0, None, None) == pgg.OK
    with pytest.raises(pgg.PggError):
        pgg.pgg_build_accept_table(4.0, -1.0)


def test_product_does_not_import_the_oracle():
    """The CUDA path and the oracle share no code and neither imports the other."""
    for p in (ROOT / "paper_1704_08098_b200").rglob("*"):
        if p.suffix in {".py", ".cu", ".cuh", ".h"}:
            text = p.read_text()
            assert "oracle" not in re.sub(r"(#|//).*", "", text), p
    for p in (ROOT / "oracle").glob("*"):
        if p.suffix in {".py", ".c"}:
            assert "import paper_1704_08098_b200" not in p.read_text()
            assert "pgg.h" not in p.read_text()


def test_variant_support_table():
    """pgg_variant_supported is pure host logic: which kernel may run which (fmt, L)."""
    sup = pgg.pgg_variant_supported
    for L in (4, 20, 64, 400, 512, 2048, 16384):
        assert sup(pgg.VARIANT_AUTO, pgg.FMT_U8, L) and sup(pgg.VARIANT_V0, pgg.FMT_U8, L)
    assert not sup(pgg.VARIANT_V0, pgg.FMT_U8, 6) and not sup(pgg.VARIANT_V0, pgg.FMT_BITS, 48)
    # smem-resident kernel: 8 <= L <= 512 (bit-packed: L % 32 == 0)
    assert sup(pgg.VARIANT_RESIDENT, pgg.FMT_U8, 8) and sup(pgg.VARIANT_RESIDENT, pgg.FMT_U8, 400)
    assert sup(pgg.VARIANT_RESIDENT, pgg.FMT_U8, 512) and sup(pgg.VARIANT_RESIDENT, pgg.FMT_BITS, 512)
    assert not sup(pgg.VARIANT_RESIDENT, pgg.FMT_U8, 4) and not sup(pgg.VARIANT_RESIDENT, pgg.FMT_U8, 516)
    # streaming kernels need rows of whole 16-byte units
    assert sup(pgg.VARIANT_RING, pgg.FMT_U8, 400) and not sup(pgg.VARIANT_RING, pgg.FMT_U8, 100)
    assert sup(pgg.VARIANT_BAND, pgg.FMT_BITS, 16384) and not sup(pgg.VARIANT_BAND, pgg.FMT_BITS, 160)
    # SPLIT and DYN are uint8 only
    assert sup(pgg.VARIANT_SPLIT, pgg.FMT_U8, 2048) and not sup(pgg.VARIANT_SPLIT, pgg.FMT_BITS, 2048)
    assert sup(pgg.VARIANT_DYN, pgg.FMT_U8, 2048) and not sup(pgg.VARIANT_DYN, pgg.FMT_BITS, 2048)
    # PACKED is uint8 in HBM with a bit-packed working copy for LEAN: LEAN's sizes, uint8 only
    assert sup(pgg.VARIANT_PACKED, pgg.FMT_U8, 1024) and sup(pgg.VARIANT_PACKED, pgg.FMT_U8, 32768)
    assert not sup(pgg.VARIANT_PACKED, pgg.FMT_BITS, 1024) and not sup(pgg.VARIANT_PACKED, pgg.FMT_U8, 512)
    assert not sup(pgg.VARIANT_PACKED, pgg.FMT_U8, 3072)
    assert not sup(99, pgg.FMT_U8, 64)


def test_prisoners_dilemma_tables_equal_oracle_tables_and_validation():
    """The library's 50 thresholds of the prisoner's dilemma (G3) against the oracle's,
    built independently; argument validation of the two entry points (no GPU needed: all fail first)."""
    import oracle as orc
    for (R, S, T, P, K) in ((1.0, 0.0, 1.3, 0.0, 0.1), (3.0, -0.5, 4.25, 0.75, 0.5), (1.0, 0.0, 2.0, 0.0, 1e-3),
                            (1.0, 0.0, 1.0, 0.0, 50.0)):
        assert pgg.pgg_pd_build_accept_table(R, S, T, P, K) == orc.pd_accept_table(R, S, T, P, K).tolist()
    h = pgg.lib()
    out = (C.c_uint32 * 50)()
    assert h.pgg_pd_build_accept_table(1.0, 0.0, 1.3, 0.0, 0.0, out) == pgg.ERR_BAD_PARAM
    assert h.pgg_pd_build_accept_table(float("nan"), 0.0, 1.3, 0.0, 0.1, out) == pgg.ERR_BAD_PARAM
    assert h.pgg_pd_build_accept_table(1.0, 0.0, 1.3, 0.0, 0.1, None) == pgg.ERR_NULL
    fake = 0x1000
    args = (1.0, 0.0, 1.3, 0.0, 0.1, 1)
    assert h.pgg_pd_sweep(None, 0, 64, *args, 0, 0, 1, None, None) == pgg.ERR_NULL
    assert h.pgg_pd_sweep(fake, 0, 6, *args, 0, 0, 1, None, None) == pgg.ERR_BAD_L
    assert h.pgg_pd_sweep(fake, 0, 64, 1.0, 0.0, float("inf"), 0.0, 0.1, 1, 0, 0, 1, None, None) == pgg.ERR_BAD_PARAM
    assert h.pgg_pd_sweep(fake, 0, 64, 1.0, 0.0, 1.3, 0.0, -1.0, 1, 0, 0, 1, None, None) == pgg.ERR_BAD_PARAM
    assert h.pgg_pd_sweep(fake, 0, 64, *args, pgg.ORDER_DTILE, 0, 1, None, None) == pgg.ERR_UNSUPPORTED

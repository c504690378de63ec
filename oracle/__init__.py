"""ctypes front-end of the CPU oracle (``oracle/pgg_oracle.c``).

TEST INFRASTRUCTURE ONLY: importable from ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs.  Nothing under
``paper_1704_08098_b200/`` imports this package and this package imports nothing
from there.  This module only marshals numpy arrays into the C functions; every
step of the method is in the C file, which cites PAPER.md for each function.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "pgg_oracle.c"
_SRC_PD = _HERE / "pd_oracle.c"   # the prisoner's dilemma, same library
_LIB = _HERE / "liboracle_pgg.so"

ORDER_IID = 0
ORDER_PERM = 1
ORDER_DTILE = 2  # the paper's double-tiling schedule


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O2, OpenMP for the optional row split)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < max(_SRC.stat().st_mtime, _SRC_PD.stat().st_mtime):
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp.so")
        cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-o", str(tmp), str(_SRC), str(_SRC_PD), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        u8p, u32p, u64p = C.POINTER(C.c_uint8), C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)
        L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.orc_philox4x32_10.restype = None
        L.orc_group_count.argtypes = [u8p, C.c_int, C.c_int, C.c_int]
        L.orc_group_count.restype = C.c_int
        L.orc_payoff_literal.argtypes = [u8p, C.c_int, C.c_int, C.c_int, C.c_double]
        L.orc_payoff_literal.restype = C.c_double
        L.orc_A.argtypes = [u8p, C.c_int, C.c_int, C.c_int]
        L.orc_A.restype = C.c_int
        L.orc_fermi.argtypes = [C.c_double, C.c_double, C.c_double]
        L.orc_fermi.restype = C.c_double
        L.orc_table_index.argtypes = [C.c_int, C.c_int]
        L.orc_table_index.restype = C.c_int
        L.orc_accept_table.argtypes = [C.c_double, C.c_double, u32p]
        L.orc_accept_table.restype = None
        L.orc_init.argtypes = [u8p, C.c_int, C.c_double, C.c_uint64]
        L.orc_init.restype = None
        L.orc_count.argtypes = [u8p, C.c_int]
        L.orc_count.restype = C.c_uint64
        L.orc_phase_classes.argtypes = [C.c_uint64, C.c_uint32, C.c_int, u8p]
        L.orc_phase_classes.restype = None
        L.orc_step_given_draw.argtypes = [u8p, C.c_int, u32p, C.c_int, C.c_int, C.c_int, C.c_uint32]
        L.orc_step_given_draw.restype = C.c_int
        L.orc_flip_threshold.argtypes = [u8p, C.c_int, u32p, C.c_int, C.c_int, C.c_int]
        L.orc_flip_threshold.restype = C.c_uint32
        L.orc_flip_thresholds_batch.argtypes = [u8p, C.c_int, C.c_int, u32p, u32p]
        L.orc_flip_thresholds_batch.restype = None
        L.orc_step_draw.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32,
                                    C.POINTER(C.c_int), u32p]
        L.orc_step_draw.restype = None
        L.orc_phase.argtypes = [u8p, C.c_int, u32p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32,
                                C.c_int, u32p, C.c_int]
        L.orc_phase.restype = C.c_int64
        L.orc_dtile_type.argtypes = [C.c_int, C.c_int]
        L.orc_dtile_type.restype = C.c_int
        L.orc_dtile_draw.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32,
                                     C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int), u32p]
        L.orc_dtile_draw.restype = None
        L.orc_dtile_part.argtypes = [u8p, C.c_int, u32p, C.c_uint64, C.c_uint32, C.c_int, C.c_int,
                                     C.c_int]
        L.orc_dtile_part.restype = C.c_int64
        L.orc_sweep.argtypes = [u8p, C.c_int, C.c_double, C.c_double, C.c_uint64, C.c_int,
                                C.c_uint32, C.c_uint32, u64p, C.c_uint32, u8p, C.c_int]
        L.orc_sweep.restype = C.c_int
        L.orc_rs_sweep.argtypes = [u8p, C.c_int, C.c_double, C.c_double, C.c_uint64, C.c_uint64,
                                   C.c_uint32, u64p]
        L.orc_rs_sweep.restype = C.c_int
        L.orc_pack_bits.argtypes = [u8p, C.c_int, u32p]
        L.orc_pack_bits.restype = None
        L.orc_unpack_bits.argtypes = [u32p, C.c_int, u8p]
        L.orc_unpack_bits.restype = None
        L.orc_max_threads.argtypes = []
        L.orc_max_threads.restype = C.c_int
        d4 = [C.c_double] * 4
        L.orc_pd_payoff_literal.argtypes = [u8p, C.c_int, C.c_int, C.c_int] + d4
        L.orc_pd_payoff_literal.restype = C.c_double
        L.orc_pd_nc.argtypes = [u8p, C.c_int, C.c_int, C.c_int]
        L.orc_pd_nc.restype = C.c_int
        L.orc_pd_payoff.argtypes = [C.c_int, C.c_int] + d4
        L.orc_pd_payoff.restype = C.c_double
        L.orc_pd_table_index.argtypes = [C.c_int, C.c_int, C.c_int]
        L.orc_pd_table_index.restype = C.c_int
        L.orc_pd_accept_table.argtypes = d4 + [C.c_double, u32p]
        L.orc_pd_accept_table.restype = None
        L.orc_pd_flip_threshold.argtypes = [u8p, C.c_int, u32p, C.c_int, C.c_int, C.c_int]
        L.orc_pd_flip_threshold.restype = C.c_uint32
        L.orc_pd_step_given_draw.argtypes = [u8p, C.c_int, u32p, C.c_int, C.c_int, C.c_int, C.c_uint32]
        L.orc_pd_step_given_draw.restype = C.c_int
        L.orc_pd_phase.argtypes = [u8p, C.c_int, u32p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_int]
        L.orc_pd_phase.restype = C.c_int64
        L.orc_pd_sweep.argtypes = [u8p, C.c_int] + d4 + [C.c_double, C.c_uint64, C.c_int, C.c_uint32, C.c_uint32, u64p]
        L.orc_pd_sweep.restype = C.c_int
        _lib = L
    return _lib


def _u8(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint8))


def _u32(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint32))


def _u64(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint64))


def _lat(a) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.uint8)
    assert a.ndim == 2 and a.shape[0] == a.shape[1], "lattice must be L x L"
    return a


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_u32(c), _u32(k), _u32(out))
    return out


def group_count(lat, i, j) -> int:
    lat = _lat(lat)
    return lib().orc_group_count(_u8(lat), lat.shape[0], i, j)


def payoff_literal(lat, i, j, r) -> float:
    lat = _lat(lat)
    return lib().orc_payoff_literal(_u8(lat), lat.shape[0], i, j, r)


def A(lat, i, j) -> int:
    lat = _lat(lat)
    return lib().orc_A(_u8(lat), lat.shape[0], i, j)


def fermi(Pi_x, Pi_y, K) -> float:
    return lib().orc_fermi(Pi_x, Pi_y, K)


def table_index(dA, ds) -> int:
    return lib().orc_table_index(dA, ds)


def accept_table(r, K) -> np.ndarray:
    out = np.zeros(153, dtype=np.uint32)
    lib().orc_accept_table(r, K, _u32(out))
    return out


def init(L, rho0, seed) -> np.ndarray:
    lat = np.zeros((L, L), dtype=np.uint8)
    lib().orc_init(_u8(lat), L, rho0, seed)
    return lat


def count(lat) -> int:
    lat = _lat(lat)
    return int(lib().orc_count(_u8(lat), lat.shape[0]))


def phase_classes(seed, t, order_mode=ORDER_IID) -> np.ndarray:
    out = np.zeros(16, dtype=np.uint8)
    lib().orc_phase_classes(seed, t, order_mode, _u8(out))
    return out


def step_given_draw(lat, table, i, j, direction, u) -> int:
    lat = _lat(lat)
    table = np.ascontiguousarray(table, dtype=np.uint32)
    return lib().orc_step_given_draw(_u8(lat), lat.shape[0], _u32(table), i, j, direction, u)


def flip_threshold(lat, table, i, j, direction) -> int:
    lat = _lat(lat)
    table = np.ascontiguousarray(table, dtype=np.uint32)
    return int(lib().orc_flip_threshold(_u8(lat), lat.shape[0], _u32(table), i, j, direction))


def flip_thresholds_batch(lats, table) -> np.ndarray:
    """lats: [n, L, L] uint8 -> thresholds [n, L, L, 4] uint32."""
    lats = np.ascontiguousarray(lats, dtype=np.uint8)
    n, L, _ = lats.shape
    table = np.ascontiguousarray(table, dtype=np.uint32)
    out = np.zeros((n, L, L, 4), dtype=np.uint32)
    lib().orc_flip_thresholds_batch(_u8(lats), n, L, _u32(table), _u32(out))
    return out


def step_draw(seed, site, t, k, c):
    d = C.c_int(0)
    u = np.zeros(1, dtype=np.uint32)
    lib().orc_step_draw(seed, site, t, k, c, C.byref(d), _u32(u))
    return d.value, int(u[0])


def phase(lat, table, seed, t, k, c, visit=0, perm=None, n_threads=1) -> int:
    """In-place phase on ``lat`` (must be a C-contiguous uint8 array); returns count delta."""
    assert lat.dtype == np.uint8 and lat.flags.c_contiguous
    table = np.ascontiguousarray(table, dtype=np.uint32)
    p = None
    if perm is not None:
        perm = np.ascontiguousarray(perm, dtype=np.uint32)
        p = _u32(perm)
    return int(lib().orc_phase(_u8(lat), lat.shape[0], _u32(table), seed, t, k, c, visit, p,
                               n_threads))


def dtile_type(I, J) -> int:
    return int(lib().orc_dtile_type(I, J))


def dtile_draw(seed, d, t, p):
    """(domain row, domain column, direction, u) of pick p of domain d in MCS t."""
    a, b, di = C.c_int(0), C.c_int(0), C.c_int(0)
    u = np.zeros(1, dtype=np.uint32)
    lib().orc_dtile_draw(seed, d, t, p, C.byref(a), C.byref(b), C.byref(di), _u32(u))
    return a.value, b.value, di.value, int(u[0])


def dtile_part(lat, table, seed, t, q, visit=0, n_threads=1) -> int:
    """In-place part q (domains of type q) of MCS t of the double-tiling schedule; count delta."""
    assert lat.dtype == np.uint8 and lat.flags.c_contiguous and lat.shape[0] % 8 == 0
    table = np.ascontiguousarray(table, dtype=np.uint32)
    return int(lib().orc_dtile_part(_u8(lat), lat.shape[0], _u32(table), seed, t, q, visit,
                                    n_threads))


def sweep(lat, r, K, seed, order_mode=ORDER_IID, t_begin=0, n_mcs=1, snap_every=0, n_threads=1):
    """In-place sweep; returns (counts[n_mcs] uint64, snaps[n_snap, L, L] uint8)."""
    assert lat.dtype == np.uint8 and lat.flags.c_contiguous
    L = lat.shape[0]
    counts = np.zeros(max(n_mcs, 1), dtype=np.uint64)
    n_snap = n_mcs // snap_every if snap_every else 0
    snaps = np.zeros((max(n_snap, 1), L, L), dtype=np.uint8)
    rc = lib().orc_sweep(_u8(lat), L, r, K, seed, order_mode, t_begin, n_mcs, _u64(counts),
                         snap_every, _u8(snaps), n_threads)
    if rc != 0:
        raise ValueError("orc_sweep: bad arguments")
    return counts[:n_mcs], snaps[:n_snap]


def rs_sweep(lat, r, K, seed, g_begin=0, n_mcs=1):
    assert lat.dtype == np.uint8 and lat.flags.c_contiguous
    counts = np.zeros(max(n_mcs, 1), dtype=np.uint64)
    rc = lib().orc_rs_sweep(_u8(lat), lat.shape[0], r, K, seed, g_begin, n_mcs, _u64(counts))
    if rc != 0:
        raise ValueError("orc_rs_sweep: bad arguments")
    return counts[:n_mcs]


def pack_bits(lat) -> np.ndarray:
    lat = _lat(lat)
    L = lat.shape[0]
    assert L % 32 == 0
    w = np.zeros((L, L // 32), dtype=np.uint32)
    lib().orc_pack_bits(_u8(lat), L, _u32(w))
    return w


def unpack_bits(words, L) -> np.ndarray:
    words = np.ascontiguousarray(words, dtype=np.uint32)
    lat = np.zeros((L, L), dtype=np.uint8)
    lib().orc_unpack_bits(_u32(words), L, _u8(lat))
    return lat


def max_threads() -> int:
    return lib().orc_max_threads()


# ---------------------------------------------------------------- prisoner's dilemma (pd_oracle.c)
def pd_payoff_literal(lat, i, j, R, S, T, P) -> float:
    lat = _lat(lat)
    return float(lib().orc_pd_payoff_literal(_u8(lat), lat.shape[0], i, j, R, S, T, P))


def pd_nc(lat, i, j) -> int:
    lat = _lat(lat)
    return lib().orc_pd_nc(_u8(lat), lat.shape[0], i, j)


def pd_payoff(s, n, R, S, T, P) -> float:
    return float(lib().orc_pd_payoff(s, n, R, S, T, P))


def pd_table_index(sx, nx, ny) -> int:
    return lib().orc_pd_table_index(sx, nx, ny)


def pd_accept_table(R, S, T, P, K) -> np.ndarray:
    out = np.zeros(50, dtype=np.uint32)
    lib().orc_pd_accept_table(R, S, T, P, K, _u32(out))
    return out


def pd_flip_threshold(lat, table, i, j, direction) -> int:
    lat = _lat(lat)
    table = np.ascontiguousarray(table, dtype=np.uint32)
    return int(lib().orc_pd_flip_threshold(_u8(lat), lat.shape[0], _u32(table), i, j, direction))


def pd_step_given_draw(lat, table, i, j, direction, u) -> int:
    lat = _lat(lat)
    table = np.ascontiguousarray(table, dtype=np.uint32)
    return lib().orc_pd_step_given_draw(_u8(lat), lat.shape[0], _u32(table), i, j, direction, u)


def pd_phase(lat, table, seed, t, k, c, visit=0) -> int:
    assert lat.dtype == np.uint8 and lat.flags.c_contiguous
    table = np.ascontiguousarray(table, dtype=np.uint32)
    return int(lib().orc_pd_phase(_u8(lat), lat.shape[0], _u32(table), seed, t, k, c, visit))


def pd_sweep(lat, R, S, T, P, K, seed, order_mode=ORDER_IID, t_begin=0, n_mcs=1):
    """In-place prisoner's-dilemma sweep under the 16-sublattice schedule; returns counts[n_mcs]."""
    assert lat.dtype == np.uint8 and lat.flags.c_contiguous
    counts = np.zeros(max(n_mcs, 1), dtype=np.uint64)
    rc = lib().orc_pd_sweep(_u8(lat), lat.shape[0], R, S, T, P, K, seed, order_mode, t_begin, n_mcs, _u64(counts))
    if rc != 0:
        raise ValueError("orc_pd_sweep: bad arguments")
    return counts[:n_mcs]

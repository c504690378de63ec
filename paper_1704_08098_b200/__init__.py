"""paper_1704_08098_b200 -- thin Python binding of libpgg (include/pgg.h).

Argument marshalling only: every step of the method (initial condition, phase-class
draw, Philox draws, payoff differences, Fermi acceptance, density) runs in the CUDA
kernels of ``libpgg.so``.  PyTorch is used for device memory and streams.  There is
no CPU fallback: if the shared library is missing or a call fails, this raises.

Functions have the names and argument order of the C ABI.  Lattices are torch
tensors on a CUDA device: ``uint8 [.., L, L]`` for ``FMT_U8`` and
``int32 [.., L, L/32]`` for ``FMT_BITS`` (bit ``j & 31`` of word ``j >> 5``).
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libpgg.so"

OK = 0
ERR_NULL, ERR_BAD_L, ERR_BAD_PARAM, ERR_ALIGN, ERR_UNSUPPORTED, ERR_CUDA = -1, -2, -3, -4, -5, -6
FMT_U8, FMT_BITS = 0, 1
ORDER_IID, ORDER_PERM, ORDER_DTILE = 0, 1, 2
VARIANT_AUTO, VARIANT_V0, VARIANT_TILE = 0, 1, 2
VARIANT_PIPE, VARIANT_BAND, VARIANT_RING, VARIANT_SPLIT, VARIANT_DYN, VARIANT_RESIDENT = 4, 5, 6, 7, 8, 9
VARIANT_DTILE, VARIANT_LEAN, VARIANT_PERSIST, VARIANT_CLUSTER, VARIANT_PACKED = 10, 11, 12, 13, 14

# name -> (restype, argtypes); also the list of symbols include/pgg.h declares
_u32p, _u64p, _u8p, _f64p = (C.POINTER(C.c_uint32), C.POINTER(C.c_uint64), C.POINTER(C.c_uint8),
                             C.POINTER(C.c_double))
SIGNATURES = {
    "pgg_build_accept_table": (C.c_int32, [C.c_double, C.c_double, _u32p]),
    "pgg_init_lattice": (C.c_int32, [C.c_void_p, C.c_int32, C.c_uint32, C.c_double, C.c_uint64,
                                     C.c_void_p]),
    "pgg_sweep": (C.c_int32, [C.c_void_p, C.c_int32, C.c_uint32, C.c_double, C.c_double, C.c_uint64,
                              C.c_int32, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p]),
    "pgg_sweep_static": (C.c_int32, [C.c_void_p, C.c_int32, C.c_uint32, C.c_double, C.c_double, C.c_uint64,
                                     C.c_int32, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p]),
    "pgg_density": (C.c_int32, [C.c_void_p, C.c_int32, C.c_uint32, C.c_void_p, C.c_void_p]),
    "pgg_run_ensemble": (C.c_int32, [C.c_void_p, C.c_int32, C.c_uint32, C.c_uint32, _f64p, C.c_double,
                                     _u64p, C.c_int32, C.c_double, C.c_uint32, C.c_uint32, C.c_void_p,
                                     C.c_void_p]),
    "pgg_pd_build_accept_table": (C.c_int32, [C.c_double] * 5 + [_u32p]),
    "pgg_pd_sweep": (C.c_int32, [C.c_void_p, C.c_int32, C.c_uint32] + [C.c_double] * 5 +
                     [C.c_uint64, C.c_int32, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p]),
    "pgg_slab_bytes": (C.c_uint64, [C.c_int32, C.c_uint32, C.c_uint32]),
    "pgg_slab_step_rows": (C.c_uint32, [C.c_int32, C.c_uint32]),
    "pgg_slab_sweep": (C.c_int32, [C.c_void_p, C.c_int32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_double, C.c_double,
                                   C.c_uint64, C.c_int32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p,
                                   C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p]),
    "pgg_pd_slab_sweep": (C.c_int32, [C.c_void_p, C.c_int32, C.c_uint32, C.c_uint32, C.c_uint32] + [C.c_double] * 5 +
                          [C.c_uint64, C.c_int32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p,
                           C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p]),
    "pgg_slab_alloc": (C.c_int32, [C.c_uint64, C.POINTER(C.c_void_p)]),
    "pgg_slab_free": (C.c_int32, [C.c_void_p]),
    "pgg_slab_ipc_export": (C.c_int32, [C.c_void_p, _u8p]),
    "pgg_slab_ipc_open": (C.c_int32, [_u8p, C.c_int32, C.POINTER(C.c_void_p)]),
    "pgg_slab_ipc_close": (C.c_int32, [C.c_void_p]),
    "pgg_phase_classes": (C.c_int32, [C.c_uint64, C.c_uint32, C.c_int32, _u8p, C.c_void_p]),
    "pgg_set_variant": (C.c_int32, [C.c_int32]),
    "pgg_get_variant_used": (C.c_int32, []),
    "pgg_variant_supported": (C.c_int32, [C.c_int32, C.c_int32, C.c_uint32]),
    "pgg_probe_draw_rate": (C.c_int32, [C.c_uint32, C.c_uint64, _u64p, C.c_void_p]),
    "pgg_count_interface": (C.c_int32, [C.c_void_p, C.c_int32, C.c_uint32, C.c_void_p, C.c_void_p]),
    "pgg_trim_workspace": (C.c_int32, []),
    "pgg_launch_count": (C.c_uint64, []),
    "pgg_last_error": (C.c_char_p, []),
}


class PggError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"libpgg error {code}: {text}")
        self.code = code


_lib = None


def lib() -> C.CDLL:
    """Load libpgg.so (built in-tree by ``python -m paper_1704_08098_b200.build``)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1704_08098_b200.build` "
                              "(there is no CPU fallback)")
        h = C.CDLL(str(LIB_PATH))
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(h, name)
            fn.restype, fn.argtypes = res, args
        _lib = h
    return _lib


def _check(rc: int) -> None:
    if rc != OK:
        raise PggError(rc, lib().pgg_last_error().decode())


def _stream(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


def _ptr(t) -> int:
    """Device address: a tensor, an int (an address from pgg_slab_alloc / pgg_slab_ipc_open) or None."""
    return 0 if t is None else t if isinstance(t, int) else t.data_ptr()


def pgg_build_accept_table(r: float, K: float):
    """-> list of 153 thresholds (host function, no CUDA)."""
    out = (C.c_uint32 * 153)()
    _check(lib().pgg_build_accept_table(r, K, out))
    return list(out)


def pgg_init_lattice(d_lat, fmt: int, L: int, rho0: float, seed: int, stream=None) -> None:
    _check(lib().pgg_init_lattice(_ptr(d_lat), fmt, L, rho0, seed, _stream(stream)))


def pgg_sweep(d_lat, fmt: int, L: int, r: float, K: float, seed: int, order_mode: int, t_begin: int,
              n_mcs: int, d_counts=None, stream=None) -> None:
    _check(lib().pgg_sweep(_ptr(d_lat), fmt, L, r, K, seed, order_mode, t_begin, n_mcs, _ptr(d_counts),
                           _stream(stream)))


STATIC_MAX_MCS = 4096  # PGG_STATIC_MAX_MCS


def pgg_sweep_static(d_lat, fmt: int, L: int, r: float, K: float, seed: int, order_mode: int, t_begin: int,
                     n_mcs: int, d_counts=None, stream=None) -> None:
    """pgg_sweep without any device allocation (temporaries in the library's static device array);
    n_mcs <= STATIC_MAX_MCS per call, calls that overlap on the GPU race (include/pgg.h)."""
    _check(lib().pgg_sweep_static(_ptr(d_lat), fmt, L, r, K, seed, order_mode, t_begin, n_mcs, _ptr(d_counts),
                                  _stream(stream)))


def pgg_density(d_lat, fmt: int, L: int, d_count, stream=None) -> None:
    _check(lib().pgg_density(_ptr(d_lat), fmt, L, _ptr(d_count), _stream(stream)))


def pgg_run_ensemble(d_lats, fmt: int, B: int, L: int, h_r, K: float, h_seeds, order_mode: int,
                     rho0: float, t_begin: int, n_mcs: int, d_counts=None, stream=None) -> None:
    r = (C.c_double * B)(*[float(x) for x in h_r])
    s = (C.c_uint64 * B)(*[int(x) for x in h_seeds])
    _check(lib().pgg_run_ensemble(_ptr(d_lats), fmt, B, L, r, K, s, order_mode, rho0, t_begin, n_mcs,
                                  _ptr(d_counts), _stream(stream)))


def pgg_pd_build_accept_table(R: float, S: float, T: float, P: float, K: float):
    """-> list of 50 thresholds of the prisoner's dilemma (host function, no CUDA)."""
    out = (C.c_uint32 * 50)()
    _check(lib().pgg_pd_build_accept_table(R, S, T, P, K, out))
    return list(out)


def pgg_pd_sweep(d_lat, fmt: int, L: int, R: float, S: float, T: float, P: float, K: float, seed: int,
                 order_mode: int, t_begin: int, n_mcs: int, d_counts=None, stream=None) -> None:
    _check(lib().pgg_pd_sweep(_ptr(d_lat), fmt, L, R, S, T, P, K, seed, order_mode, t_begin, n_mcs,
                              _ptr(d_counts), _stream(stream)))


SLAB_MAX_MCS = 4096  # PGG_SLAB_MAX_MCS
SLAB_IPC_HANDLE_BYTES = 64


def pgg_slab_bytes(fmt: int, L: int, n_rows: int) -> int:
    return int(lib().pgg_slab_bytes(fmt, L, n_rows))


def pgg_slab_step_rows(fmt: int, L: int) -> int:
    """Row granularity (row0, n_rows) at which a slab runs the fast kernel; needs a CUDA device."""
    return int(lib().pgg_slab_step_rows(fmt, L))


def pgg_slab_sweep(d_slab, fmt: int, L: int, row0: int, n_rows: int, r: float, K: float, seed: int, order_mode: int,
                   t_begin: int, k_begin: int, n_phases: int, d_up_halo, d_dn_halo, d_flags=None, d_up_flag=None,
                   d_dn_flag=None, epoch0: int = 0, d_deltas=None, stream=None) -> None:
    """n_phases phases on one row slab of a sharded lattice (include/pgg.h); pointers are tensors or addresses."""
    _check(lib().pgg_slab_sweep(_ptr(d_slab), fmt, L, row0, n_rows, r, K, seed, order_mode, t_begin, k_begin, n_phases,
                                _ptr(d_up_halo), _ptr(d_dn_halo), _ptr(d_flags), _ptr(d_up_flag), _ptr(d_dn_flag),
                                epoch0, _ptr(d_deltas), _stream(stream)))


def pgg_pd_slab_sweep(d_slab, fmt: int, L: int, row0: int, n_rows: int, R: float, S: float, T: float, P: float, K: float,
                      seed: int, order_mode: int, t_begin: int, k_begin: int, n_phases: int, d_up_halo, d_dn_halo,
                      d_flags=None, d_up_flag=None, d_dn_flag=None, epoch0: int = 0, d_deltas=None, stream=None) -> None:
    """pgg_slab_sweep for the prisoner's dilemma: payoffs (R, S, T, P) in place of r."""
    _check(lib().pgg_pd_slab_sweep(_ptr(d_slab), fmt, L, row0, n_rows, R, S, T, P, K, seed, order_mode, t_begin, k_begin,
                                   n_phases, _ptr(d_up_halo), _ptr(d_dn_halo), _ptr(d_flags), _ptr(d_up_flag),
                                   _ptr(d_dn_flag), epoch0, _ptr(d_deltas), _stream(stream)))


def pgg_slab_alloc(n_bytes: int) -> int:
    """-> device address of a zeroed cudaMalloc allocation of its own (exportable by pgg_slab_ipc_export)."""
    p = C.c_void_p(0)
    _check(lib().pgg_slab_alloc(n_bytes, C.byref(p)))
    return int(p.value)


def pgg_slab_free(d_ptr: int) -> None:
    _check(lib().pgg_slab_free(d_ptr))


def pgg_slab_ipc_export(d_ptr: int) -> bytes:
    h = (C.c_uint8 * SLAB_IPC_HANDLE_BYTES)()
    _check(lib().pgg_slab_ipc_export(d_ptr, h))
    return bytes(h)


def pgg_slab_ipc_open(handle: bytes, peer_device: int = -1) -> int:
    h = (C.c_uint8 * SLAB_IPC_HANDLE_BYTES)(*handle)
    p = C.c_void_p(0)
    _check(lib().pgg_slab_ipc_open(h, peer_device, C.byref(p)))
    return int(p.value)


def pgg_slab_ipc_close(d_ptr: int) -> None:
    _check(lib().pgg_slab_ipc_close(d_ptr))


def pgg_phase_classes(seed: int, t: int, order_mode: int, stream=None):
    out = (C.c_uint8 * 16)()
    _check(lib().pgg_phase_classes(seed, t, order_mode, out, _stream(stream)))
    return list(out)


def pgg_set_variant(variant: int) -> None:
    _check(lib().pgg_set_variant(variant))


def pgg_get_variant_used() -> int:
    return lib().pgg_get_variant_used()


def pgg_variant_supported(variant: int, fmt: int, L: int) -> bool:
    return bool(lib().pgg_variant_supported(variant, fmt, L))


def pgg_probe_draw_rate(iters: int, seed: int = 1, stream=None) -> int:
    """Enqueue one launch of the Philox-only probe; -> number of STEP draws it makes."""
    n = C.c_uint64(0)
    _check(lib().pgg_probe_draw_rate(iters, seed, C.byref(n), _stream(stream)))
    return int(n.value)


def pgg_count_interface(d_lat, fmt: int, L: int, d_count, stream=None) -> None:
    _check(lib().pgg_count_interface(_ptr(d_lat), fmt, L, _ptr(d_count), _stream(stream)))


def pgg_trim_workspace() -> None:
    """Give the unused part of the library's memory pool (current device) back to the driver."""
    _check(lib().pgg_trim_workspace())


def pgg_launch_count() -> int:
    return int(lib().pgg_launch_count())

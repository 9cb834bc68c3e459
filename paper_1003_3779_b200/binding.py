"""Thin ctypes binding over libqw.so — same names as include/qw.h, argument marshalling only.

Every function forwards to the C ABI; buffers may be numpy arrays (host), torch tensors (host,
pinned or CUDA) or raw integer addresses.  Non-zero return codes raise ``QwError`` carrying
``qw_last_error()``.  There is no fallback: if the CUDA library cannot be loaded, ``load()`` raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqw.so")

QW_OK, QW_EINVAL, QW_ENOMEM, QW_ECUDA, QW_ESTATE, QW_EUNSUPPORTED = 0, -1, -2, -3, -4, -5
QW_C64, QW_C128 = 0, 1
QW_PERIODIC, QW_OPEN = 0, 1
QW_NATURAL, QW_DIAGONAL = 0, 1
QW_COIN_UNIFORM, QW_COIN_PER_WALK, QW_COIN_PER_SITE = 0, 1, 2
QW_SCHED_AUTO, QW_SCHED_GENERIC, QW_SCHED_FUSED, QW_SCHED_BLOCKED, QW_SCHED_RESIDENT, QW_SCHED_TILED = 0, 1, 2, 3, 4, 5
QW_INFO_LAUNCHES, QW_INFO_TIME, QW_INFO_LAST_SCHEDULE, QW_INFO_LAST_K, QW_INFO_STATE_BYTES, QW_INFO_WINDOW, \
    QW_INFO_SITES_TOUCHED = range(7)
QW_OPT_MAX_CTAS, QW_OPT_BLOCKED1D_KERNEL, QW_OPT_TILED2D_KERNEL = 0, 1, 2

# every symbol include/qw.h declares (tests/test_abi.py checks the header against this list)
SYMBOLS = (
    "qw_create", "qw_create_batch", "qw_destroy", "qw_set_stream", "qw_set_lattice", "qw_set_coin",
    "qw_set_site_phases", "qw_set_broken_links", "qw_set_random_broken_links", "qw_set_state", "qw_set_state_delta", "qw_get_state",
    "qw_step", "qw_step_inverse", "qw_probabilities", "qw_probabilities_mean", "qw_moments", "qw_moments_static", "qw_set_schedule", "qw_set_window",
    "qw_set_option", "qw_get_info", "qw_measure_alu_peak", "qw_synchronize", "qw_last_error",
)


class QwError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__("libqw error %d: %s" % (code, message))
        self.code = code


_lib = None


def load(path: Optional[str] = None) -> ctypes.CDLL:
    """Load libqw.so (built by paper_1003_3779_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise OSError("%s not found: build the CUDA library first (python -m paper_1003_3779_b200.build); "
                      "there is no CPU fallback" % p)
    lib = ctypes.CDLL(p)
    vp, i64, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
    i64p = ctypes.POINTER(ctypes.c_int64)
    sig = {
        "qw_create": [ci, i64p, ci, ci, ci, ctypes.POINTER(vp)],
        "qw_create_batch": [i64, ci, i64p, ci, ci, ci, ctypes.POINTER(vp)],
        "qw_destroy": [vp],
        "qw_set_stream": [vp, vp],
        "qw_set_lattice": [vp, ci],
        "qw_set_coin": [vp, ci, vp],
        "qw_set_site_phases": [vp, vp],
        "qw_set_broken_links": [vp, vp],
        "qw_set_random_broken_links": [vp, ci, ctypes.c_double, ctypes.c_uint64],
        "qw_set_state": [vp, vp],
        "qw_set_state_delta": [vp, i64p, vp],
        "qw_get_state": [vp, vp],
        "qw_step": [vp, i64],
        "qw_step_inverse": [vp, i64],
        "qw_probabilities": [vp, vp],
        "qw_probabilities_mean": [vp, vp],
        "qw_moments": [vp, vp],
        "qw_moments_static": [vp, vp],
        "qw_set_schedule": [vp, ci, ci],
        "qw_set_window": [vp, ci],
        "qw_set_option": [vp, ci, i64],
        "qw_get_info": [vp, ci, i64p],
        "qw_measure_alu_peak": [ci, ci, ctypes.POINTER(ctypes.c_double)],
        "qw_synchronize": [vp],
    }
    for name, args in sig.items():
        f = getattr(lib, name)
        f.argtypes = args
        f.restype = ci
    lib.qw_last_error.argtypes = []
    lib.qw_last_error.restype = ctypes.c_char_p
    if path is None:
        _lib = lib
    return lib


def _ptr(buf) -> Optional[int]:
    """Address of a numpy array / torch tensor / int; keeps no reference (caller holds the buffer)."""
    if buf is None:
        return None
    if isinstance(buf, int):
        return buf
    if isinstance(buf, np.ndarray):
        if not buf.flags.c_contiguous:
            raise ValueError("buffer must be C-contiguous")
        return buf.ctypes.data
    if hasattr(buf, "data_ptr"):
        if not buf.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return buf.data_ptr()
    raise TypeError("unsupported buffer type %r" % type(buf))


def _check(rc: int) -> None:
    if rc != QW_OK:
        raise QwError(rc, load().qw_last_error().decode("utf-8", "replace"))


def _i64(values: Sequence[int]):
    return (ctypes.c_int64 * len(values))(*[int(v) for v in values])


def qw_last_error() -> str:
    return load().qw_last_error().decode("utf-8", "replace")


def qw_create(dim, extents, coin_dim, dtype, boundary) -> int:
    h = ctypes.c_void_p()
    _check(load().qw_create(dim, _i64(extents), coin_dim, dtype, boundary, ctypes.byref(h)))
    return h.value


def qw_create_batch(batch, dim, extents, coin_dim, dtype, boundary) -> int:
    h = ctypes.c_void_p()
    _check(load().qw_create_batch(batch, dim, _i64(extents), coin_dim, dtype, boundary, ctypes.byref(h)))
    return h.value


def qw_destroy(h) -> None:
    _check(load().qw_destroy(h))


def qw_set_stream(h, cuda_stream) -> None:
    _check(load().qw_set_stream(h, cuda_stream))


def qw_set_lattice(h, lattice) -> None:
    _check(load().qw_set_lattice(h, lattice))


def qw_set_coin(h, mode, coin) -> None:
    _check(load().qw_set_coin(h, mode, _ptr(coin)))


def qw_set_site_phases(h, phases) -> None:
    _check(load().qw_set_site_phases(h, _ptr(phases)))


def qw_set_broken_links(h, mask) -> None:
    _check(load().qw_set_broken_links(h, _ptr(mask)))


def qw_set_random_broken_links(h, enable, p=0.0, seed=0) -> None:
    _check(load().qw_set_random_broken_links(h, int(enable), float(p), int(seed)))


def qw_set_state(h, amps) -> None:
    _check(load().qw_set_state(h, _ptr(amps)))


def qw_set_state_delta(h, site, coin_vec) -> None:
    _check(load().qw_set_state_delta(h, _i64(site), _ptr(coin_vec)))


def qw_get_state(h, amps) -> None:
    _check(load().qw_get_state(h, _ptr(amps)))


def qw_step(h, n) -> None:
    _check(load().qw_step(h, n))


def qw_step_inverse(h, n) -> None:
    _check(load().qw_step_inverse(h, n))


def qw_probabilities(h, out) -> None:
    _check(load().qw_probabilities(h, _ptr(out)))


def qw_probabilities_mean(h, out) -> None:
    _check(load().qw_probabilities_mean(h, _ptr(out)))


def qw_moments(h, out) -> None:
    _check(load().qw_moments(h, _ptr(out)))


def qw_moments_static(h, out) -> None:
    """qw_moments without any allocation: `out` must be a device tensor (include/qw.h)."""
    _check(load().qw_moments_static(h, _ptr(out)))


def qw_set_schedule(h, schedule, k=0) -> None:
    _check(load().qw_set_schedule(h, schedule, k))


def qw_set_window(h, enable) -> None:
    _check(load().qw_set_window(h, int(enable)))


def qw_set_option(h, key, value) -> None:
    _check(load().qw_set_option(h, int(key), int(value)))


def qw_get_info(h, what) -> int:
    out = ctypes.c_int64()
    _check(load().qw_get_info(h, what, ctypes.byref(out)))
    return out.value


QW_PEAK_ADD, QW_PEAK_FMA = 0, 1


def qw_measure_alu_peak(dtype, op) -> float:
    out = ctypes.c_double()
    _check(load().qw_measure_alu_peak(int(dtype), int(op), ctypes.byref(out)))
    return out.value


def qw_synchronize(h) -> None:
    _check(load().qw_synchronize(h))


# ---------------------------------------------------------------------------------------------
# Convenience for tests / bench: create a handle for an inputs.Workload and load its inputs.
# Marshalling only — every arithmetic step still happens inside libqw.
# ---------------------------------------------------------------------------------------------
def dtype_code(np_dtype) -> int:
    return QW_C128 if np.dtype(np_dtype) == np.complex128 else QW_C64


def create_for(w) -> int:
    """Handle with the workload's lattice, coin family, phases; the state is NOT set."""
    h = qw_create_batch(w.batch, w.dim, w.extents, w.coin_dim, dtype_code(w.dtype), w.boundary)
    try:
        if w.lattice != QW_NATURAL:
            qw_set_lattice(h, w.lattice)
        qw_set_coin(h, w.coin_mode, np.ascontiguousarray(w.coin, dtype=w.dtype))
        if w.phases is not None:
            qw_set_site_phases(h, np.ascontiguousarray(w.phases, dtype=w.dtype))
    except Exception:
        qw_destroy(h)
        raise
    return h


def load_state(h, w) -> None:
    if w.state is not None:
        qw_set_state(h, w.state)
    else:
        qw_set_state_delta(h, w.delta_site, np.ascontiguousarray(w.delta_coin, dtype=w.dtype))

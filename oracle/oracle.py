"""numpy front end of the C++ oracle (see qw_oracle.cpp for conventions and citations)."""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qw_oracle.cpp")
_LIB = os.path.join(_HERE, "libqw_oracle.so")
_lock = threading.Lock()
_lib = None

PERIODIC, OPEN = 0, 1
NATURAL, DIAGONAL = 0, 1
COIN_UNIFORM, COIN_PER_WALK, COIN_PER_SITE = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile qw_oracle.cpp -> libqw_oracle.so (g++ -O2, no fast-math, no FMA contraction)."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + ".tmp.%d" % os.getpid()
            subprocess.check_call(
                ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-o", tmp, _SRC]
            )
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64p = ctypes.POINTER(ctypes.c_int64)
        vp = ctypes.c_void_p
        lib.qwo_step.argtypes = [ctypes.c_int, i64p, ctypes.c_int64, ctypes.c_int, ctypes.c_int,
                                 ctypes.c_int, vp, vp, vp, ctypes.c_int64]
        lib.qwo_step_inverse.argtypes = lib.qwo_step.argtypes
        lib.qwo_probabilities.argtypes = [ctypes.c_int, i64p, ctypes.c_int64, vp, vp]
        lib.qwo_moments.argtypes = [ctypes.c_int, i64p, ctypes.c_int64, vp, vp]
        lib.qwo_probabilities_mean.argtypes = [ctypes.c_int, i64p, ctypes.c_int64, vp, vp]
        lib.qwo_dense_unitary.argtypes = [ctypes.c_int, i64p, ctypes.c_int, ctypes.c_int,
                                          ctypes.c_int, vp, vp, vp]
        lib.qwo_step_rbl.argtypes = [ctypes.c_int, i64p, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp,
                                     ctypes.c_double, ctypes.c_uint64, ctypes.c_int64, vp, ctypes.c_int64]
        lib.qwo_step_inverse_rbl.argtypes = lib.qwo_step_rbl.argtypes
        lib.qwo_rbl_mask.argtypes = [ctypes.c_int, i64p, ctypes.c_int64, ctypes.c_int, ctypes.c_int,
                                     ctypes.c_double, ctypes.c_uint64, ctypes.c_int64, vp]
        lib.qwo_philox4x32_10.argtypes = [vp, vp, vp]
        lib.qwo_philox4x32_10.restype = None
        for f in (lib.qwo_step, lib.qwo_step_inverse, lib.qwo_probabilities, lib.qwo_moments, lib.qwo_probabilities_mean,
                  lib.qwo_dense_unitary, lib.qwo_step_rbl, lib.qwo_step_inverse_rbl, lib.qwo_rbl_mask):
            f.restype = ctypes.c_int
        _lib = lib
    return _lib


def _ext(extents):
    extents = [int(e) for e in extents]
    return len(extents), (ctypes.c_int64 * len(extents))(*extents), int(np.prod(extents))


def _coin(coin, cdim, coin_mode, batch, sites):
    coin = np.ascontiguousarray(coin, dtype=np.complex128)
    want = {COIN_UNIFORM: 1, COIN_PER_WALK: batch, COIN_PER_SITE: batch * sites}[coin_mode]
    if coin.size != want * cdim * cdim:
        raise ValueError("coin has %d entries, expected %d" % (coin.size, want * cdim * cdim))
    return coin


def _state(state, batch, sites, cdim):
    if state.dtype != np.complex128 or not state.flags.c_contiguous:
        raise ValueError("state must be a C-contiguous complex128 array")
    if state.size != batch * sites * cdim:
        raise ValueError("state has %d entries, expected %d" % (state.size, batch * sites * cdim))


def _run(fn, extents, coin, state, n, boundary, coin_mode, batch, lattice, broken):
    dim, ext, sites = _ext(extents)
    cdim = 2 * dim
    _state(state, batch, sites, cdim)
    coin = _coin(coin, cdim, coin_mode, batch, sites)
    bptr = None
    if broken is not None:
        broken = np.ascontiguousarray(broken, dtype=np.uint8)
        if broken.size != batch * sites * cdim:
            raise ValueError("broken mask has wrong size")
        bptr = broken.ctypes.data
    rc = fn(dim, ext, batch, boundary, lattice, coin_mode, coin.ctypes.data, bptr,
            state.ctypes.data, int(n))
    if rc:
        raise ValueError("oracle rejected the arguments (rc=%d)" % rc)
    return state


def step(extents, coin, state, n, *, boundary=PERIODIC, coin_mode=COIN_UNIFORM, batch=1,
         lattice=NATURAL, broken=None):
    """Apply U n times in place to ``state`` ([batch][site][coin] complex128) and return it."""
    return _run(_load().qwo_step, extents, coin, state, n, boundary, coin_mode, batch, lattice, broken)


def step_inverse(extents, coin, state, n, *, boundary=PERIODIC, coin_mode=COIN_UNIFORM, batch=1,
                 lattice=NATURAL, broken=None):
    """Apply U^dagger n times in place."""
    return _run(_load().qwo_step_inverse, extents, coin, state, n, boundary, coin_mode, batch,
                lattice, broken)


def probabilities(extents, state, *, batch=1):
    """P[w][x] = sum_a |psi[w][x][a]|^2."""
    dim, ext, sites = _ext(extents)
    _state(state, batch, sites, 2 * dim)
    out = np.empty((batch, sites), dtype=np.float64)
    rc = _load().qwo_probabilities(dim, ext, batch, state.ctypes.data, out.ctypes.data)
    if rc:
        raise ValueError("oracle rejected the arguments")
    return out


def probabilities_mean(extents, state, *, batch=1):
    """Pbar[x] = (1/batch) sum_w sum_a |psi[w][x][a]|^2: the ensemble average over the batch."""
    dim, ext, sites = _ext(extents)
    _state(state, batch, sites, 2 * dim)
    out = np.empty((sites,), dtype=np.float64)
    rc = _load().qwo_probabilities_mean(dim, ext, batch, state.ctypes.data, out.ctypes.data)
    if rc:
        raise ValueError("oracle rejected the arguments")
    return out


def moments(extents, state, *, batch=1):
    """Per walk: 1D (norm, mean, var); 2D (norm, mean_m, mean_n, var_m, var_n, cov_mn)."""
    dim, ext, sites = _ext(extents)
    _state(state, batch, sites, 2 * dim)
    out = np.empty((batch, 3 if dim == 1 else 6), dtype=np.float64)
    rc = _load().qwo_moments(dim, ext, batch, state.ctypes.data, out.ctypes.data)
    if rc:
        raise ValueError("oracle rejected the arguments")
    return out


def dense_unitary(extents, coin, *, boundary=PERIODIC, coin_mode=COIN_UNIFORM, lattice=NATURAL,
                  broken=None):
    """Explicit (sites*cdim)^2 matrix of U for one walk (<= 64 sites)."""
    dim, ext, sites = _ext(extents)
    cdim = 2 * dim
    coin = _coin(coin, cdim, coin_mode, 1, sites)
    bptr = None
    if broken is not None:
        broken = np.ascontiguousarray(broken, dtype=np.uint8)
        bptr = broken.ctypes.data
    D = sites * cdim
    U = np.empty((D, D), dtype=np.complex128)
    rc = _load().qwo_dense_unitary(dim, ext, boundary, lattice, coin_mode, coin.ctypes.data, bptr,
                                   U.ctypes.data)
    if rc:
        raise ValueError("oracle rejected the arguments")
    return U


def _run_rbl(fn, extents, coin, state, n, p, seed, t0, boundary, coin_mode, batch, lattice):
    dim, ext, sites = _ext(extents)
    cdim = 2 * dim
    _state(state, batch, sites, cdim)
    coin = _coin(coin, cdim, coin_mode, batch, sites)
    rc = fn(dim, ext, batch, boundary, lattice, coin_mode, coin.ctypes.data, float(p), int(seed), int(t0),
            state.ctypes.data, int(n))
    if rc:
        raise ValueError("oracle rejected the arguments (rc=%d)" % rc)
    return state


def step_rbl(extents, coin, state, n, p, seed, *, t0=0, boundary=PERIODIC, coin_mode=COIN_UNIFORM, batch=1,
             lattice=NATURAL):
    """Apply U(t0) .. U(t0+n-1) in place, every link redrawn broken with probability p at every step
    (eqs. 9-10; Philox4x32-10 keyed by ``seed``, see qw_oracle.cpp)."""
    return _run_rbl(_load().qwo_step_rbl, extents, coin, state, n, p, seed, t0, boundary, coin_mode, batch, lattice)


def step_inverse_rbl(extents, coin, state, n, p, seed, *, t0, boundary=PERIODIC, coin_mode=COIN_UNIFORM, batch=1,
                     lattice=NATURAL):
    """Undo steps t0-1 .. t0-n of a random-broken-links walk in place (t0 = current time)."""
    return _run_rbl(_load().qwo_step_inverse_rbl, extents, coin, state, n, p, seed, t0, boundary, coin_mode, batch,
                    lattice)


def rbl_mask(extents, p, seed, t, *, boundary=PERIODIC, batch=1, lattice=NATURAL):
    """The broken-link mask [batch][site][coin] (uint8) of step t, in the form ``step(..., broken=)`` takes."""
    dim, ext, sites = _ext(extents)
    out = np.empty((batch, sites, 2 * dim), dtype=np.uint8)
    rc = _load().qwo_rbl_mask(dim, ext, batch, boundary, lattice, float(p), int(seed), int(t), out.ctypes.data)
    if rc:
        raise ValueError("oracle rejected the arguments")
    return out


def philox4x32_10(counter, key):
    """The raw generator: 4 counter words, 2 key words -> 4 output words (uint32)."""
    c = np.ascontiguousarray(counter, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    _load().qwo_philox4x32_10(c.ctypes.data, k.ctypes.data, out.ctypes.data)
    return out

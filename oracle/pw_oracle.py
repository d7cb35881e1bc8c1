"""ctypes wrapper around oracle/pw_oracle.c (plain C, FP64).  TEST INFRASTRUCTURE, not the product.

Blocks are numpy complex128 arrays of shape (nband, npw), C-contiguous: the paper's N x M matrix Psi
 stored column-major with leading dimension npw.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pw_oracle.c")
_SRCS = [_SRC, os.path.join(_HERE, "rr_oracle.c")]     # rr_oracle.c: Rayleigh-Ritz companion steps (oracle/rr_oracle.py)
_LIB = os.path.join(_HERE, "libpw_oracle.so")
_lock = threading.Lock()
_lib = None

TERM_KIN, TERM_LOC, TERM_NL, TERM_ALL = 1, 2, 4, 7


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP over bands).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(f) for f in _SRCS):
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB] + _SRCS + ["-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    with _lock:
        if _lib is None:
            build()
            L = ctypes.CDLL(_LIB)
            c_dp = ctypes.c_void_p
            i64, i32, dbl = ctypes.c_int64, ctypes.c_int, ctypes.c_double
            L.orc_dft1d.argtypes = [i32, i32, c_dp, c_dp]
            L.orc_fft1d.argtypes = [i32, i32, c_dp, c_dp]
            L.orc_dft3d.argtypes = [c_dp, i32, c_dp, i32]
            L.orc_kinetic.argtypes = [c_dp, c_dp, i64, c_dp, c_dp]
            L.orc_apply_h.argtypes = [c_dp, c_dp, c_dp, i64, c_dp, c_dp, i64, c_dp, i64, c_dp, i64, c_dp, i64, c_dp,
                                      i64, i32, i32]
            L.orc_apply_h.restype = i32
            L.orc_cheb_filter.argtypes = [c_dp, c_dp, c_dp, i64, c_dp, c_dp, i64, c_dp, i64, c_dp, i64, c_dp, i64,
                                          i32, dbl, dbl, dbl, i32]
            L.orc_cheb_filter.restype = i32
            L.orc_gram.argtypes = [i64, i64, c_dp, i64, i64, c_dp, i64, c_dp, i64]
            _lib = L
    return _lib


def n_threads() -> int:
    """Threads the OpenMP loops will use (OMP_NUM_THREADS or the affinity mask)."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env:
        return int(env.split(",")[0])
    return len(os.sched_getaffinity(0))


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _c128(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.complex128)


def dft1d(x, sign: int) -> np.ndarray:
    x = _c128(x)
    out = np.empty_like(x)
    _load().orc_dft1d(x.size, sign, _p(x), _p(out))
    return out


def fft1d(x, sign: int) -> np.ndarray:
    x = _c128(x)
    out = np.empty_like(x)
    _load().orc_fft1d(x.size, sign, _p(x), _p(out))
    return out


def dft3d(box, sign: int, use_fft: int = -1) -> np.ndarray:
    """box: (n3, n2, n1) complex128.  Returns the unnormalised transform with exp(sign 2 pi i ...)."""
    box = _c128(box).copy()
    n3, n2, n1 = box.shape
    dims = np.asarray([n1, n2, n3], dtype=np.int32)
    _load().orc_dft3d(_p(dims), sign, _p(box), use_fft)
    return box


def kinetic(lattice, kpt, gvec) -> np.ndarray:
    lattice = np.ascontiguousarray(lattice, dtype=np.float64)
    kpt = np.ascontiguousarray(kpt, dtype=np.float64)
    gvec = np.ascontiguousarray(gvec, dtype=np.int32)
    kin = np.empty(gvec.shape[0], dtype=np.float64)
    _load().orc_kinetic(_p(lattice), _p(kpt), gvec.shape[0], _p(gvec), _p(kin))
    return kin


def _ham_args(lattice, kpt, fft_dims, gvec, vloc, proj, dij):
    lattice = np.ascontiguousarray(lattice, dtype=np.float64)
    kpt = np.ascontiguousarray(kpt, dtype=np.float64)
    dims = np.ascontiguousarray(fft_dims, dtype=np.int32)
    gvec = np.ascontiguousarray(gvec, dtype=np.int32)
    vloc = np.ascontiguousarray(vloc, dtype=np.float64)
    assert vloc.shape == (dims[2], dims[1], dims[0]), "vloc must be (n3, n2, n1)"
    npw = gvec.shape[0]
    if proj is None or len(proj) == 0:
        proj = np.zeros((0, npw), dtype=np.complex128)
        dij = np.zeros((0,), dtype=np.float64)
    proj = _c128(proj)
    dij = np.ascontiguousarray(dij, dtype=np.float64)
    assert proj.shape[1] == npw and dij.shape[0] == proj.shape[0]
    keep = (lattice, kpt, dims, gvec, vloc, proj, dij)
    args = [_p(lattice), _p(kpt), _p(dims), npw, _p(gvec), _p(vloc), proj.shape[0], _p(proj), npw, _p(dij)]
    return keep, args, npw


def apply_h(lattice, kpt, fft_dims, gvec, vloc, proj, dij, psi, terms: int = TERM_ALL, use_fft: int = -1):
    """H psi for a block psi of shape (nband, npw)."""
    keep, args, npw = _ham_args(lattice, kpt, fft_dims, gvec, vloc, proj, dij)
    psi = _c128(psi)
    squeeze = psi.ndim == 1
    psi2 = psi.reshape(-1, npw)
    out = np.empty_like(psi2)
    rc = _load().orc_apply_h(*args, psi2.shape[0], _p(psi2), npw, _p(out), npw, terms, use_fft)
    if rc != 0:
        raise RuntimeError(f"orc_apply_h failed rc={rc}")
    return out[0] if squeeze else out


def cheb_filter(lattice, kpt, fft_dims, gvec, vloc, proj, dij, psi, degree, a, b, a0, use_fft: int = -1):
    """Scaled Chebyshev filter of `degree` applied to the block psi (nband, npw); returns a new array."""
    keep, args, npw = _ham_args(lattice, kpt, fft_dims, gvec, vloc, proj, dij)
    out = _c128(psi).reshape(-1, npw).copy()
    rc = _load().orc_cheb_filter(*args, out.shape[0], _p(out), npw, int(degree), float(a), float(b), float(a0),
                                 use_fft)
    if rc != 0:
        raise RuntimeError(f"orc_cheb_filter failed rc={rc}")
    return out.reshape(np.shape(psi))


def gram(x, y) -> np.ndarray:
    """G = X^H Y for blocks x (nx, npw), y (ny, npw); returns (nx, ny) with G[i, j] = <x_i, y_j>."""
    x = _c128(x)
    y = _c128(y)
    nx, npw = x.shape
    ny = y.shape[0]
    assert y.shape[1] == npw
    g_cm = np.empty((ny, nx), dtype=np.complex128)  # column-major nx x ny
    _load().orc_gram(npw, nx, _p(x), npw, ny, _p(y), npw, _p(g_cm), nx)
    return np.ascontiguousarray(g_cm.T)

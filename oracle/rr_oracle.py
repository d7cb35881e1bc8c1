"""ctypes wrapper around oracle/rr_oracle.c plus the Rayleigh-Ritz / Chebyshev-filtering iteration written on top of it
-- TEST INFRASTRUCTURE, not the product.

One Chebyshev-filtering iteration (Algorithm 12 with S = I, i.e. Sinv = identity and HX_SX = HX; garbled loop
body read as DESIGN.md R2) is, step by step:

    1-2  H Psi                                                         (HX)
    3    Rayleigh quotients lambda_i, their minimum and maximum
    4-8  Psi <- p_m(H) Psi, the scaled Chebyshev filter of degree m    (oracle.cheb_filter; bounds from step 3, R5)
    10   Rayleigh-Ritz: H_Psi = Psi^H (H Psi), S_Psi = Psi^H Psi, H_Psi X = S_Psi X Lambda, Psi <- Psi X, H Psi <- (H Psi) X
                                                                       (Algorithm 10; Algorithm 5)
    11   W = H Psi - Psi Lambda                                        (S = I)
    12   residual norms ||W_i||

Blocks are numpy complex128 arrays of shape (nband, npw), C-contiguous (column-major npw x nband, as everywhere in
oracle/); small matrices are returned as ordinary numpy (row, column) arrays.
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import pw_oracle as _pw

_declared = False


def _lib():
    global _declared
    L = _pw._load()
    if not _declared:
        vp, i64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
        L.orc_rayleigh.argtypes = [i64, i64, vp, i64, vp, i64, vp, vp]
        L.orc_rotate.argtypes = [i64, i64, vp, i64, i64, vp, i64, vp, i64]
        L.orc_residual.argtypes = [i64, i64, vp, i64, vp, i64, vp, vp, i64, vp]
        L.orc_potrf_upper.argtypes = [i64, vp, i64]
        L.orc_potrf_upper.restype = i32
        L.orc_trsm_right_upper.argtypes = [i64, i64, vp, i64, vp, i64]
        L.orc_heev_jacobi.argtypes = [i64, vp, i64, vp, vp, i64]
        L.orc_heev_jacobi.restype = i32
        L.orc_hegv.argtypes = [i64, vp, i64, vp, i64, vp, vp, i64]
        L.orc_hegv.restype = i32
        _declared = True
    return L


_p = _pw._p
_c128 = _pw._c128


def _cm_copy(a) -> np.ndarray:
    """A fresh C-contiguous array holding the transpose of `a`, i.e. `a` in column-major order (always a copy: the C
    routines work in place)."""
    return np.array(np.asarray(a, dtype=np.complex128).T, dtype=np.complex128, order="C", copy=True)


def rayleigh(psi, hpsi):
    """lambda_i = Re <psi_i, H psi_i> / <psi_i, psi_i> and the squared norms <psi_i, psi_i>."""
    psi, hpsi = _c128(psi), _c128(hpsi)
    nb, npw = psi.shape
    lam = np.empty(nb)
    nrm2 = np.empty(nb)
    _lib().orc_rayleigh(npw, nb, _p(psi), npw, _p(hpsi), npw, _p(lam), _p(nrm2))
    return lam, nrm2


def rotate(x, q):
    """Y = X Q for a block x (m, npw) and an m x n matrix q[i, j]; returns (n, npw): band j of Y = sum_i q[i, j] band i of X."""
    x = _c128(x)
    m, npw = x.shape
    q_cm = np.ascontiguousarray(np.asarray(q, dtype=np.complex128).T)     # column-major m x n
    n = q_cm.shape[0]
    assert q_cm.shape[1] == m
    y = np.empty((n, npw), dtype=np.complex128)
    _lib().orc_rotate(npw, m, _p(x), npw, n, _p(q_cm), m, _p(y), npw)
    return y


def residual(psi, hpsi, lam):
    """W = H psi - psi diag(lam) and the column norms ||W_i||_2."""
    psi, hpsi = _c128(psi), _c128(hpsi)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    nb, npw = psi.shape
    w = np.empty_like(psi)
    norms = np.empty(nb)
    _lib().orc_residual(npw, nb, _p(psi), npw, _p(hpsi), npw, _p(lam), _p(w), npw, _p(norms))
    return w, norms


def potrf_upper(s):
    """U (ordinary row/column array, upper triangular, positive diagonal) with S = U^H U."""
    a_cm = _cm_copy(s)
    n = a_cm.shape[0]
    rc = _lib().orc_potrf_upper(n, _p(a_cm), n)
    if rc:
        raise np.linalg.LinAlgError(f"matrix is not positive definite at pivot {rc - 1}")
    return np.ascontiguousarray(a_cm.T)


def trsm_right_upper(x, u):
    """X U^-1 for a block x (n, npw) -- band j of the result = (x_j - sum_{k<j} y_k U[k, j]) / U[j, j]."""
    y = _c128(x).copy()
    n, npw = y.shape
    u_cm = np.ascontiguousarray(np.asarray(u, dtype=np.complex128).T)
    _lib().orc_trsm_right_upper(npw, n, _p(y), npw, _p(u_cm), n)
    return y


def heev(a):
    """Eigenvalues (ascending) and eigenvectors (columns of the returned matrix) of a Hermitian matrix; cyclic Jacobi."""
    a_cm = _cm_copy(a)
    n = a_cm.shape[0]
    w = np.empty(n)
    v_cm = np.empty((n, n), dtype=np.complex128)
    _lib().orc_heev_jacobi(n, _p(a_cm), n, _p(w), _p(v_cm), n)
    return w, np.ascontiguousarray(v_cm.T)


def hegv(a, b):
    """A X = B X diag(w) with X^H B X = I; returns (w ascending, X)."""
    a_cm = _cm_copy(a)
    b_cm = _cm_copy(b)
    n = a_cm.shape[0]
    w = np.empty(n)
    x_cm = np.empty((n, n), dtype=np.complex128)
    rc = _lib().orc_hegv(n, _p(a_cm), n, _p(b_cm), n, _p(w), _p(x_cm), n)
    if rc:
        raise np.linalg.LinAlgError(f"B is not positive definite at pivot {rc - 1}")
    return w, np.ascontiguousarray(x_cm.T)


def chol_ortho(psi, hpsi=None):
    """Algorithm 9 (S-Ortho, S = I): S_Psi = Psi^H Psi = U^H U, Psi <- Psi U^-1 (and H Psi <- (H Psi) U^-1).
    Returns (psi_new, hpsi_new or None, U)."""
    s = _pw.gram(psi, psi)
    u = potrf_upper(s)
    out = trsm_right_upper(psi, u)
    hout = trsm_right_upper(hpsi, u) if hpsi is not None else None
    return out, hout, u


def rayleigh_ritz(psi, hpsi):
    """Algorithm 10 / 5 with S = I: returns (lam, psi X, (H psi) X, X)."""
    h_sub = _pw.gram(psi, hpsi)
    h_sub = 0.5 * (h_sub + h_sub.conj().T)
    s_sub = _pw.gram(psi, psi)
    s_sub = 0.5 * (s_sub + s_sub.conj().T)
    lam, x = hegv(h_sub, s_sub)
    return lam, rotate(psi, x), rotate(hpsi, x), x


def chebfi_iteration(lattice, kpt, fft_dims, gvec, vloc, proj, dij, psi, degree, b, a0_margin=0.0):
    """One Chebyshev-filtering iteration, Algorithm 12 with S = I (module docstring).  The filter's damped interval is
    [a, b] with a = the largest Rayleigh quotient and the normalisation point a0 = the smallest one minus `a0_margin`
    (R5: the paper takes min/max of the Rayleigh quotients; b, an upper bound of the spectrum, is an
    input).  Returns a dict with lam (Ritz values), psi, hpsi (rotated), resid (norms), a, a0."""
    args = (lattice, kpt, fft_dims, gvec, vloc, proj, dij)
    hpsi = _pw.apply_h(*args, psi)
    rq, _ = rayleigh(psi, hpsi)
    a, a0 = float(rq.max()), float(rq.min()) - float(a0_margin)
    y = _pw.cheb_filter(*args, psi, degree, a, b, a0)
    hy = _pw.apply_h(*args, y)
    lam, y2, hy2, x = rayleigh_ritz(y, hy)
    _, norms = residual(y2, hy2, lam)
    return {"lam": lam, "psi": y2, "hpsi": hy2, "resid": norms, "a": a, "a0": a0, "rq": rq, "x": x}

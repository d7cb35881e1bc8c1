"""CPU oracle of the PAW-style generalised problem H Psi = Lambda S Psi -- TEST INFRASTRUCTURE ONLY.

    V_nonloc = sum_{R,i,j} |p_i^R> D_ij^R <p_j^R|            per-atom dense Hermitian blocks D^R
    S        = I + sum_{R,i,j} |p_i^R> Q_ij^R <p_j^R|        the PAW overlap operator, S != I
    HX_SX    : H Psi and S Psi from ONE set of projections C = P^H Psi
    Sinv     : S^-1 applied through the Woodbury identity
               S^-1 = I - P Q (I + G Q)^-1 P^H,  G = P^H P   (valid for singular Q as well)
    filter   : the scaled Chebyshev polynomial of S^-1 H, Algorithm 12 lines 4-8:
               each degree is  S^-1 (H Y_j)  followed by the three-term axpy
    RR       : H_Psi = Psi^H (H Psi), S_Psi = Psi^H (S Psi), H_Psi X = S_Psi X Lambda (Algorithm 10)
    residual : W = (H - Lambda S) Psi (Algorithm 12 line 11)

Plain definitions in numpy on top of the C oracle's kinetic + local application (oracle.apply_h with the nonlocal term
switched off); the block sums and the small J x J solve are numpy matmul / numpy.linalg.solve calls (library primitives
used as steps).  Blocks are given as `offsets` (natom + 1 integers into the projector index) and lists of n_R x n_R
arrays indexed [i, j].  Pins: tests/test_paw_oracle_pins.py.  Shares no code with the CUDA path.
"""
from __future__ import annotations

import numpy as np

from . import pw_oracle as _pw
from . import rr_oracle as _rr


def blockdiag_apply(offsets, blocks, c):
    """(blockdiag(B^R) c): c is (nproj, nband); plain per-block products."""
    out = np.zeros_like(c)
    for r in range(len(offsets) - 1):
        lo, hi = int(offsets[r]), int(offsets[r + 1])
        out[lo:hi] = np.asarray(blocks[r], dtype=np.complex128) @ c[lo:hi]
    return out


def blockdiag_dense(offsets, blocks):
    n = int(offsets[-1])
    m = np.zeros((n, n), dtype=np.complex128)
    for r in range(len(offsets) - 1):
        lo, hi = int(offsets[r]), int(offsets[r + 1])
        m[lo:hi, lo:hi] = blocks[r]
    return m


def projections(proj, psi):
    """C[i, b] = <p_i | psi_b> = sum_G conj(P[G, i]) psi_b(G);  proj (nproj, npw), psi (nband, npw) -> (nproj, nband)."""
    return np.asarray(proj).conj() @ np.asarray(psi).T


def apply_hs(lattice, kpt, fft_dims, gvec, vloc, proj, offsets, dblocks, qblocks, psi):
    """HX_SX: returns (H psi, S psi) for a block psi (nband, npw)."""
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    hpsi = _pw.apply_h(lattice, kpt, fft_dims, gvec, vloc, None, None, psi, terms=_pw.TERM_KIN | _pw.TERM_LOC)
    c = projections(proj, psi)
    p = np.asarray(proj, dtype=np.complex128)
    hpsi = hpsi + (p.T @ blockdiag_apply(offsets, dblocks, c)).T
    spsi = psi + (p.T @ blockdiag_apply(offsets, qblocks, c)).T
    return np.ascontiguousarray(hpsi), np.ascontiguousarray(spsi)


def apply_sinv(proj, offsets, qblocks, x):
    """Sinv: y = S^-1 x = x - P Q (I + G Q)^-1 P^H x with G = P^H P  (Woodbury / push-through identity)."""
    p = np.asarray(proj, dtype=np.complex128)
    x = np.ascontiguousarray(x, dtype=np.complex128)
    g = p.conj() @ p.T                                       # G[i, j] = <p_i | p_j>
    q = blockdiag_dense(offsets, qblocks)
    c = projections(p, x)                                    # P^H x
    t = np.linalg.solve(np.eye(g.shape[0]) + g @ q, c)
    return np.ascontiguousarray(x - (p.T @ (q @ t)).T)


def cheb_filter_gen(lattice, kpt, fft_dims, gvec, vloc, proj, offsets, dblocks, qblocks, psi, degree, a, b, a0):
    """Scaled Chebyshev filter of degree m of the operator S^-1 H (same recurrence as oracle.cheb_filter, R1):
    Y_1 = (sigma_1/e)(S^-1 H - c) Y_0,  Y_{j+1} = (2 sigma_{j+1}/e)(S^-1 H - c) Y_j - sigma_j sigma_{j+1} Y_{j-1}."""
    if degree < 0 or not (b > a) or not (a0 < a):
        raise ValueError("bad filter parameters")
    args = (lattice, kpt, fft_dims, gvec, vloc, proj, offsets, dblocks, qblocks)
    y_prev = np.ascontiguousarray(psi, dtype=np.complex128).copy()
    if degree == 0:
        return y_prev
    e, c = 0.5 * (b - a), 0.5 * (b + a)
    sigma1 = e / (a0 - c)
    sigma = sigma1

    def sinv_h(y):
        hy, _ = apply_hs(*args, y)
        return apply_sinv(proj, offsets, qblocks, hy)

    y_cur = (sigma1 / e) * (sinv_h(y_prev) - c * y_prev)
    for _ in range(1, degree):
        sigma_new = 1.0 / (2.0 / sigma1 - sigma)
        y_new = (2.0 * sigma_new / e) * (sinv_h(y_cur) - c * y_cur) - (sigma * sigma_new) * y_prev
        y_prev, y_cur = y_cur, y_new
        sigma = sigma_new
    return np.ascontiguousarray(y_cur)


def rayleigh_gen(psi, hpsi, spsi):
    """lambda_i = Re <psi_i, H psi_i> / Re <psi_i, S psi_i>."""
    num = np.einsum("bg,bg->b", np.conj(psi), hpsi).real
    den = np.einsum("bg,bg->b", np.conj(psi), spsi).real
    return num / den


def rayleigh_ritz_gen(psi, hpsi, spsi):
    """Algorithm 10: returns (lam, psi X, (H psi) X, (S psi) X, X) with X^H S_Psi X = I."""
    h_sub = _pw.gram(psi, hpsi)
    s_sub = _pw.gram(psi, spsi)
    h_sub = 0.5 * (h_sub + h_sub.conj().T)
    s_sub = 0.5 * (s_sub + s_sub.conj().T)
    lam, x = _rr.hegv(h_sub, s_sub)
    return lam, _rr.rotate(psi, x), _rr.rotate(hpsi, x), _rr.rotate(spsi, x), x


def residual_gen(psi, hpsi, spsi, lam):
    """W_i = H psi_i - lam_i S psi_i and the norms ||W_i||_2."""
    w = np.asarray(hpsi) - np.asarray(lam)[:, None] * np.asarray(spsi)
    return w, np.linalg.norm(w, axis=1)


def chebfi_iteration_gen(lattice, kpt, fft_dims, gvec, vloc, proj, offsets, dblocks, qblocks, psi, degree, b,
                         a0_margin=0.0):
    """One iteration of Algorithm 12 with the PAW overlap (all lines): HX_SX, Rayleigh quotients -> [a0, a], the
    S^-1 H filter, HX_SX, Rayleigh-Ritz, residuals."""
    args = (lattice, kpt, fft_dims, gvec, vloc, proj, offsets, dblocks, qblocks)
    hpsi, spsi = apply_hs(*args, psi)
    rq = rayleigh_gen(psi, hpsi, spsi)
    a, a0 = float(rq.max()), float(rq.min()) - float(a0_margin)
    y = cheb_filter_gen(*args, psi, degree, a, b, a0)
    hy, sy = apply_hs(*args, y)
    lam, y2, hy2, sy2, x = rayleigh_ritz_gen(y, hy, sy)
    _, norms = residual_gen(y2, hy2, sy2, lam)
    return {"lam": lam, "psi": y2, "hpsi": hy2, "spsi": sy2, "resid": norms, "a": a, "a0": a0, "rq": rq}

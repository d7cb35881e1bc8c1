"""CPU oracle of one LOBPCG block solve, Algorithm 11 of the paper (outline Algorithm 6)
with S = I (`lobpcg`) and with the PAW overlap S (`lobpcg_gen`) -- TEST INFRASTRUCTURE ONLY.

Followed line by line, in the paper's order and notation, on top of the already pinned pieces (oracle.apply_h = HX,
oracle.gram, rr.potrf_upper / trsm_right_upper = S-Ortho, rr.hegv = the Rayleigh-Ritz eigen-solve, rr.rotate):

    for every block Psi_i of M/b bands (lines 1-30):
        3      Psi_i <- S-Deflate against the blocks already solved       (Algorithm 8: Psi <- Psi - Psi_0 (Psi_0^H Psi))
        6      H Psi_i                                                    (HX)
        8      S-Ortho(Psi_i, H Psi_i)                                    (Algorithm 9)
        9      Lambda_i, Psi_i, H Psi_i <- RR(M/b)                        (Algorithm 10)
        for n = 1..k (lines 10-28):
            11     W_i <- (H - Lambda_i) Psi_i
            12     residual norms (returned; the early exit of line 12 is taken only when `tol` > 0)
            13     W_i <- K W_i, K the diagonal preconditioner
            15     W_i <- S-Deflate against the solved blocks
            18     H W_i
            21/24  S-Ortho of [Psi_i, W_i] (n = 1) or [Psi_i, W_i, P_i]
            22/25  RR of that basis: the lowest M/b Ritz pairs give the new Psi_i; P_i is their part outside span(Psi_i)
            26     Psi_i <- Psi_i + P_i  (in the rotated basis: new Psi_i = B' C, P_i = B'[W, P columns] C[W, P rows])
        29     residual norms
    31-34  if b > 1: S-Ortho and RR over all M bands

Readings: the paper calls K "the preconditioner (diagonal matrix)" without a formula; the oracle
takes the Teter-Payne-Allan polynomial that plane-wave codes (ABINIT included) use, K(x) = t / (t + 16 x^4) with
t = 27 + 18 x + 12 x^2 + 8 x^3 and x = kin(G) / <T>_band, <T>_band the kinetic energy of the band being corrected.
"""
from __future__ import annotations

import numpy as np

from . import pw_oracle as _pw
from . import rr_oracle as _rr


def tpa_preconditioner(kin: np.ndarray, ekin: np.ndarray) -> np.ndarray:
    """K[b, G] of Teter-Payne-Allan for bands with kinetic energies ekin[b]."""
    x = kin[None, :] / ekin[:, None]
    t = 27.0 + 18.0 * x + 12.0 * x * x + 8.0 * x ** 3
    return t / (t + 16.0 * x ** 4)


def band_kinetic(kin: np.ndarray, psi: np.ndarray) -> np.ndarray:
    """<T>_b = sum_G kin(G) |psi_b(G)|^2 / sum_G |psi_b(G)|^2."""
    w = psi.real ** 2 + psi.imag ** 2
    return (w @ kin) / w.sum(axis=1)


def deflate(x: np.ndarray, basis: np.ndarray) -> np.ndarray:
    """Algorithm 8 with S = I: x <- x - basis (basis^H x), rows = bands."""
    if basis is None or len(basis) == 0:
        return x
    s = _pw.gram(basis, x)                     # s[i, j] = <basis_i, x_j>
    return np.ascontiguousarray(x - _rr.rotate(basis, s))


def deflate_gen(x: np.ndarray, basis: np.ndarray, sbasis: np.ndarray) -> np.ndarray:
    """Algorithm 8 (S-Deflate): x <- x - basis ((S basis)^H x), i.e. the S-orthogonal projection away from span(basis)."""
    if basis is None or len(basis) == 0:
        return x
    s = _pw.gram(sbasis, x)                    # s[i, j] = <S basis_i, x_j> = <basis_i, S x_j>
    return np.ascontiguousarray(x - _rr.rotate(basis, s))


def chol_ortho_gen(x, hx, sx):
    """Algorithm 9 (S-Ortho): S_X = X^H (S X) = U^H U, then X, H X, S X <- . U^-1.  Returns (x, hx, sx, U)."""
    s = _pw.gram(x, sx)
    u = _rr.potrf_upper(0.5 * (s + s.conj().T))
    return _rr.trsm_right_upper(x, u), _rr.trsm_right_upper(hx, u), _rr.trsm_right_upper(sx, u), u


def lobpcg_gen(lattice, kpt, fft_dims, gvec, vloc, proj, offsets, dblocks, qblocks, psi, nblocks: int, nline: int,
               tol: float = 0.0):
    """Algorithm 11 as printed, with the PAW overlap S = I + P Q P^H (HX_SX, S-Deflate, S-Ortho, RR of
    PAPER.md:224-238): the same steps as `lobpcg` with <.,.> replaced by <., S .>, the residual by (H - lambda S) Psi, and
    H X, S X coming from one call of the paw oracle's apply_hs.  Returns dict(lam, psi, hpsi, spsi, resid, history)."""
    from . import paw_oracle as _paw
    args = (lattice, kpt, fft_dims, gvec, vloc, proj, offsets, dblocks, qblocks)
    kin = _pw.kinetic(lattice, kpt, gvec)
    psi = np.ascontiguousarray(psi, dtype=np.complex128).copy()
    M = psi.shape[0]
    assert M % nblocks == 0
    m = M // nblocks
    hpsi, spsi = np.empty_like(psi), np.empty_like(psi)
    lam_all = np.empty(M)
    history = []
    for i in range(nblocks):
        lo, hi = i * m, (i + 1) * m
        done, sdone = psi[:lo], spsi[:lo]
        x = deflate_gen(psi[lo:hi], done, sdone)                                # line 3
        hx, sx = _paw.apply_hs(*args, x)                                        # line 6
        x, hx, sx, _ = chol_ortho_gen(x, hx, sx)                                # line 8
        lam, x, hx, sx, _ = _paw.rayleigh_ritz_gen(x, hx, sx)                   # line 9
        p = hp = sp = None
        hist = []
        for n in range(1, nline + 1):                                           # line 10
            w, norms = _paw.residual_gen(x, hx, sx, lam)                        # lines 11-12
            hist.append(norms)
            if tol > 0.0 and norms.max() <= tol:
                break
            w = np.ascontiguousarray(tpa_preconditioner(kin, band_kinetic(kin, x)) * w)   # line 13
            w = deflate_gen(w, done, sdone)                                     # line 15
            hw, sw = _paw.apply_hs(*args, w)                                    # line 18
            cat = lambda parts: np.ascontiguousarray(np.concatenate(parts, axis=0))
            bmat = cat([x, w] if p is None else [x, w, p])
            hb = cat([hx, hw] if p is None else [hx, hw, hp])
            sb = cat([sx, sw] if p is None else [sx, sw, sp])
            bmat, hb, sb, _ = chol_ortho_gen(bmat, hb, sb)                      # lines 21 / 24
            h_sub = _pw.gram(bmat, hb)
            s_sub = _pw.gram(bmat, sb)
            theta, c = _rr.hegv(0.5 * (h_sub + h_sub.conj().T), 0.5 * (s_sub + s_sub.conj().T))   # lines 22 / 25
            cm = c[:, :m]
            lam = theta[:m]
            c_out = cm.copy()
            c_out[:m, :] = 0.0
            p, hp, sp = _rr.rotate(bmat, c_out), _rr.rotate(hb, c_out), _rr.rotate(sb, c_out)
            x, hx, sx = _rr.rotate(bmat, cm), _rr.rotate(hb, cm), _rr.rotate(sb, cm)        # line 26
        history.append(hist)
        psi[lo:hi], hpsi[lo:hi], spsi[lo:hi], lam_all[lo:hi] = x, hx, sx, lam
    if nblocks > 1:                                                             # lines 31-34
        psi, hpsi, spsi, _ = chol_ortho_gen(psi, hpsi, spsi)
        lam_all, psi, hpsi, spsi, _ = _paw.rayleigh_ritz_gen(psi, hpsi, spsi)
    _, resid = _paw.residual_gen(psi, hpsi, spsi, lam_all)                      # line 29
    return {"lam": lam_all, "psi": psi, "hpsi": hpsi, "spsi": spsi, "resid": resid, "history": history}


def lobpcg(lattice, kpt, fft_dims, gvec, vloc, proj, dij, psi, nblocks: int, nline: int, tol: float = 0.0):
    """Returns dict(lam (M,), psi (M, npw), hpsi, resid (M,) final residual norms, history = list per block of the
    residual-norm arrays seen at line 12)."""
    args = (lattice, kpt, fft_dims, gvec, vloc, proj, dij)
    kin = _pw.kinetic(lattice, kpt, gvec)
    psi = np.ascontiguousarray(psi, dtype=np.complex128).copy()
    M = psi.shape[0]
    assert M % nblocks == 0
    m = M // nblocks
    hpsi = np.empty_like(psi)
    lam_all = np.empty(M)
    history = []
    for i in range(nblocks):
        lo, hi = i * m, (i + 1) * m
        done = psi[:lo]
        x = deflate(psi[lo:hi], done)                                           # line 3
        hx = _pw.apply_h(*args, x)                                              # line 6
        x, hx, _ = _rr.chol_ortho(x, hx)                                        # line 8
        lam, x, hx, _ = _rr.rayleigh_ritz(x, hx)                                # line 9
        p = hp = None
        hist = []
        for n in range(1, nline + 1):                                           # line 10
            w, norms = _rr.residual(x, hx, lam)                                 # lines 11-12
            hist.append(norms)
            if tol > 0.0 and norms.max() <= tol:
                break
            w = np.ascontiguousarray(tpa_preconditioner(kin, band_kinetic(kin, x)) * w)   # line 13
            w = deflate(w, done)                                                # line 15
            hw = _pw.apply_h(*args, w)                                          # line 18
            basis = [x, w] if p is None else [x, w, p]
            hbasis = [hx, hw] if p is None else [hx, hw, hp]
            bmat = np.ascontiguousarray(np.concatenate(basis, axis=0))
            hb = np.ascontiguousarray(np.concatenate(hbasis, axis=0))
            bmat, hb, _ = _rr.chol_ortho(bmat, hb)                              # lines 21 / 24
            h_sub = _pw.gram(bmat, hb)
            s_sub = _pw.gram(bmat, bmat)
            theta, c = _rr.hegv(0.5 * (h_sub + h_sub.conj().T), 0.5 * (s_sub + s_sub.conj().T))   # lines 22 / 25
            cm = c[:, :m]                                                       # the lowest M/b Ritz vectors
            lam = theta[:m]
            c_out = cm.copy()
            c_out[:m, :] = 0.0                                                  # the part outside span(Psi_i)
            p, hp = _rr.rotate(bmat, c_out), _rr.rotate(hb, c_out)
            x, hx = _rr.rotate(bmat, cm), _rr.rotate(hb, cm)                    # line 26: Psi_i = (Psi_i part) + P_i
        history.append(hist)
        psi[lo:hi], hpsi[lo:hi], lam_all[lo:hi] = x, hx, lam
    if nblocks > 1:                                                             # lines 31-34
        psi, hpsi, _ = _rr.chol_ortho(psi, hpsi)
        lam_all, psi, hpsi, _ = _rr.rayleigh_ritz(psi, hpsi)
    _, resid = _rr.residual(psi, hpsi, lam_all)                                 # line 29
    return {"lam": lam_all, "psi": psi, "hpsi": hpsi, "resid": resid, "history": history}

"""Brute-force dense Hamiltonian (smallest config only) -- TEST INFRASTRUCTURE, part of the oracle's pins.

H[G,G'] = kin(G) delta_GG' + Vhat[wrap(n_G - n_G')] + sum_i P[G,i] D_i conj(P[G',i])
with Vhat(m) = (1/F) sum_r V_loc(r) exp(-2 pi i m.r/n).  It is built from the convolution theorem with numpy's own
FFT and linear algebra, NOT by calling the oracle's apply, so that it independently checks the oracle's
scatter / transform / gather indexing, its normalisation and its projector sums (H is an N x N
Hermitian matrix; V_nonloc = sum |p_i> D_ij <p_j|).
"""
import numpy as np


def dense_h(lattice, kpt, fft_dims, gvec, vloc, proj, dij) -> np.ndarray:
    lattice = np.asarray(lattice, dtype=np.float64)
    n1, n2, n3 = (int(v) for v in fft_dims)
    g = np.asarray(gvec, dtype=np.int64)
    recip = 2.0 * np.pi * np.linalg.inv(lattice).T
    q = (g + np.asarray(kpt, dtype=np.float64)[None, :]) @ recip
    kin = 0.5 * np.einsum("ij,ij->i", q, q)
    vhat = np.fft.fftn(np.asarray(vloc, dtype=np.float64)) / (n1 * n2 * n3)   # axes (i3, i2, i1), exp(-i...)
    d = g[:, None, :] - g[None, :, :]
    h = vhat[d[..., 2] % n3, d[..., 1] % n2, d[..., 0] % n1].astype(np.complex128)
    h[np.diag_indices_from(h)] += kin
    if proj is not None and len(proj):
        p = np.asarray(proj, dtype=np.complex128)          # (nproj, npw): p[i, G] = P[G, i]
        h += (p.T * np.asarray(dij)[None, :]) @ p.conj()
    return h

"""Pins of the LOBPCG oracle (oracle/lobpcg_oracle.py, Algorithm 11 of the paper): hand values of the
preconditioner, projector properties of S-Deflate, the nline = 0 special case (= Rayleigh-Ritz of the input, separately
pinned), convergence to the dense spectrum (numpy.linalg.eigvalsh of oracle.dense_h) with Ritz values bounding it from
above, fixed points (an exact invariant subspace stays put).  CPU only."""
import numpy as np
import pytest

import oracle
from oracle import lobpcg_oracle as lo
from oracle import rr
from paper_2604_11139_b200 import synth


def ham_args(w):
    return (w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, w.proj, w.dij)


def test_tpa_preconditioner_hand_values():
    kin = np.array([0.0, 1.0, 2.0, 1e6])
    k = lo.tpa_preconditioner(kin, np.array([1.0, 2.0]))
    assert k[0, 0] == 1.0                                               # x = 0
    assert k[0, 1] == pytest.approx(65.0 / 81.0, rel=1e-15)             # x = 1: (27+18+12+8) / (65 + 16)
    assert k[1, 2] == pytest.approx(65.0 / 81.0, rel=1e-15)             # x = kin / ekin = 2 / 2
    assert k[0, 3] * 2e6 == pytest.approx(1.0, rel=1e-5)                # x -> infinity: K -> 1 / (2 x)
    assert np.all(np.diff(lo.tpa_preconditioner(np.linspace(0, 50, 200), np.array([1.0]))[0]) < 0)   # decreasing in x


def test_band_kinetic_and_deflate(cfg1):
    w = cfg1
    kin = oracle.kinetic(w.lattice, w.kpt, w.gvec)
    e = np.zeros((2, w.npw), dtype=np.complex128)
    e[0, 7] = 3.0j
    e[1, 7], e[1, 100] = 1.0, 1.0
    ek = lo.band_kinetic(kin, e)
    assert ek[0] == pytest.approx(kin[7]) and ek[1] == pytest.approx(0.5 * (kin[7] + kin[100]))
    basis = w.psi[:5]                                                   # orthonormal (cfg 1's block is)
    x = w.psi[5:9] + 0.3 * w.psi[:4]
    y = lo.deflate(x, basis)
    assert np.abs(oracle.gram(basis, y)).max() <= 1e-14                 # orthogonal to the basis afterwards
    assert np.abs(lo.deflate(y, basis) - y).max() <= 1e-14              # idempotent
    assert np.abs(y - w.psi[5:9]).max() <= 1e-13                        # the admixture is removed exactly
    assert lo.deflate(x, basis[:0]) is x


def test_nline_zero_is_rayleigh_ritz_of_the_input(cfg1):
    w = cfg1
    out = lo.lobpcg(*ham_args(w), w.psi, 1, 0)
    hpsi = oracle.apply_h(*ham_args(w), w.psi)
    lam_ref = np.linalg.eigvalsh(oracle.gram(w.psi, hpsi))              # psi is orthonormal: standard problem (library)
    assert np.abs(out["lam"] - lam_ref).max() <= 1e-12 * np.abs(lam_ref).max()
    assert np.abs(out["psi"] @ out["psi"].conj().T - np.eye(w.psi.shape[0])).max() <= 1e-12


@pytest.mark.parametrize("nblocks", [1, 2, 4])
def test_converges_to_the_dense_spectrum(cfg1, nblocks):
    w = cfg1
    ev = np.linalg.eigvalsh(oracle.dense_h(*ham_args(w)))
    M = w.psi.shape[0]
    out = lo.lobpcg(*ham_args(w), w.psi, nblocks, 12)
    lam = out["lam"]
    assert np.all(np.diff(lam) >= -1e-12)
    assert np.all(lam >= ev[:M] - 1e-9)                                 # Ritz values bound the spectrum from above
    assert np.abs(lam[: M // 2] - ev[: M // 2]).max() < 1e-5
    assert np.abs(out["psi"] @ out["psi"].conj().T - np.eye(M)).max() <= 1e-10
    assert np.abs(out["hpsi"] - oracle.apply_h(*ham_args(w), out["psi"])).max() <= 1e-9
    for hist in out["history"]:                                         # residuals of a block shrink along the line minimisations
        assert hist[-1].max() < 0.1 * hist[0].max()
    # more line minimisations never raise a Ritz value (the search space contains the previous iterate)
    fewer = lo.lobpcg(*ham_args(w), w.psi, nblocks, 4)["lam"]
    if nblocks == 1:
        assert np.all(lam <= fewer + 1e-10)


def test_exact_invariant_subspace_is_a_fixed_point(cfg1):
    w = cfg1
    ev, vec = np.linalg.eigh(oracle.dense_h(*ham_args(w)))
    psi = np.ascontiguousarray(vec[:, :6].T)
    out = lo.lobpcg(*ham_args(w), psi, 1, 2)
    assert np.abs(out["lam"] - ev[:6]).max() <= 1e-10 * np.abs(ev).max()
    assert out["resid"].max() <= 1e-8
    p_ref = vec[:, :6] @ vec[:, :6].conj().T
    assert np.abs(out["psi"].T @ out["psi"].conj() - p_ref).max() <= 1e-8


# ---- Algorithm 11 with the PAW overlap S (lobpcg_gen) ----------------------------------------------------------------------
def dense_hs(w, off, db, qb):
    from oracle import paw
    hd = oracle.dense_h(w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, None, None)
    p = w.proj                                           # (nproj, npw): p[i, G] = P[G, i]
    hd = hd + p.T @ paw.blockdiag_dense(off, db) @ p.conj()
    sd = np.eye(w.npw) + p.T @ paw.blockdiag_dense(off, qb) @ p.conj()
    return hd, sd


def gen_args(w, off, db, qb):
    return (w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, w.proj, off, db, qb)


def test_gen_reduces_to_the_s_identity_oracle_for_diagonal_d_and_zero_q(cfg1):
    """Q = 0 and diagonal D blocks: S = I, and every step of lobpcg_gen must reproduce lobpcg (separately pinned above)."""
    w = cfg1
    off = np.arange(0, w.nproj + 1, 4, dtype=np.int32)
    db = [np.diag(w.dij[lo_:lo_ + 4]).astype(np.complex128) for lo_ in off[:-1]]
    qb = [np.zeros((4, 4), dtype=np.complex128) for _ in off[:-1]]
    a = lo.lobpcg_gen(*gen_args(w, off, db, qb), w.psi, 2, 3)
    b = lo.lobpcg(*ham_args(w), w.psi, 2, 3)
    assert np.abs(a["lam"] - b["lam"]).max() <= 1e-10 * np.abs(b["lam"]).max()
    assert np.abs(a["resid"] - b["resid"]).max() <= 1e-8 * max(b["resid"].max(), 1e-3)
    assert np.abs(a["spsi"] - a["psi"]).max() <= 1e-13
    for ha, hb in zip(a["history"], b["history"]):
        for na, nb in zip(ha, hb):
            assert np.abs(na - nb).max() <= 1e-8 * max(nb.max(), 1e-3)


def test_gen_deflate_and_ortho_properties(cfg1):
    from oracle import paw
    w = cfg1
    off, db, qb = synth.paw_blocks(w.nproj, w.dij, seed=3)
    _, sd = dense_hs(w, off, db, qb)
    x = w.psi[:6]
    hx, sx = paw.apply_hs(*gen_args(w, off, db, qb), x)
    y, hy, sy, u = lo.chol_ortho_gen(x, hx, sx)
    assert np.abs(np.conj(y) @ sd @ y.T - np.eye(6)).max() <= 1e-12        # Y^H S Y = I with the dense S (numpy)
    assert np.abs(np.tril(u, -1)).max() == 0 and np.all(np.diag(u).real > 0)
    assert np.abs(sy - (sd @ y.T).T).max() <= 1e-12                         # S Y is carried along consistently
    z = w.psi[6:10] + 0.25 * y[:4]
    zd = lo.deflate_gen(z, y, sy)
    assert np.abs(np.conj(y) @ sd @ zd.T).max() <= 1e-12                   # S-orthogonal to the basis afterwards
    assert np.abs(lo.deflate_gen(zd, y, sy) - zd).max() <= 1e-12            # idempotent


@pytest.mark.parametrize("nblocks", [1, 2])
def test_gen_converges_to_the_generalised_spectrum(cfg1, nblocks):
    import scipy.linalg as sl
    w = cfg1
    off, db, qb = synth.paw_blocks(w.nproj, w.dij, seed=3)
    hd, sd = dense_hs(w, off, db, qb)
    ev = sl.eigh(hd, sd, eigvals_only=True)
    M = w.psi.shape[0]
    out = lo.lobpcg_gen(*gen_args(w, off, db, qb), w.psi, nblocks, 14)
    lam = out["lam"]
    assert np.all(lam >= ev[:M] - 1e-10)                                   # Ritz values bound the spectrum from above
    assert np.abs(lam[: M // 2] - ev[: M // 2]).max() <= 1e-5 * np.abs(ev).max()
    assert out["resid"][: M // 2].max() <= 1e-3
    assert np.abs(np.conj(out["psi"]) @ sd @ out["psi"].T - np.eye(M)).max() <= 1e-10   # S-orthonormal Ritz vectors
    first = np.max(out["history"][0][0])
    last = np.max(out["history"][0][-1])
    assert last < 0.05 * first                                             # the residuals do come down


def test_gen_exact_invariant_subspace_is_a_fixed_point(cfg1):
    import scipy.linalg as sl
    w = cfg1
    off, db, qb = synth.paw_blocks(w.nproj, w.dij, seed=3)
    hd, sd = dense_hs(w, off, db, qb)
    ev, v = sl.eigh(hd, sd)
    psi = np.ascontiguousarray(v[:, :4].T)                                 # exact generalised eigenvectors, S-orthonormal
    out = lo.lobpcg_gen(*gen_args(w, off, db, qb), psi, 1, 2)
    assert np.abs(out["lam"] - ev[:4]).max() <= 1e-11 * np.abs(ev).max()
    assert out["history"][0][0].max() <= 1e-10

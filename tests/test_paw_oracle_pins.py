"""Pins of the PAW-style generalised-problem oracle (oracle/paw_oracle.py): special cases that reduce to
the already pinned S = I oracle, dense matrices built with numpy, the Sherman-Morrison closed form, exact generalised
eigenvectors (scipy) through the filter's closed form.  CPU only; nothing here compares the oracle with itself."""
import math

import numpy as np
import pytest
import scipy.linalg as sl

import oracle
from oracle import paw, rr
from paper_2604_11139_b200 import synth


def ham_args(w):
    return (w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, w.proj)


def dense_hs(w, off, db, qb):
    hd = oracle.dense_h(w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, None, None)
    p = w.proj                                           # (nproj, npw): p[i, G] = P[G, i]
    hd = hd + p.T @ paw.blockdiag_dense(off, db) @ p.conj()
    sd = np.eye(w.npw) + p.T @ paw.blockdiag_dense(off, qb) @ p.conj()
    return hd, sd


@pytest.fixture(scope="module")
def small():
    w = synth.random_problem((8, 6, 10), (5.0, 4.0, 6.0), (0.25, 0.0, -0.125), 4.0, 11, 5, seed=300)
    off, db, qb = synth.paw_blocks(w.nproj, w.dij, seed=1)
    return w, off, db, qb


def test_blocks_are_hermitian_and_cover_the_projectors(cfg1):
    off, db, qb = synth.paw_blocks(cfg1.nproj, cfg1.dij, seed=0)
    assert off[0] == 0 and off[-1] == cfg1.nproj and np.all(np.diff(off) > 0)
    for d, q in zip(db, qb):
        assert np.abs(d - d.conj().T).max() == 0 and np.abs(q - q.conj().T).max() == 0
    off2, _, _ = synth.paw_blocks(11, np.zeros(11), seed=0)
    assert list(np.diff(off2)) == [4, 1, 5, 1]


def test_reduces_to_the_pinned_oracle_for_diagonal_d_and_zero_q(cfg1):
    """Diagonal D blocks and Q = 0: H psi must equal the (separately pinned) S = I oracle's, S psi = psi, S^-1 = identity."""
    w = cfg1
    off = np.arange(0, w.nproj + 1, 4, dtype=np.int32)
    db = [np.diag(w.dij[lo:lo + 4]).astype(np.complex128) for lo in off[:-1]]
    qb = [np.zeros((4, 4), dtype=np.complex128) for _ in off[:-1]]
    h, s = paw.apply_hs(*ham_args(w), off, db, qb, w.psi)
    ref = oracle.apply_h(*ham_args(w), w.dij, w.psi)
    assert np.abs(h - ref).max() <= 1e-12 * np.abs(ref).max()
    assert np.array_equal(s, w.psi)
    assert np.abs(paw.apply_sinv(w.proj, off, qb, w.psi) - w.psi).max() == 0
    y = paw.cheb_filter_gen(*ham_args(w), off, db, qb, w.psi, 5, w.a, w.b, w.a0)
    ref_y = oracle.cheb_filter(*ham_args(w), w.dij, w.psi, 5, w.a, w.b, w.a0)
    assert np.abs(y - ref_y).max() <= 1e-11 * np.abs(ref_y).max()


def test_apply_hs_against_dense_matrices(small):
    w, off, db, qb = small
    hd, sd = dense_hs(w, off, db, qb)
    assert np.abs(hd - hd.conj().T).max() <= 1e-13 and np.abs(sd - sd.conj().T).max() <= 1e-13
    assert np.linalg.eigvalsh(sd).min() > 0.5                      # S is positive definite
    h, s = paw.apply_hs(*ham_args(w), off, db, qb, w.psi)
    assert np.abs(h - (hd @ w.psi.T).T).max() <= 1e-12 * np.abs(h).max()
    assert np.abs(s - (sd @ w.psi.T).T).max() <= 1e-12 * np.abs(s).max()
    # off-diagonal block entries matter: zeroing them changes the result
    db0 = [np.diag(np.diag(d)) for d in db]
    h0, _ = paw.apply_hs(*ham_args(w), off, db0, qb, w.psi)
    assert np.abs(h - h0).max() > 1e-3 * np.abs(h).max()


def test_sinv_closed_form_dense_solve_and_identity(small):
    w, off, db, qb = small
    _, sd = dense_hs(w, off, db, qb)
    x = w.psi
    y = paw.apply_sinv(w.proj, off, qb, x)
    assert np.abs(y - np.linalg.solve(sd, x.T).T).max() <= 1e-12 * np.abs(y).max()       # library special case
    _, sy = paw.apply_hs(*ham_args(w), off, db, qb, y)
    assert np.abs(sy - x).max() <= 1e-12 * np.abs(x).max()                                # S S^-1 = I
    # one projector: Sherman-Morrison, S^-1 = I - q / (1 + q |p|^2) |p><p|
    p = w.proj[:1]
    q = 0.7
    y1 = paw.apply_sinv(p, np.array([0, 1]), [np.array([[q]])], x)
    coef = q / (1.0 + q * np.vdot(p[0], p[0]).real)
    ref = x - coef * (x @ p[0].conj())[:, None] * p[0][None, :]
    assert np.abs(y1 - ref).max() <= 1e-14 * np.abs(ref).max()
    # a singular Q (a zero block) is fine for the push-through form
    qz = [qb[0]] + [np.zeros_like(b) for b in qb[1:]]
    _, sdz = np.eye(w.npw), None
    sz = np.eye(w.npw) + w.proj.T @ paw.blockdiag_dense(off, qz) @ w.proj.conj()
    yz = paw.apply_sinv(w.proj, off, qz, x)
    assert np.abs(yz - np.linalg.solve(sz, x.T).T).max() <= 1e-12 * np.abs(yz).max()


def test_filter_scales_exact_generalised_eigenvectors_by_the_closed_form(small):
    w, off, db, qb = small
    hd, sd = dense_hs(w, off, db, qb)
    ev, vec = sl.eigh(hd, sd)                                   # H v = lambda S v  (LAPACK)
    a0, a, b = ev[0] - 0.1, ev[len(ev) // 3], ev[-1] + 0.1
    e, c = 0.5 * (b - a), 0.5 * (b + a)
    for m in (1, 2, 5, 9):
        for i in (0, 1, 3):
            v = np.ascontiguousarray(vec[:, i][None, :])
            y = paw.cheb_filter_gen(*ham_args(w), off, db, qb, v, m, a, b, a0)
            tm = lambda t: math.cosh(m * math.acosh(-t)) * (-1) ** m if t < -1 else math.cos(m * math.acos(t))
            rho = tm((ev[i] - c) / e) / tm((a0 - c) / e)
            assert np.abs(y - rho * v).max() <= 1e-9 * abs(rho) * np.abs(v).max(), (m, i)
    assert np.array_equal(paw.cheb_filter_gen(*ham_args(w), off, db, qb, w.psi, 0, a, b, a0), w.psi)


def test_rayleigh_ritz_gen_on_an_invariant_subspace(small):
    w, off, db, qb = small
    hd, sd = dense_hs(w, off, db, qb)
    ev, vec = sl.eigh(hd, sd)
    sel = [0, 1, 2, 6]
    rng = np.random.default_rng(3)
    mix = rng.standard_normal((4, 4)) + 1j * rng.standard_normal((4, 4)) + 2 * np.eye(4)
    psi = np.ascontiguousarray((vec[:, sel] @ mix).T)
    h, s = paw.apply_hs(*ham_args(w), off, db, qb, psi)
    rq = paw.rayleigh_gen(psi, h, s)
    assert np.all(rq >= ev[0] - 1e-10) and np.all(rq <= ev[-1] + 1e-10)
    lam, y, hy, sy, x = paw.rayleigh_ritz_gen(psi, h, s)
    assert np.abs(lam - ev[sel]).max() <= 1e-10 * np.abs(ev).max()
    assert np.abs(y.conj() @ sy.T - np.eye(4)).max() <= 1e-10            # S-orthonormal Ritz vectors
    _, norms = paw.residual_gen(y, hy, sy, lam)
    assert norms.max() <= 1e-9 * np.abs(ev).max()
    # Rayleigh quotient of an exact generalised eigenvector is its eigenvalue
    v = np.ascontiguousarray(vec[:, 2][None, :])
    hv, sv = paw.apply_hs(*ham_args(w), off, db, qb, v)
    assert paw.rayleigh_gen(v, hv, sv)[0] == pytest.approx(ev[2], abs=1e-11)


def test_chebfi_iteration_gen_converges_to_the_generalised_spectrum(small):
    w, off, db, qb = small
    hd, sd = dense_hs(w, off, db, qb)
    ev = sl.eigh(hd, sd, eigvals_only=True)
    b = ev[-1] + 0.5
    psi = w.psi
    prev = None
    for _ in range(5):
        out = paw.chebfi_iteration_gen(*ham_args(w), off, db, qb, psi, 6, b, a0_margin=0.05)
        lam = out["lam"]
        assert np.all(lam >= ev[: len(lam)] - 1e-9)                      # Ritz values bound the spectrum from above
        if prev is not None:
            assert np.all(lam <= prev + 1e-9)
        prev, psi = lam, out["psi"]
    assert np.abs(lam[:3] - ev[:3]).max() < 1e-3

"""Pins of the Rayleigh-Ritz oracle (oracle/rr_oracle.c, oracle/rr_oracle.py) against what the mathematics and the paper
fix -- closed forms, invariants, textbook special cases and library routines -- so that a plausible mistake anywhere in
it (a missing conjugate, a transposed operand, a wrong sign in the rotation, an unsorted spectrum) fails one of them.
None of these tests compares the oracle with itself or with the CUDA path.  CPU only.
"""
import math

import numpy as np
import pytest

import oracle
from oracle import rr
from paper_2604_11139_b200 import synth


def rand_herm(n, seed, scale=1.0):
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    return scale * (a + a.conj().T) / 2.0


def rand_block(nb, npw, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((nb, npw)) + 1j * rng.standard_normal((nb, npw))


def ham_args(w):
    return (w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, w.proj, w.dij)


# ----------------------------------------------------------------------------------------------------------------
# Rayleigh quotients (Algorithm 12 line 3)
# ----------------------------------------------------------------------------------------------------------------
def test_rayleigh_plane_waves_constant_potential(cfg1):
    """A plane wave in a constant potential V0 without projectors is an eigenvector: its Rayleigh quotient is the closed
    form 1/2|k+G|^2 + V0, whatever its norm and phase."""
    w = cfg1
    v0 = 0.37
    vloc = np.full_like(w.vloc, v0)
    idx = [0, 5, 100, w.npw - 1]
    psi = np.zeros((len(idx), w.npw), dtype=np.complex128)
    for r, g in enumerate(idx):
        psi[r, g] = (2.0 + r) * np.exp(0.7j * r)
    hpsi = oracle.apply_h(w.lattice, w.kpt, w.fft_dims, w.gvec, vloc, None, None, psi)
    lam, nrm2 = rr.rayleigh(psi, hpsi)
    b = 2.0 * math.pi / 10.26                                    # cubic cell of cfg 1 (BASELINE.json)
    closed = 0.5 * b * b * (w.gvec[idx].astype(float) ** 2).sum(axis=1) + v0
    assert np.abs(lam - closed).max() <= 1e-13 * closed.max()
    assert np.allclose(nrm2, [(2.0 + r) ** 2 for r in range(len(idx))], rtol=1e-15)


def test_rayleigh_of_dense_eigenvectors_and_bounds(cfg1):
    """Rayleigh quotients of exact eigenvectors of the dense H are its eigenvalues (numpy.linalg.eigh on oracle.dense_h);
    for any vector the quotient lies inside [lambda_min, lambda_max]; it is invariant under scaling by a complex number."""
    w = cfg1
    hd = oracle.dense_h(*ham_args(w))
    ev, vec = np.linalg.eigh(hd)
    psi = np.ascontiguousarray(vec[:, :7].T)
    lam, _ = rr.rayleigh(psi, np.ascontiguousarray((hd @ psi.T).T))
    assert np.abs(lam - ev[:7]).max() <= 1e-12 * np.abs(ev).max()
    x = rand_block(5, w.npw, 3)
    hx = np.ascontiguousarray((hd @ x.T).T)
    lam, _ = rr.rayleigh(x, hx)
    assert np.all(lam >= ev[0] - 1e-12) and np.all(lam <= ev[-1] + 1e-12)
    lam2, _ = rr.rayleigh((3.0 - 2.0j) * x, (3.0 - 2.0j) * hx)
    assert np.abs(lam - lam2).max() <= 1e-13 * np.abs(lam).max()
    # hand-computed 2-component case: psi = (1, i), H psi = (2, 3i)  ->  (1*2 + (-i)(3i)) / 2 = 5/2
    lam3, _ = rr.rayleigh(np.array([[1.0, 1.0j]]), np.array([[2.0, 3.0j]]))
    assert lam3[0] == pytest.approx(2.5, abs=1e-15)


# ----------------------------------------------------------------------------------------------------------------
# rotations (Algorithm 5 steps 4-5)
# ----------------------------------------------------------------------------------------------------------------
def test_rotate_permutation_givens_and_numpy():
    x = rand_block(6, 37, 1)
    perm = [3, 0, 5, 1, 4, 2]
    q = np.zeros((6, 6))
    for j, i in enumerate(perm):
        q[i, j] = 1.0                                   # column j of Q picks band perm[j]
    assert np.array_equal(rr.rotate(x, q), x[perm])
    # a complex Givens rotation of bands 1 and 4: closed form
    c, s, ph = math.cos(0.3), math.sin(0.3), np.exp(0.9j)
    g = np.eye(6, dtype=np.complex128)
    g[1, 1], g[4, 1], g[1, 4], g[4, 4] = c, -s * np.conj(ph), s, c * np.conj(ph)
    y = rr.rotate(x, g)
    assert np.abs(y[1] - (c * x[1] - s * np.conj(ph) * x[4])).max() <= 1e-15
    assert np.abs(y[4] - (s * x[1] + c * np.conj(ph) * x[4])).max() <= 1e-15
    assert np.array_equal(y[[0, 2, 3, 5]], x[[0, 2, 3, 5]])
    # rectangular Q, orientation (no transpose, no conjugate) against numpy
    q2 = rand_block(6, 4, 2)                             # 6 x 4 matrix
    assert np.abs(rr.rotate(x, q2) - (q2.T @ x)).max() <= 1e-13


# ----------------------------------------------------------------------------------------------------------------
# residuals (Algorithm 12 lines 11-12)
# ----------------------------------------------------------------------------------------------------------------
def test_residual_zero_on_eigenvectors_and_closed_form_when_perturbed(cfg1):
    w = cfg1
    hd = oracle.dense_h(*ham_args(w))
    ev, vec = np.linalg.eigh(hd)
    psi = np.ascontiguousarray(vec[:, :5].T)
    hpsi = oracle.apply_h(*ham_args(w), psi)
    _, norms = rr.residual(psi, hpsi, ev[:5])
    assert norms.max() <= 1e-11 * np.abs(ev).max()
    # psi = v_i + eps v_j with lambda = lambda_i:  W = eps (lambda_j - lambda_i) v_j,  ||W|| = |eps| |lambda_j - lambda_i|
    eps = 1e-3 * np.exp(0.4j)
    i, j = 2, 40
    p = (vec[:, i] + eps * vec[:, j])[None, :]
    hp = oracle.apply_h(*ham_args(w), p)
    wres, norms = rr.residual(p, hp, np.array([ev[i]]))
    assert norms[0] == pytest.approx(abs(eps) * abs(ev[j] - ev[i]), rel=1e-9)
    assert np.abs(wres[0] - eps * (ev[j] - ev[i]) * vec[:, j]).max() <= 1e-11
    # definition on random data
    x, hx, lam = rand_block(3, 11, 5), rand_block(3, 11, 6), np.array([0.5, -1.0, 2.0])
    wres, norms = rr.residual(x, hx, lam)
    assert np.abs(wres - (hx - lam[:, None] * x)).max() <= 1e-15
    assert np.allclose(norms, np.linalg.norm(hx - lam[:, None] * x, axis=1), rtol=1e-14)


# ----------------------------------------------------------------------------------------------------------------
# Cholesky orthonormalisation (Algorithm 9)
# ----------------------------------------------------------------------------------------------------------------
def test_potrf_matches_library_and_hand_example():
    # hand example: [[4, 2i], [-2i, 5]] = U^H U with U = [[2, i], [0, 2]]
    u = rr.potrf_upper(np.array([[4.0, 2.0j], [-2.0j, 5.0]]))
    assert np.abs(u - np.array([[2.0, 1.0j], [0.0, 2.0]])).max() <= 1e-15
    for n, seed in ((1, 0), (7, 1), (64, 2), (130, 3)):
        x = rand_block(n, n + 5, seed)
        s = x @ x.conj().T
        u = rr.potrf_upper(s)
        assert np.allclose(np.tril(u, -1), 0.0) and np.all(np.diag(u).real > 0) and np.all(np.diag(u).imag == 0)
        assert np.abs(u - np.linalg.cholesky(s).conj().T).max() <= 1e-12 * np.abs(s).max()      # library special case
        assert np.abs(u.conj().T @ u - s).max() <= 1e-12 * np.abs(s).max()
    with pytest.raises(np.linalg.LinAlgError):
        rr.potrf_upper(np.array([[1.0, 2.0], [2.0, 1.0]]))


def test_chol_ortho_gives_orthonormal_block_with_same_span():
    x = rand_block(9, 200, 11)
    hx = rand_block(9, 200, 12)
    y, hy, u = rr.chol_ortho(x, hx)
    assert np.abs(y @ y.conj().T - np.eye(9)).max() <= 1e-13             # Psi^H Psi = I afterwards
    # Psi = Y U exactly means band j of X = sum_k U[k, j] band k of Y
    assert np.abs(u.T @ y - x).max() <= 1e-12
    assert np.abs(u.T @ hy - hx).max() <= 1e-12                          # the same transformation applied to H Psi
    # upper triangular U: the first band is only rescaled, band j stays in span(x_0..x_j) (Gram-Schmidt property)
    assert np.abs(y[0] - x[0] / np.linalg.norm(x[0])).max() <= 1e-14
    # library: the Q factor of numpy's QR with positive diagonal R
    qm, r = np.linalg.qr(x.T)
    ph = np.diag(r) / np.abs(np.diag(r))
    assert np.abs(y - (qm * ph[None, :]).T).max() <= 1e-12


# ----------------------------------------------------------------------------------------------------------------
# Hermitian eigen-solve (Algorithm 5 / 10 step 3)
# ----------------------------------------------------------------------------------------------------------------
def check_eig(a, w, v, tol=1e-12):
    n = a.shape[0]
    scale = max(np.abs(a).max(), 1e-300)
    assert np.all(np.diff(w) >= 0)
    assert np.abs(v.conj().T @ v - np.eye(n)).max() <= tol * n
    assert np.abs(a @ v - v * w[None, :]).max() <= tol * n * scale


def test_heev_closed_forms():
    # 2 x 2: [[a, g], [conj g, b]] has eigenvalues (a+b)/2 -/+ sqrt(((a-b)/2)^2 + |g|^2)
    a, b, g = 1.5, -0.25, 0.3 - 0.8j
    m = np.array([[a, g], [np.conj(g), b]])
    w, v = rr.heev(m)
    r = math.sqrt(((a - b) / 2) ** 2 + abs(g) ** 2)
    assert np.abs(w - [(a + b) / 2 - r, (a + b) / 2 + r]).max() <= 1e-15
    check_eig(m, w, v)
    # diagonal: sorted diagonal, V a permutation
    d = np.array([3.0, -1.0, 2.0, 0.5])
    w, v = rr.heev(np.diag(d))
    assert np.array_equal(w, np.sort(d)) and np.abs(np.abs(v).sum(axis=0) - 1).max() == 0
    # rank one u u^H: eigenvalues 0 (n-1 times) and |u|^2
    u = np.array([1.0, 2.0j, -1.0 + 1.0j, 0.5, 3.0])
    w, v = rr.heev(np.outer(u, u.conj()))
    assert np.abs(w[:-1]).max() <= 1e-14 and w[-1] == pytest.approx(np.vdot(u, u).real, rel=1e-14)
    # Hermitian circulant: eigenvalues are the DFT of its first column
    n = 12
    c = np.random.default_rng(4).standard_normal(n) + 1j * np.random.default_rng(5).standard_normal(n)
    c[0] = c[0].real
    for k in range(1, n):
        c[n - k] = np.conj(c[k]) if k < n - k else c[n - k]
    if n % 2 == 0:
        c[n // 2] = c[n // 2].real
    circ = np.array([[c[(i - j) % n] for j in range(n)] for i in range(n)])
    assert np.abs(circ - circ.conj().T).max() == 0
    w, v = rr.heev(circ)
    dft = np.array([sum(c[j] * np.exp(-2j * math.pi * j * k / n) for j in range(n)) for k in range(n)])
    assert np.abs(dft.imag).max() <= 1e-13
    assert np.abs(w - np.sort(dft.real)).max() <= 1e-13 * np.abs(c).sum()
    check_eig(circ, w, v)


@pytest.mark.parametrize("n,seed", [(1, 0), (3, 1), (17, 2), (64, 3), (150, 4)])
def test_heev_matches_library(n, seed):
    a = rand_herm(n, seed, scale=3.0)
    w, v = rr.heev(a)
    assert np.abs(w - np.linalg.eigvalsh(a)).max() <= 1e-12 * np.abs(w).max() * max(1.0, math.sqrt(n))
    check_eig(a, w, v)


def test_heev_degenerate_cluster_projector():
    """Degenerate eigenvalues (cubic cells have them): eigenvectors are not unique, the spectral projector is."""
    rng = np.random.default_rng(9)
    qm, _ = np.linalg.qr(rng.standard_normal((10, 10)) + 1j * rng.standard_normal((10, 10)))
    lam = np.array([-2.0, -2.0, -2.0, 0.5, 0.5, 1.0, 3.0, 3.0, 3.0, 3.0])
    a = (qm * lam) @ qm.conj().T
    a = (a + a.conj().T) / 2
    w, v = rr.heev(a)
    assert np.abs(w - lam).max() <= 1e-13
    for lo, hi in ((0, 3), (3, 5), (5, 6), (6, 10)):
        p_ref = qm[:, lo:hi] @ qm[:, lo:hi].conj().T
        p = v[:, lo:hi] @ v[:, lo:hi].conj().T
        assert np.abs(p - p_ref).max() <= 1e-12


def test_heev_on_the_dense_hamiltonian_subspace(cfg1):
    """The matrix the path really feeds it: H_Psi = Psi^H (H Psi) of cfg 1; against numpy.linalg.eigvalsh."""
    w = cfg1
    hpsi = oracle.apply_h(*ham_args(w), w.psi)
    hs = oracle.gram(w.psi, hpsi)
    hs = (hs + hs.conj().T) / 2
    lam, x = rr.heev(hs)
    assert np.abs(lam - np.linalg.eigvalsh(hs)).max() <= 1e-13 * np.abs(lam).max()
    check_eig(hs, lam, x)
    # Ritz values of an orthonormal block interlace the spectrum of the dense H (Cauchy): lam_i >= ev_i
    ev = np.linalg.eigvalsh(oracle.dense_h(*ham_args(w)))
    assert np.all(lam >= ev[: len(lam)] - 1e-10)


def test_hegv_special_cases_and_library():
    import scipy.linalg as sl
    a = rand_herm(20, 1)
    # B = I reduces to the standard problem
    w, x = rr.hegv(a, np.eye(20))
    assert np.abs(w - np.linalg.eigvalsh(a)).max() <= 1e-13 * np.abs(w).max()
    # B = diagonal d: the standard problem of D^-1/2 A D^-1/2
    d = np.random.default_rng(2).uniform(0.5, 3.0, 20)
    w, x = rr.hegv(a, np.diag(d))
    assert np.abs(w - np.linalg.eigvalsh(a / np.sqrt(d[:, None] * d[None, :]))).max() <= 1e-12 * np.abs(w).max()
    # general Hermitian positive definite B: scipy (LAPACK zhegvd), B-orthonormality, residual
    for n, seed in ((5, 3), (48, 4), (130, 5)):
        a = rand_herm(n, seed)
        m = rand_block(n, n, seed + 10)
        b = m @ m.conj().T / n + 0.5 * np.eye(n)
        w, x = rr.hegv(a, b)
        assert np.abs(w - sl.eigh(a, b, eigvals_only=True)).max() <= 1e-11 * np.abs(w).max()
        assert np.abs(x.conj().T @ b @ x - np.eye(n)).max() <= 1e-11
        assert np.abs(a @ x - (b @ x) * w[None, :]).max() <= 1e-11 * np.abs(a).max() * n
    with pytest.raises(np.linalg.LinAlgError):
        rr.hegv(a, -np.eye(a.shape[0]))


# ----------------------------------------------------------------------------------------------------------------
# Rayleigh-Ritz and one whole Chebyshev-filtering iteration (Algorithms 10 and 12)
# ----------------------------------------------------------------------------------------------------------------
def test_rayleigh_ritz_on_an_invariant_subspace(cfg1):
    """A non-orthogonal basis of an exactly invariant subspace: Rayleigh-Ritz returns the exact eigenvalues of that
    subspace, S-orthonormal (here orthonormal) Ritz vectors and zero residuals."""
    w = cfg1
    hd = oracle.dense_h(*ham_args(w))
    ev, vec = np.linalg.eigh(hd)
    sel = [0, 1, 2, 5, 9, 30]
    mix = rand_block(6, 6, 21) + 3 * np.eye(6)
    psi = np.ascontiguousarray((vec[:, sel] @ mix).T)
    hpsi = oracle.apply_h(*ham_args(w), psi)
    lam, y, hy, x = rr.rayleigh_ritz(psi, hpsi)
    assert np.abs(lam - ev[sel]).max() <= 1e-11 * np.abs(ev).max()
    assert np.abs(y @ y.conj().T - np.eye(6)).max() <= 1e-11
    assert np.abs(hy - oracle.apply_h(*ham_args(w), y)).max() <= 1e-10          # H Psi rotated == H applied to rotated Psi
    _, norms = rr.residual(y, hy, lam)
    assert norms.max() <= 1e-10 * np.abs(ev).max()


def test_chebfi_iteration_converges_towards_the_dense_spectrum(cfg1):
    """Algorithm 12 repeated: Ritz values decrease monotonically towards the lowest eigenvalues of the dense H (they
    are upper bounds, Cauchy interlacing) and the residual norms shrink."""
    w = cfg1
    ev = np.linalg.eigvalsh(oracle.dense_h(*ham_args(w)))
    psi = w.psi
    prev_lam, first_res = None, None
    for it in range(4):
        out = rr.chebfi_iteration(*ham_args(w), psi, 8, w.b)
        lam = out["lam"]
        assert np.all(lam >= ev[: len(lam)] - 1e-10)
        assert out["a0"] <= out["rq"].min() and out["a"] == pytest.approx(out["rq"].max())
        if prev_lam is not None:
            assert np.all(lam <= prev_lam + 1e-10)
        prev_lam = lam
        first_res = out["resid"].max() if first_res is None else first_res
        psi = out["psi"]
    assert out["resid"][:8].max() < 0.05 * first_res
    assert np.abs(lam[:8] - ev[:8]).max() < 1e-2

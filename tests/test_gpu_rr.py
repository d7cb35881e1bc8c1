"""GPU parity of the Rayleigh-Ritz companion steps (include/pwham.h, second half) against the CPU
oracle (oracle/rr_oracle.*) on the same seeded inputs.  Unique results (Rayleigh quotients, rotations, residuals, the
Cholesky factor with positive diagonal, eigenvalues) are compared element by element at the north_star tolerance 1e-11;
where several results are correct (eigenvectors: phases, bases of degenerate eigenspaces) the tests compare what is unique
-- eigenvalues, residuals, orthonormality, spectral projectors of eigenvalue clusters -- and check that the rest is valid.
"""
import math

import numpy as np
import pytest

import oracle
from oracle import rr
from paper_2604_11139_b200 import synth

pytestmark = pytest.mark.gpu

TOL = 1e-11


def relerr(x, ref):
    return float(np.linalg.norm(np.asarray(x) - np.asarray(ref)) / max(np.linalg.norm(ref), 1e-300))


def ham_args(w):
    return (w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, w.proj, w.dij)


@pytest.fixture(scope="module")
def gpu():
    import torch
    from paper_2604_11139_b200 import binding
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    binding.load_library()
    return binding


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rand_block(nb, npw, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((nb, npw)) + 1j * rng.standard_normal((nb, npw))


def rand_herm(n, seed):
    a = rand_block(n, n, seed)
    return (a + a.conj().T) / 2


# ----------------------------------------------------------------------------------------------------------------
# column statistics and rotations
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nb,npw", [(1, 1), (5, 257), (16, 7153), (130, 4099)])
def test_rayleigh_quotients_and_residuals(gpu, nb, npw):
    x, hx = rand_block(nb, npw, nb), rand_block(nb, npw, nb + 1)
    lam, mm = gpu.rayleigh_quotients(dev(x), dev(hx))
    lam_ref, _ = rr.rayleigh(x, hx)
    assert np.abs(lam.cpu().numpy() - lam_ref).max() <= TOL * np.abs(lam_ref).max()
    assert mm.cpu().numpy()[0] == lam.cpu().numpy().min() and mm.cpu().numpy()[1] == lam.cpu().numpy().max()
    norms, w = gpu.residual_norms(dev(x), dev(hx), dev(lam_ref), want_w=True)
    w_ref, n_ref = rr.residual(x, hx, lam_ref)
    assert relerr(w.cpu().numpy(), w_ref) <= TOL
    assert np.abs(norms.cpu().numpy() - n_ref).max() <= TOL * n_ref.max()
    only = gpu.residual_norms(dev(x), dev(hx), dev(lam_ref))
    assert np.array_equal(only.cpu().numpy(), norms.cpu().numpy())


def test_rayleigh_quotients_of_the_hamiltonian(gpu, cfg2):
    w = cfg2
    ham = gpu.ham_setup(*ham_args(w))
    psi = dev(w.psi)
    lam, mm = gpu.rayleigh_quotients(psi, gpu.apply_h(ham, psi))
    lam_ref, _ = rr.rayleigh(w.psi, oracle.apply_h(*ham_args(w), w.psi))
    assert np.abs(lam.cpu().numpy() - lam_ref).max() <= TOL * np.abs(lam_ref).max()
    ham.destroy()


@pytest.mark.parametrize("m,n,npw", [(1, 1, 3), (6, 6, 257), (16, 9, 1000), (130, 67, 4099), (128, 128, 7153)])
def test_rotate(gpu, m, n, npw):
    x, q = rand_block(m, npw, m), rand_block(m, n, n + 50)
    y = gpu.rotate(dev(x), dev(q)).cpu().numpy()
    assert y.shape == (n, npw)
    assert relerr(y, rr.rotate(x, q)) <= TOL


# ----------------------------------------------------------------------------------------------------------------
# dense M x M steps
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 5, 32, 33, 100, 257])
def test_potrf(gpu, n):
    x = rand_block(n, n + 7, n)
    s = x @ x.conj().T / n + 0.1 * np.eye(n)
    u, info = gpu.potrf(dev(s))
    u = u.cpu().numpy()
    assert info == 0
    ref = rr.potrf_upper(s)
    assert np.abs(u - ref).max() <= TOL * np.abs(ref).max()
    assert np.all(np.tril(u, -1) == 0) and np.all(np.diag(u).imag == 0) and np.all(np.diag(u).real > 0)


def test_potrf_reports_the_failing_pivot(gpu):
    s = np.eye(40, dtype=np.complex128)
    s[17, 17] = -1.0
    _, info = gpu.potrf(dev(s))
    assert info == 18


def check_eig(a, w, x, w_ref, tol=TOL):
    n = a.shape[0]
    scale = max(np.abs(w_ref).max(), 1e-300)
    assert np.all(np.diff(w) >= 0)
    assert np.abs(w - w_ref).max() <= tol * scale                           # eigenvalues are unique
    assert np.abs(x.conj().T @ x - np.eye(n)).max() <= 1e-12 * max(n, 8)    # any valid eigenbasis is orthonormal ...
    assert np.abs(a @ x - x * w[None, :]).max() <= 1e-12 * max(n, 8) * max(np.abs(a).max(), 1e-300)   # ... and satisfies A x = w x


@pytest.mark.parametrize("n", [1, 2, 3, 17, 64, 129, 300])
def test_heev(gpu, n):
    a = 3.0 * rand_herm(n, n + 3)
    w, x, sweeps = gpu.heev(dev(a))
    w_ref, _ = rr.heev(a)
    check_eig(a, w.cpu().numpy(), x.cpu().numpy(), w_ref)
    assert n == 1 or 0 < sweeps < 40


def test_heev_degenerate_clusters_and_indefinite_spectrum(gpu):
    """Degenerate eigenvalues (cubic cells have them) and a spectrum symmetric about zero (+lambda and -lambda both present):
    eigenvalues and the spectral projector of every cluster against the oracle's."""
    rng = np.random.default_rng(9)
    qm, _ = np.linalg.qr(rng.standard_normal((12, 12)) + 1j * rng.standard_normal((12, 12)))
    lam = np.array([-3.0, -3.0, -3.0, -3.0, -1.0, -1.0, 0.0, 1.0, 1.0, 3.0, 3.0, 3.0])
    a = (qm * lam) @ qm.conj().T
    a = (a + a.conj().T) / 2
    w, x, _ = gpu.heev(dev(a))
    w, x = w.cpu().numpy(), x.cpu().numpy()
    w_ref, v_ref = rr.heev(a)
    check_eig(a, w, x, w_ref)
    for lo, hi in ((0, 4), (4, 6), (6, 7), (7, 9), (9, 12)):
        p_ref = v_ref[:, lo:hi] @ v_ref[:, lo:hi].conj().T
        assert np.abs(x[:, lo:hi] @ x[:, lo:hi].conj().T - p_ref).max() <= 1e-11


def test_heev_on_the_subspace_hamiltonian(gpu, cfg2):
    """The matrix the path feeds it: H_Psi = Psi^H (H Psi) of cfg 2 (128 x 128)."""
    w = cfg2
    hs = oracle.gram(w.psi, oracle.apply_h(*ham_args(w), w.psi))
    hs = (hs + hs.conj().T) / 2
    lam, x, _ = gpu.heev(dev(hs))
    lam_ref, _ = rr.heev(hs)
    check_eig(hs, lam.cpu().numpy(), x.cpu().numpy(), lam_ref)


@pytest.mark.parametrize("n", [1, 4, 33, 128, 200])
def test_hegv(gpu, n):
    a = rand_herm(n, n)
    m = rand_block(n, n, n + 11)
    b = m @ m.conj().T / n + 0.5 * np.eye(n)
    w, x, info = gpu.hegv(dev(a), dev(b))
    w, x = w.cpu().numpy(), x.cpu().numpy()
    w_ref, _ = rr.hegv(a, b)
    assert info >= 0
    assert np.abs(w - w_ref).max() <= TOL * max(np.abs(w_ref).max(), 1.0) * 10
    assert np.abs(x.conj().T @ b @ x - np.eye(n)).max() <= 1e-11 * max(n, 8)
    assert np.abs(a @ x - (b @ x) * w[None, :]).max() <= 1e-11 * max(n, 8) * np.abs(a).max()


def test_hegv_flags_an_indefinite_overlap(gpu):
    a = rand_herm(20, 1)
    b = np.eye(20, dtype=np.complex128)
    b[5, 5] = -2.0
    _, _, info = gpu.hegv(dev(a), dev(b))
    assert info == -6


# ----------------------------------------------------------------------------------------------------------------
# N x M steps: Cholesky orthonormalisation, Rayleigh-Ritz, one Chebyshev-filtering iteration
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nb,npw", [(1, 9), (9, 200), (67, 4099), (128, 7153)])
def test_chol_ortho(gpu, nb, npw):
    x, hx = rand_block(nb, npw, nb), rand_block(nb, npw, nb + 1)
    xd, hxd = dev(x), dev(hx)
    u, info = gpu.chol_ortho(xd, hxd)
    y_ref, hy_ref, u_ref = rr.chol_ortho(x, hx)
    assert info == 0
    assert np.abs(u.cpu().numpy() - u_ref).max() <= TOL * np.abs(u_ref).max()      # unique: positive diagonal
    assert relerr(xd.cpu().numpy(), y_ref) <= TOL * 100                           # cond(U) enters the solve
    assert relerr(hxd.cpu().numpy(), hy_ref) <= TOL * 100
    y = xd.cpu().numpy()
    assert np.abs(y @ y.conj().T - np.eye(nb)).max() <= 1e-12 * max(nb, 8)


def ritz_checks(psi0, hpsi0, lam, y, hy, lam_ref, y_ref, tol=1e-10):
    """What is unique about a Rayleigh-Ritz result: the Ritz values; the rotated blocks span the input span with Psi^H Psi
    = I and Psi^H (H Psi) = diag(lambda); the projector on each cluster of Ritz vectors."""
    nb = len(lam)
    scale = np.abs(lam_ref).max()
    assert np.abs(lam - lam_ref).max() <= tol * scale
    assert np.abs(y @ y.conj().T - np.eye(nb)).max() <= tol * nb
    assert np.abs(y.conj() @ hy.T - np.diag(lam)).max() <= tol * nb * scale
    # same span: projecting the oracle's Ritz vectors on the GPU's leaves them unchanged
    assert np.abs(y_ref - (y_ref @ y.conj().T) @ y).max() <= tol * nb
    # clusters (gaps > 1e-6 scale) : projector against the oracle's
    cuts = [0] + [i + 1 for i in range(nb - 1) if lam_ref[i + 1] - lam_ref[i] > 1e-6 * scale] + [nb]
    for lo, hi in zip(cuts[:-1], cuts[1:]):
        p = y[lo:hi].T @ y[lo:hi].conj()
        p_ref = y_ref[lo:hi].T @ y_ref[lo:hi].conj()
        assert np.abs(p - p_ref).max() <= 1e-7


@pytest.mark.parametrize("cfg,nb", [("cfg1", 16), ("cfg2", 48)])
def test_rayleigh_ritz(gpu, cfg, nb, request):
    w = request.getfixturevalue(cfg)
    rng = np.random.default_rng(5)
    mix = rng.standard_normal((nb, nb)) + 1j * rng.standard_normal((nb, nb)) + 2 * np.eye(nb)
    psi0 = np.ascontiguousarray(mix @ w.psi[:nb])                      # a non-orthonormal basis
    hpsi0 = oracle.apply_h(*ham_args(w), psi0)
    psi, hpsi = dev(psi0), dev(hpsi0)
    lam, info = gpu.rayleigh_ritz(psi, hpsi)
    lam_ref, y_ref, hy_ref, _ = rr.rayleigh_ritz(psi0, hpsi0)
    assert info > 0
    y, hy = psi.cpu().numpy(), hpsi.cpu().numpy()
    ritz_checks(psi0, hpsi0, lam.cpu().numpy(), y, hy, lam_ref, y_ref)
    assert relerr(hy, oracle.apply_h(*ham_args(w), y)) <= 1e-9          # H Psi rotated == H applied to the rotated Psi


@pytest.mark.parametrize("cfg,degree", [("cfg1", 4), ("cfg2", 8)])
def test_chebfi_iteration(gpu, cfg, degree, request):
    """Algorithm 12, whole: bounds from Rayleigh quotients, filter, Rayleigh-Ritz, residuals -- twice in a row."""
    import torch
    w = request.getfixturevalue(cfg)
    ham = gpu.ham_setup(*ham_args(w))
    nb = min(40, w.psi.shape[0])                  # the oracle filters at ~25 band-applications/s on cfg 2
    psi = dev(w.psi[:nb])
    hpsi = torch.empty_like(psi)
    psi_ref = np.ascontiguousarray(w.psi[:nb])
    for it in range(2):
        out = gpu.chebfi_iteration(ham, psi, hpsi, degree, w.b, a0_margin=0.01, block=24)
        ref = rr.chebfi_iteration(*ham_args(w), psi_ref, degree, w.b, a0_margin=0.01)
        assert out["info"] > 0
        assert out["a"] == pytest.approx(ref["a"], rel=1e-12) and out["a0"] == pytest.approx(ref["a0"], rel=1e-12)
        y, hy = psi.cpu().numpy(), hpsi.cpu().numpy()
        ritz_checks(None, None, out["lam"].cpu().numpy(), y, hy, ref["lam"], ref["psi"], tol=1e-9)
        scale = np.abs(ref["lam"]).max()
        assert np.abs(out["resid"].cpu().numpy() - ref["resid"]).max() <= 1e-8 * scale
        psi_ref = ref["psi"]
    ham.destroy()

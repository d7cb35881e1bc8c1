"""GPU parity of pwh_lobpcg (Algorithm 11 of the paper with S = I) against the CPU
oracle (oracle/lobpcg_oracle.py) on the same seeded inputs.

LOBPCG is an iteration whose intermediate bases are not unique (phases of Ritz vectors; mixing inside degenerate Ritz
clusters, which also changes the per-band preconditioner), so the tests run on unstructured problems without symmetry
(general k-point, random V_loc, dense random projectors: no degenerate levels) and compare what is unique: the Ritz values,
the residual norms of every line minimisation (invariant under phases), the final residual norms, and the Ritz vectors up to
a phase per band (through orthonormality, the span and the per-cluster projectors).  Tolerances: 1e-9 relative on the Ritz
values and 1e-8 on norms and projectors -- a handful of line minimisations from a random start keep every Cholesky / Ritz
step well conditioned, so rounding-order differences (1e-15 per step) stay far below them."""
import numpy as np
import pytest

import oracle
from oracle import lobpcg_oracle as lo
from paper_2604_11139_b200 import synth

pytestmark = pytest.mark.gpu


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


PROBLEMS = {
    "box30": ((30, 20, 24), (11.0, 8.0, 9.0), (0.25, 0.125, -0.375), 5.0, 9, 12, 401),
    "box48": ((48, 48, 36), (20.0, 20.0, 15.0), (0.125, 0.25, 0.0625), 3.0, 20, 24, 402),
    "tric": ((24, 24, 30), ((9.0, 0.0, 0.0), (1.5, 8.5, 0.0), (-1.0, 2.0, 10.0)), (0.1, 0.2, 0.3), 5.0, 7, 8, 403),
}


def problem(name):
    dims, cell, kpt, ecut, nproj, nband, seed = PROBLEMS[name]
    return synth.random_problem(dims, np.asarray(cell) if np.ndim(cell) == 2 else cell, kpt, ecut, nproj, nband, seed=seed)


def compare(out, ref, y, hy, w, tol_vec=1e-8):
    lam, lam_ref = out["lam"].cpu().numpy(), ref["lam"]
    nb = len(lam_ref)
    scale = np.abs(lam_ref).max()
    assert np.abs(lam - lam_ref).max() <= 1e-9 * scale
    assert np.abs(out["resid"].cpu().numpy() - ref["resid"]).max() <= 1e-8 * scale
    hist = out["history"].cpu().numpy()
    for i, per_block in enumerate(ref["history"]):
        for n, norms in enumerate(per_block):
            assert np.abs(hist[i, n] - norms).max() <= 1e-8 * scale, (i, n)
        assert np.isnan(hist[i, len(per_block):]).all()                     # passes the early exit skipped stay untouched
    assert np.abs(y @ y.conj().T - np.eye(nb)).max() <= 1e-10 * nb           # Psi^H Psi = I
    assert np.abs(y.conj() @ hy.T - np.diag(lam)).max() <= 1e-9 * nb * scale   # Psi^H H Psi = Lambda
    assert np.linalg.norm(hy - oracle.apply_h(*ham_args(w), y)) <= 1e-9 * np.linalg.norm(hy)   # hpsi really is H psi
    y_ref = ref["psi"]
    gaps = np.diff(lam_ref)
    assert gaps.min() > 1e-4 * scale, "test problem has (nearly) degenerate levels: pick another seed"
    for b in range(nb):                                                      # band by band, up to a phase
        ph = np.vdot(y_ref[b], y[b])
        assert abs(abs(ph) - 1.0) <= tol_vec / gaps.min() * scale
        assert np.abs(y[b] - ph / abs(ph) * y_ref[b]).max() <= tol_vec / gaps.min() * scale


@pytest.mark.parametrize("name,nblocks,nline", [("box30", 1, 4), ("box30", 3, 3), ("box48", 2, 3), ("tric", 1, 5),
                                                ("tric", 4, 2), ("box30", 1, 0), ("box30", 12, 2)])
def test_lobpcg_matches_oracle(gpu, name, nblocks, nline):
    import torch
    w = problem(name)
    ham = gpu.ham_setup(*ham_args(w))
    psi = dev(w.psi)
    hpsi = torch.empty_like(psi)
    out = gpu.lobpcg(ham, psi, hpsi, nblocks, nline)
    ref = lo.lobpcg(*ham_args(w), w.psi, nblocks, nline)
    assert out["info"] > 0
    compare(out, ref, psi.cpu().numpy(), hpsi.cpu().numpy(), w)
    ham.destroy()


def test_lobpcg_early_exit_and_convergence(gpu):
    """tol > 0: a block stops once its residuals are below tol (Algorithm 11 line 12); run to convergence, the Ritz values are
    the lowest eigenvalues of the dense H (numpy on oracle.dense_h) and the pass counts equal the oracle's."""
    import torch
    w = problem("tric")
    ham = gpu.ham_setup(*ham_args(w))
    psi = dev(w.psi)
    hpsi = torch.empty_like(psi)
    tol = 1e-6
    out = gpu.lobpcg(ham, psi, hpsi, 1, 60, tol=tol)
    ref = lo.lobpcg(*ham_args(w), w.psi, 1, 60, tol=tol)
    hist = out["history"].cpu().numpy()[0]
    used = int((~np.isnan(hist[:, 0])).sum())
    assert used == len(ref["history"][0]) and used < 60
    assert out["resid"].cpu().numpy().max() <= 2 * tol
    ev = np.linalg.eigvalsh(oracle.dense_h(*ham_args(w)))[: w.psi.shape[0]]
    assert np.abs(out["lam"].cpu().numpy() - ev).max() <= 1e-10 * np.abs(ev).max()
    ham.destroy()


def test_lobpcg_padded_leading_dimensions_and_errors(gpu):
    import torch
    w = problem("box30")
    ham = gpu.ham_setup(*ham_args(w))
    nb, npw = w.psi.shape
    big = torch.full((nb, npw + 7), 7.0 + 0j, dtype=torch.complex128, device="cuda")
    big[:, :npw] = dev(w.psi)
    hbig = torch.full((nb, npw + 3), 5.0 + 0j, dtype=torch.complex128, device="cuda")
    out = gpu.lobpcg(ham, big[:, :npw], hbig[:, :npw], 2, 2)
    ref = lo.lobpcg(*ham_args(w), w.psi, 2, 2)
    compare(out, ref, big[:, :npw].cpu().numpy(), hbig[:, :npw].cpu().numpy(), w)
    assert (big[:, npw:] == 7.0).all() and (hbig[:, npw:] == 5.0).all()      # padding rows untouched
    with pytest.raises(gpu.PwhamError):
        gpu.lobpcg(ham, dev(w.psi), torch.empty_like(dev(w.psi)), 5, 1)      # 12 bands do not split into 5 blocks
    ham.destroy()


# ---- Algorithm 11 with the PAW overlap S (pwh_lobpcg_gen) ---------------------------------------------------------------------
def gen_setup(gpu, w, seed):
    off, db, qb = synth.paw_blocks(w.nproj, w.dij, seed=seed)
    ham = gpu.ham_setup(*ham_args(w))
    assert gpu.ham_set_paw(ham, off, db, qb) == 0
    return ham, (w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, w.proj, off, db, qb)


def compare_gen(out, ref, y, hy, sy, gargs):
    from oracle import paw
    lam, lam_ref = out["lam"].cpu().numpy(), ref["lam"]
    nb = len(lam_ref)
    scale = np.abs(lam_ref).max()
    assert np.abs(lam - lam_ref).max() <= 1e-9 * scale
    assert np.abs(out["resid"].cpu().numpy() - ref["resid"]).max() <= 1e-8 * scale
    hist = out["history"].cpu().numpy()
    for i, per_block in enumerate(ref["history"]):
        for n, norms in enumerate(per_block):
            assert np.abs(hist[i, n] - norms).max() <= 1e-8 * scale, (i, n)
    assert np.abs(y.conj() @ sy.T - np.eye(nb)).max() <= 1e-10 * nb          # Psi^H S Psi = I
    assert np.abs(y.conj() @ hy.T - np.diag(lam)).max() <= 1e-9 * nb * scale  # Psi^H H Psi = Lambda
    h_ref, s_ref = paw.apply_hs(*gargs, y)
    assert np.linalg.norm(hy - h_ref) <= 1e-9 * np.linalg.norm(h_ref)          # hpsi, spsi really are H psi, S psi
    assert np.linalg.norm(sy - s_ref) <= 1e-9 * np.linalg.norm(s_ref)
    y_ref, sy_ref = ref["psi"], ref["spsi"]
    gaps = np.diff(lam_ref)
    assert gaps.min() > 1e-4 * scale, "test problem has (nearly) degenerate levels: pick another seed"
    for b in range(nb):                                                      # band by band, up to a phase (S inner product)
        ph = np.vdot(sy_ref[b], y[b])
        assert abs(abs(ph) - 1.0) <= 1e-8 / gaps.min() * scale
        assert np.abs(y[b] - ph / abs(ph) * y_ref[b]).max() <= 1e-8 / gaps.min() * scale


@pytest.mark.parametrize("name,nblocks,nline", [("box30", 1, 4), ("box30", 3, 3), ("box48", 2, 3), ("tric", 4, 2), ("tric", 1, 0)])
def test_lobpcg_gen_matches_oracle(gpu, name, nblocks, nline):
    import torch
    w = problem(name)
    ham, gargs = gen_setup(gpu, w, seed=11)
    psi = dev(w.psi)
    hpsi, spsi = torch.empty_like(psi), torch.empty_like(psi)
    out = gpu.lobpcg_gen(ham, psi, hpsi, spsi, nblocks, nline)
    ref = lo.lobpcg_gen(*gargs, w.psi, nblocks, nline)
    assert out["info"] > 0
    compare_gen(out, ref, psi.cpu().numpy(), hpsi.cpu().numpy(), spsi.cpu().numpy(), gargs)
    ham.destroy()


def test_chol_ortho_gen_matches_oracle(gpu):
    from oracle import paw
    w = problem("box30")
    ham, gargs = gen_setup(gpu, w, seed=12)
    h_ref, s_ref = paw.apply_hs(*gargs, w.psi)
    y_ref, hy_ref, sy_ref, u_ref = lo.chol_ortho_gen(w.psi, h_ref, s_ref)
    psi, hpsi, spsi = dev(w.psi), dev(h_ref), dev(s_ref)
    u, info = gpu.chol_ortho_gen(psi, hpsi, spsi)
    assert info == 0
    # the Cholesky factor with positive diagonal is unique: compare everything element by element
    assert np.abs(u.cpu().numpy() - u_ref).max() <= 1e-11 * np.abs(u_ref).max()
    for got, ref in ((psi, y_ref), (hpsi, hy_ref), (spsi, sy_ref)):
        assert np.linalg.norm(got.cpu().numpy() - ref) <= 1e-10 * np.linalg.norm(ref)
    y = psi.cpu().numpy()
    assert np.abs(y.conj() @ spsi.cpu().numpy().T - np.eye(y.shape[0])).max() <= 1e-12 * y.shape[0]
    ham.destroy()


def test_lobpcg_gen_converges_to_the_generalised_spectrum(gpu):
    import scipy.linalg as sl
    import torch
    from oracle import paw
    w = problem("tric")
    ham, gargs = gen_setup(gpu, w, seed=13)
    off, db, qb = gargs[6:]
    hd = oracle.dense_h(w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, None, None)
    p = w.proj
    hd = hd + p.T @ paw.blockdiag_dense(off, db) @ p.conj()
    sd = np.eye(w.npw) + p.T @ paw.blockdiag_dense(off, qb) @ p.conj()
    ev = sl.eigh(hd, sd, eigvals_only=True)[: w.psi.shape[0]]
    psi = dev(w.psi)
    hpsi, spsi = torch.empty_like(psi), torch.empty_like(psi)
    out = gpu.lobpcg_gen(ham, psi, hpsi, spsi, 1, 80, tol=1e-6)
    assert out["resid"].cpu().numpy().max() <= 2e-6
    assert np.abs(out["lam"].cpu().numpy() - ev).max() <= 1e-9 * np.abs(ev).max()
    with pytest.raises(gpu.PwhamError):
        gpu.lobpcg_gen(ham, psi, hpsi, spsi, 5, 1)
    ham.destroy()

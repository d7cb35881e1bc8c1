"""GPU parity of the electronic density accumulation (pwh_density_accumulate; Algorithm 3
steps 9-10) against oracle/density_oracle.py, element by element on the same seeded inputs, through the C ABI.  Tolerance:
relative Frobenius error 1e-11 (the inverse half of the H.Psi transforms followed by one FP64 multiply-add per band and
point).  Needs a B200 (`-m gpu`)."""
import numpy as np
import pytest

from oracle import density_oracle as dn
from paper_2604_11139_b200 import synth

pytestmark = pytest.mark.gpu

TOL_RHO = 1e-11


def relerr(x, ref):
    return float(np.linalg.norm(np.asarray(x) - np.asarray(ref)) / max(np.linalg.norm(ref), 1e-300))


@pytest.fixture(scope="module")
def gpu():
    import torch
    from paper_2604_11139_b200 import binding
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    binding.load_library()
    return binding


def setup(binding, w):
    return binding.ham_setup(w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, w.proj, w.dij)


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def zeros_rho(w):
    import torch
    n1, n2, n3 = (int(v) for v in w.fft_dims)
    return torch.zeros((n3, n2, n1), dtype=torch.float64, device="cuda")


def occupations(nband, seed):
    occ = np.random.default_rng(seed).uniform(0.0, 2.0, nband)
    occ[-1] = 0.0                                        # an empty band contributes nothing
    return occ


@pytest.mark.parametrize("cfg", ["cfg1", "cfg2"])
def test_density_matches_oracle(gpu, cfg, request):
    w = request.getfixturevalue(cfg)
    occ = occupations(w.nband, 1)
    ham = setup(gpu, w)
    rho = gpu.density_accumulate(ham, to_dev(w.psi), occ, zeros_rho(w), weight=0.37).cpu().numpy()
    ref = dn.density(w.fft_dims, w.gvec, w.psi, occ, 0.37)
    assert relerr(rho, ref) <= TOL_RHO
    assert rho.min() >= 0.0
    ham.destroy()


CASES = [
    ((20, 24, 30), (8.0, 9.0, 11.0), (0.25, -0.125, 0.375), 4.0, 5),      # two-pass transforms on every axis
    ((15, 16, 45), (6.0, 6.5, 14.0), (0.0, 0.25, 0.0), 4.0, 4),           # single-pass x and y
    ((125, 6, 4), (30.0, 4.0, 3.0), (0.25, 0.0, 0.0), 2.0, 3),            # 125 = 5^3: generic stage plan
    ((2, 2, 2), (2.0, 2.0, 2.0), (0.0, 0.0, 0.0), 0.1, 2),                # one plane wave
    ((128, 128, 4), (54.0, 54.0, 2.0), (0.0, 0.0, 0.0), 6.95, 3),         # cfg 4's plane
    ((120, 120, 6), (50.0, 50.0, 3.0), (0.25, 0.25, 0.25), 8.0, 3),       # cfg 5's plane
]


@pytest.mark.parametrize("case", range(len(CASES)))
def test_density_random_boxes(gpu, case):
    dims, cell, kpt, ecut, nband = CASES[case]
    w = synth.random_problem(dims, cell, kpt, ecut, 0, nband, seed=500 + case)
    occ = occupations(nband, case)
    ham = setup(gpu, w)
    rho = gpu.density_accumulate(ham, to_dev(w.psi), occ, zeros_rho(w)).cpu().numpy()
    assert relerr(rho, dn.density(w.fft_dims, w.gvec, w.psi, occ)) <= TOL_RHO, ham.kernels()
    ham.destroy()


@pytest.mark.parametrize("env", [("PWH_FORCE_GENERIC_FFT",), ("PWH_NO_ZW",), ("PWH_NO_ZW", "PWH_NO_V2")])
def test_density_other_kernel_families(gpu, cfg2, monkeypatch, env):
    for e in env:
        monkeypatch.setenv(e, "1")
    w = cfg2
    occ = occupations(12, 3)
    ham = setup(gpu, w)
    rho = gpu.density_accumulate(ham, to_dev(w.psi[:12]), occ, zeros_rho(w)).cpu().numpy()
    assert relerr(rho, dn.density(w.fft_dims, w.gvec, w.psi[:12], occ)) <= TOL_RHO, ham.kernels()
    ham.destroy()


def test_density_accumulates_over_calls_and_kpoints(gpu):
    """Algorithm 3 steps 9-10: one rho collects the bands of several calls and the k-points of several handles."""
    dims, cell = (24, 20, 18), (9.0, 8.0, 7.0)
    wa = synth.random_problem(dims, cell, (0.0, 0.0, 0.0), 4.0, 0, 6, seed=601)
    wb = synth.random_problem(dims, cell, (0.25, 0.25, -0.25), 4.0, 0, 4, seed=602)
    assert wa.npw != wb.npw
    occ_a, occ_b = occupations(6, 7), occupations(4, 8)
    ha, hb = setup(gpu, wa), setup(gpu, wb)
    rho = zeros_rho(wa)
    gpu.density_accumulate(ha, to_dev(wa.psi[:2]), occ_a[:2], rho, weight=0.75)
    gpu.density_accumulate(hb, to_dev(wb.psi), occ_b, rho, weight=0.25)
    gpu.density_accumulate(ha, to_dev(wa.psi[2:]), occ_a[2:], rho, weight=0.75)
    ref = dn.density_kpoints(dims, [(wa.gvec, wa.psi, occ_a, 0.75), (wb.gvec, wb.psi, occ_b, 0.25)])
    assert relerr(rho.cpu().numpy(), ref) <= TOL_RHO
    ha.destroy()
    hb.destroy()


def test_density_several_band_groups_padded_ld_and_determinism(gpu, monkeypatch):
    """cfg 3's box with more bands than one band group of the local kernels (ragged last group); padded leading dimension;
    two runs bit-identical."""
    import torch
    monkeypatch.setenv("PWH_BAND_GROUP", "7")
    w = synth.make_workload(3, nband=24, qr="none")
    occ = occupations(24, 9)
    ham = setup(gpu, w)
    assert ham.info()["band_group"] < 24
    pad = torch.zeros((24, w.npw + 5), dtype=torch.complex128, device="cuda")
    pad[:, w.npw:] = float("nan")
    pad[:, :w.npw] = to_dev(w.psi)
    r1 = gpu.density_accumulate(ham, pad[:, :w.npw], occ, zeros_rho(w)).cpu().numpy()
    r2 = gpu.density_accumulate(ham, pad[:, :w.npw], occ, zeros_rho(w)).cpu().numpy()
    assert np.array_equal(r1, r2)
    assert relerr(r1, dn.density(w.fft_dims, w.gvec, w.psi, occ)) <= TOL_RHO
    ham.destroy()


def test_density_full_size_cfg4_sampled_points_and_parseval(gpu):
    """cfg 4 at full box size, 16 bands: sampled grid points against the defining sum evaluated one by one, and
    sum_r rho(r) = F sum_i f_i |psi_i|^2 (Parseval), which holds at any size."""
    w = synth.make_workload(4, nband=16, qr="none")
    occ = occupations(16, 10)
    ham = setup(gpu, w)
    rho = gpu.density_accumulate(ham, to_dev(w.psi), occ, zeros_rho(w)).cpu().numpy()
    n1, n2, n3 = (int(v) for v in w.fft_dims)
    f = n1 * n2 * n3
    want = f * float((occ * (np.abs(w.psi) ** 2).sum(axis=1)).sum())
    assert abs(rho.sum() - want) <= 1e-11 * want
    rng = np.random.default_rng(11)
    g = w.gvec.astype(np.float64)
    for _ in range(24):
        r = (int(rng.integers(n1)), int(rng.integers(n2)), int(rng.integers(n3)))
        phase = np.exp(2j * np.pi * (g[:, 0] * r[0] / n1 + g[:, 1] * r[1] / n2 + g[:, 2] * r[2] / n3))
        u = w.psi @ phase
        ref = float((occ * np.abs(u) ** 2).sum())
        assert abs(rho[r[2], r[1], r[0]] - ref) <= 1e-10 * max(ref, rho.max() * 1e-3)
    ham.destroy()


def test_density_error_codes(gpu, cfg1):
    import torch
    ham = setup(gpu, cfg1)
    psi = to_dev(cfg1.psi)
    with pytest.raises(gpu.PwhamError):
        gpu.density_accumulate(ham, psi, np.ones(3), zeros_rho(cfg1))
    with pytest.raises(gpu.PwhamError):
        gpu.density_accumulate(ham, psi, np.ones(cfg1.nband), torch.zeros((4, 4, 4), dtype=torch.float64, device="cuda"))
    L = gpu.load_library()
    assert L.pwh_density_accumulate(ham.handle, 1, psi.data_ptr(), cfg1.npw, None, 1.0, None, None, 0, None) == -1
    ham.destroy()

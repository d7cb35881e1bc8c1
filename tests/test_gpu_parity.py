"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json's: relative Frobenius error 1e-11 for H.Psi and Gram
matrices, 1e-9 for filtered blocks (complex128).  Every test here needs a B200 (`-m gpu`).
"""
import math

import numpy as np
import pytest

import oracle
from paper_2604_11139_b200 import synth

pytestmark = pytest.mark.gpu

TOL_H = 1e-11
TOL_F = 1e-9


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


def setup(binding, w, proj="default", vloc=None):
    p = w.proj if isinstance(proj, str) else proj
    d = w.dij if isinstance(proj, str) else (w.dij[: 0 if proj is None else len(proj)])
    return binding.ham_setup(w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc if vloc is None else vloc, p, d)


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# ----------------------------------------------------------------------------------------------------------------
# apply_h
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg", ["cfg1", "cfg2"])
def test_apply_h_matches_oracle(gpu, cfg, request):
    w = request.getfixturevalue(cfg)
    ham = setup(gpu, w)
    out = gpu.apply_h(ham, to_dev(w.psi)).cpu().numpy()
    ref = oracle.apply_h(*ham_args(w), w.psi)
    assert relerr(out, ref) <= TOL_H
    # element by element, scaled by the block's largest entry
    assert np.abs(out - ref).max() <= 1e-11 * np.abs(ref).max()
    ham.destroy()


@pytest.mark.parametrize("term", ["kin", "loc", "nl"])
def test_apply_h_single_terms_cfg2(gpu, cfg2, term):
    """Each additive term alone (kinetic, local, nonlocal), so that a large term cannot mask a small one."""
    w = cfg2
    psi = w.psi[:24]
    if term == "kin":
        ham = setup(gpu, w, proj=None, vloc=np.zeros_like(w.vloc))
        ref = oracle.apply_h(*ham_args(w), psi, terms=oracle.TERM_KIN)
    elif term == "loc":
        ham = setup(gpu, w, proj=None)
        ref = oracle.apply_h(*ham_args(w), psi, terms=oracle.TERM_KIN | oracle.TERM_LOC)
    else:
        ham = setup(gpu, w, vloc=np.zeros_like(w.vloc))
        ref = oracle.apply_h(*ham_args(w), psi, terms=oracle.TERM_KIN | oracle.TERM_NL)
    out = gpu.apply_h(ham, to_dev(psi)).cpu().numpy()
    if term == "loc":   # subtract the (exactly diagonal) kinetic part so the local term is compared on its own scale
        kin = oracle.kinetic(w.lattice, w.kpt, w.gvec)
        assert relerr(out - kin[None, :] * psi, ref - kin[None, :] * psi) <= 10 * TOL_H
    assert relerr(out, ref) <= TOL_H
    ham.destroy()


RANDOM_CASES = [
    # dims,           cell,             kpt,                     ecut, nproj, nband   (radices exercised)
    ((20, 24, 30), (8.0, 9.0, 11.0), (0.25, -0.125, 0.375), 4.0, 7, 5),     # 4*5, 8*3, 5*3*2
    ((10, 12, 18), (5.0, 6.0, 9.0), (0.0, 0.0, 0.0), 2.5, 3, 3),            # 5*2, 4*3, 3*3*2
    ((25, 27, 32), (9.0, 9.5, 11.0), (0.5, 0.5, 0.5), 4.0, 130, 67),        # 5*5, 3*3*3, 8*4; ragged GEMM tiles
    ((6, 6, 6), (4.0, 4.0, 4.0), (0.1, 0.2, 0.3), 1.5, 1, 1),               # 5 plane waves, one band, one projector
    ((64, 40, 36), (14.0, 9.0, 8.0), (0.25, 0.25, 0.25), 6.0, 0, 9),        # no projectors
    ((2, 2, 2), (2.0, 2.0, 2.0), (0.0, 0.0, 0.0), 0.1, 2, 2),               # one plane wave, smallest box
    ((125, 6, 4), (30.0, 4.0, 3.0), (0.25, 0.0, 0.0), 2.0, 4, 3),           # 125 = 5^3: generic-stage fallback plan
    ((15, 16, 45), (6.0, 6.5, 14.0), (0.0, 0.25, 0.0), 4.0, 6, 4),          # single-pass 15 and 16, 45 = 9*5
    ((180, 120, 8), (75.0, 50.0, 4.0), (0.25, 0.25, 0.25), 3.0, 5, 3),      # cfg 5's axis lengths 15*12 and 12*10
    # the large planes of the size-specialised plane kernel: cfg 4's with its 65 x-lines, cfg 5's and cfg 3's with a k-point,
    # a small sphere in a large box, and a sphere wider than half the box (too large for it: generic-size kernel)
    ((128, 128, 12), (54.0, 54.0, 5.0), (0.0, 0.0, 0.0), 6.95, 6, 5),
    ((120, 120, 6), (50.0, 50.0, 3.0), (0.25, 0.25, 0.25), 8.0, 4, 3),
    ((96, 96, 8), (40.0, 40.0, 4.0), (0.25, 0.25, 0.25), 7.1, 4, 3),
    ((128, 128, 4), (54.0, 54.0, 2.0), (0.25, -0.25, 0.0), 0.8, 3, 4),
    ((128, 128, 4), (54.0, 54.0, 2.0), (0.0, 0.0, 0.0), 11.0, 3, 3),
]


@pytest.mark.parametrize("case", range(len(RANDOM_CASES)))
def test_random_boxes_apply_filter_gram(gpu, case):
    dims, cell, kpt, ecut, nproj, nband = RANDOM_CASES[case]
    w = synth.random_problem(dims, cell, kpt, ecut, nproj, nband, seed=case)
    ham = setup(gpu, w)
    psi = to_dev(w.psi)
    hpsi = gpu.apply_h(ham, psi)
    ref_h = oracle.apply_h(*ham_args(w), w.psi)
    assert relerr(hpsi.cpu().numpy(), ref_h) <= TOL_H
    g = gpu.gram(psi, hpsi).cpu().numpy()
    assert relerr(g, oracle.gram(w.psi, ref_h)) <= TOL_H
    for m in (1, 2, 3, 5):
        y = gpu.cheb_filter(ham, psi.clone(), m, w.a, w.b, w.a0).cpu().numpy()
        ref = oracle.cheb_filter(*ham_args(w), w.psi, m, w.a, w.b, w.a0)
        assert relerr(y, ref) <= TOL_F, (case, m)
    ham.destroy()


def test_generic_fft_fallback_cfg2(gpu, cfg2, monkeypatch):
    """The radix-2/3/4/5/8 shared-memory stage plan (used when an axis does not factor as r1*r2) on config 2."""
    monkeypatch.setenv("PWH_FORCE_GENERIC_FFT", "1")
    w = cfg2
    ham = setup(gpu, w)
    monkeypatch.delenv("PWH_FORCE_GENERIC_FFT")
    psi = w.psi[:40]
    out = gpu.apply_h(ham, to_dev(psi)).cpu().numpy()
    assert relerr(out, oracle.apply_h(*ham_args(w), psi)) <= TOL_H
    y = gpu.cheb_filter(ham, to_dev(psi), 3, w.a, w.b, w.a0).cpu().numpy()
    assert relerr(y, oracle.cheb_filter(*ham_args(w), psi, 3, w.a, w.b, w.a0)) <= TOL_F
    ham.destroy()


@pytest.mark.parametrize("env", [("PWH_NO_ZW",), ("PWH_NO_V2",), ("PWH_NO_ZW", "PWH_NO_V2")])
def test_fallback_kernels_cfg2(gpu, cfg2, monkeypatch, env):
    """The CTA-per-column-group z kernels and the generic-size plane kernel (local_fast.cu), which serve boxes the
    size-specialised kernels are not instantiated for, on config 2."""
    for e in env:
        monkeypatch.setenv(e, "1")
    w = cfg2
    ham = setup(gpu, w)
    for e in env:
        monkeypatch.delenv(e)
    psi = w.psi[:40]
    out = gpu.apply_h(ham, to_dev(psi)).cpu().numpy()
    assert relerr(out, oracle.apply_h(*ham_args(w), psi)) <= TOL_H
    y = gpu.cheb_filter(ham, to_dev(psi), 3, w.a, w.b, w.a0).cpu().numpy()
    assert relerr(y, oracle.cheb_filter(*ham_args(w), psi, 3, w.a, w.b, w.a0)) <= TOL_F
    ham.destroy()


@pytest.mark.parametrize("env", ["PWH_V2_NO_PRUNE", "PWH_LOCAL_ONE_STREAM", "PWH_LOCAL_TWO_STREAMS"])
@pytest.mark.parametrize("case", ["cfg2", "plane128", "plane120"])
def test_unpruned_passes_and_single_stream(gpu, cfg2, monkeypatch, env, case):
    """The full-length strided-role passes (taken by themselves only for spheres wider than half an axis) and the in-order
    local stage, on boxes whose default is the pruned / two-stream path; more bands than one band group."""
    monkeypatch.setenv(env, "1")
    if case == "cfg2":
        w = cfg2
    elif case == "plane128":
        w = synth.random_problem((128, 128, 12), (54.0, 54.0, 5.0), (0.0, 0.0, 0.0), 6.95, 6, 40, seed=77)
    else:
        w = synth.random_problem((120, 120, 6), (50.0, 50.0, 3.0), (0.25, 0.25, 0.25), 8.0, 4, 70, seed=78)
    ham = setup(gpu, w)
    psi = to_dev(w.psi)
    assert relerr(gpu.apply_h(ham, psi).cpu().numpy(), oracle.apply_h(*ham_args(w), w.psi)) <= TOL_H
    y = gpu.cheb_filter(ham, psi.clone(), 3, w.a, w.b, w.a0).cpu().numpy()
    assert relerr(y, oracle.cheb_filter(*ham_args(w), w.psi, 3, w.a, w.b, w.a0)) <= TOL_F
    ham.destroy()


@pytest.mark.parametrize("group", [1, 5, 64])
def test_band_groups_alternate_between_two_streams(gpu, cfg2, monkeypatch, group):
    """Many small band groups (ragged last one for 5) on the two internal streams, and exactly two groups (64): every band goes
    through the same kernels whatever the grouping, so the result must not depend on it at all."""
    monkeypatch.setenv("PWH_BAND_GROUP", str(group))
    monkeypatch.setenv("PWH_LOCAL_TWO_STREAMS", "1")
    w = cfg2
    ham = setup(gpu, w)
    assert ham.info()["band_group"] == group
    psi = to_dev(w.psi)
    h1 = gpu.apply_h(ham, psi).cpu().numpy()
    assert relerr(h1, oracle.apply_h(*ham_args(w), w.psi)) <= TOL_H
    y = gpu.cheb_filter(ham, psi.clone(), 4, w.a, w.b, w.a0).cpu().numpy()
    assert relerr(y, oracle.cheb_filter(*ham_args(w), w.psi, 4, w.a, w.b, w.a0)) <= TOL_F
    ham.destroy()
    monkeypatch.delenv("PWH_BAND_GROUP")
    monkeypatch.delenv("PWH_LOCAL_TWO_STREAMS")
    ham = setup(gpu, w)
    assert np.array_equal(gpu.apply_h(ham, psi).cpu().numpy(), h1)       # bit-identical to the default grouping
    ham.destroy()


def test_stream_choice_is_measured_without_changing_results(gpu, cfg2, monkeypatch):
    """Default handle: the first four multi-group H applications alternate between two streams and one and are timed with
    events, later ones use the faster -- ten applications in a row must all be bit-identical."""
    monkeypatch.setenv("PWH_BAND_GROUP", "16")
    ham = setup(gpu, cfg2)
    psi = to_dev(cfg2.psi)
    ref = gpu.apply_h(ham, psi).cpu().numpy()
    assert relerr(ref, oracle.apply_h(*ham_args(cfg2), cfg2.psi)) <= TOL_H
    import torch
    for i in range(10):
        if i == 6:
            torch.cuda.synchronize()
        assert np.array_equal(gpu.apply_h(ham, psi).cpu().numpy(), ref), i
    y = gpu.cheb_filter(ham, psi.clone(), 8, cfg2.a, cfg2.b, cfg2.a0).cpu().numpy()
    assert relerr(y, oracle.cheb_filter(*ham_args(cfg2), cfg2.psi, 8, cfg2.a, cfg2.b, cfg2.a0)) <= TOL_F
    ham.destroy()


def test_zgemm_without_tma(gpu, cfg2, monkeypatch):
    """The cp.async (LDGSTS) 3M ZGEMM kernels that serve when cuTensorMapEncodeTiled is unavailable or refuses an operand,
    against the oracle: projector path of apply_h and a ragged Gram product."""
    monkeypatch.setenv("PWH_ZGEMM_NO_TMA", "1")
    w = cfg2
    ham = setup(gpu, w)
    psi = w.psi[:67]
    out = gpu.apply_h(ham, to_dev(psi)).cpu().numpy()
    ref = oracle.apply_h(*ham_args(w), psi)
    assert relerr(out, ref) <= TOL_H
    g = gpu.gram(to_dev(psi), to_dev(ref)).cpu().numpy()
    assert relerr(g, oracle.gram(psi, ref)) <= TOL_H
    ham.destroy()


def test_cfg3_band_subset(gpu):
    """Config 3 (k = 1/4 1/4 1/4, 96^3, 57925 plane waves, 512 projectors) at full N and J on a subset of bands --
    exact, since bands never interact before gram."""
    w = synth.make_workload(3, nband=12, qr="numpy")
    ham = setup(gpu, w)
    info = ham.info()
    assert info["npw"] == synth.EXPECTED_NPW[3] and info["n_zcolumns"] == 1808 and info["n_xlines"] == 48
    psi = to_dev(w.psi)
    hpsi = gpu.apply_h(ham, psi)
    ref_h = oracle.apply_h(*ham_args(w), w.psi)
    assert relerr(hpsi.cpu().numpy(), ref_h) <= TOL_H
    y = gpu.cheb_filter(ham, psi.clone(), 4, w.a, w.b, w.a0).cpu().numpy()
    assert relerr(y, oracle.cheb_filter(*ham_args(w), w.psi, 4, w.a, w.b, w.a0)) <= TOL_F
    g = gpu.gram(psi, hpsi).cpu().numpy()
    assert relerr(g, oracle.gram(w.psi, ref_h)) <= TOL_H
    ham.destroy()


# ----------------------------------------------------------------------------------------------------------------
# cheb_filter
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,degrees", [("cfg1", (0, 1, 2, 3, 4, 7, 16)), ("cfg2", (1, 8))])
def test_cheb_filter_matches_oracle(gpu, cfg, degrees, request):
    w = request.getfixturevalue(cfg)
    ham = setup(gpu, w)
    for m in degrees:
        y = gpu.cheb_filter(ham, to_dev(w.psi), m, w.a, w.b, w.a0).cpu().numpy()
        ref = oracle.cheb_filter(*ham_args(w), w.psi, m, w.a, w.b, w.a0)
        assert relerr(y, ref) <= TOL_F, m
    ham.destroy()


def test_cheb_filter_paper_bounds_rule(gpu, cfg1):
    """Bounds from Rayleigh quotients as in Algorithm 12 line 3: a0 = min RQ, a = max RQ."""
    w = cfg1
    hp = oracle.apply_h(*ham_args(w), w.psi)
    rq = np.real(np.einsum("bg,bg->b", w.psi.conj(), hp))
    a0, a = float(rq.min()) - 1e-3, float(rq.max())
    ham = setup(gpu, w)
    y = gpu.cheb_filter(ham, to_dev(w.psi), 6, a, w.b, a0).cpu().numpy()
    assert relerr(y, oracle.cheb_filter(*ham_args(w), w.psi, 6, a, w.b, a0)) <= TOL_F
    ham.destroy()


def test_filter_is_m_applications_of_h(gpu, cfg1):
    """Degree-1 filter == (sigma_1/e)(H - c) psi computed from apply_h (the recurrence's first step)."""
    w = cfg1
    ham = setup(gpu, w)
    psi = to_dev(w.psi)
    e, c = 0.5 * (w.b - w.a), 0.5 * (w.b + w.a)
    s1 = e / (w.a0 - c)
    y1 = gpu.cheb_filter(ham, psi.clone(), 1, w.a, w.b, w.a0)
    manual = (s1 / e) * (gpu.apply_h(ham, psi) - c * psi)
    assert relerr(y1.cpu().numpy(), manual.cpu().numpy()) <= 1e-13
    ham.destroy()


# ----------------------------------------------------------------------------------------------------------------
# gram
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nx,ny,npw", [(1, 1, 1), (3, 5, 17), (16, 16, 257), (128, 128, 7153), (130, 67, 4099),
                                       (64, 200, 33)])
def test_gram_matches_oracle(gpu, nx, ny, npw):
    rng = np.random.default_rng(nx * 1000 + ny)
    x = (rng.standard_normal((nx, npw)) + 1j * rng.standard_normal((nx, npw)))
    y = (rng.standard_normal((ny, npw)) + 1j * rng.standard_normal((ny, npw)))
    g = gpu.gram(to_dev(x), to_dev(y)).cpu().numpy()
    ref = oracle.gram(x, y)
    assert g.shape == (nx, ny)
    assert relerr(g, ref) <= TOL_H
    assert np.abs(g - ref).max() <= 1e-11 * np.abs(ref).max() * math.sqrt(npw)


def test_gram_of_orthonormal_block_and_hermiticity(gpu, cfg2):
    w = cfg2
    ham = setup(gpu, w)
    psi = to_dev(w.psi)
    s = gpu.gram(psi, psi).cpu().numpy()
    assert np.abs(s - np.eye(w.nband)).max() <= 1e-13
    hpsi = gpu.apply_h(ham, psi)
    hsub = gpu.gram(psi, hpsi).cpu().numpy()
    assert np.abs(hsub - hsub.conj().T).max() <= 1e-12 * np.abs(hsub).max()
    assert relerr(hsub, oracle.gram(w.psi, oracle.apply_h(*ham_args(w), w.psi))) <= TOL_H
    # deterministic: the split-K reduction has a fixed order
    assert np.array_equal(hsub, gpu.gram(psi, hpsi).cpu().numpy())
    ham.destroy()


# ----------------------------------------------------------------------------------------------------------------
# layout, ownership, errors, host entry points
# ----------------------------------------------------------------------------------------------------------------
def test_padded_leading_dimension_is_untouched(gpu, cfg1):
    import torch
    w = cfg1
    ham = setup(gpu, w)
    ld = w.npw + 7
    buf = torch.full((w.nband, ld), complex(7.0, -3.0), dtype=torch.complex128, device="cuda")
    buf[:, : w.npw] = to_dev(w.psi)
    out = torch.full((w.nband, ld + 2), complex(1.0, 2.0), dtype=torch.complex128, device="cuda")
    gpu.apply_h(ham, buf[:, : w.npw], out[:, : w.npw])
    ref = oracle.apply_h(*ham_args(w), w.psi)
    assert relerr(out[:, : w.npw].cpu().numpy(), ref) <= TOL_H
    assert torch.all(out[:, w.npw:] == complex(1.0, 2.0))
    gpu.cheb_filter(ham, buf[:, : w.npw], 5, w.a, w.b, w.a0)
    assert relerr(buf[:, : w.npw].cpu().numpy(), oracle.cheb_filter(*ham_args(w), w.psi, 5, w.a, w.b, w.a0)) <= TOL_F
    assert torch.all(buf[:, w.npw:] == complex(7.0, -3.0))
    ham.destroy()


def test_band_independence_and_blocking(gpu, cfg2):
    """Filtering a block == filtering its column blocks separately (cfg 5's 'blocks of 512'), bit for bit."""
    w = cfg2
    ham = setup(gpu, w)
    full = gpu.cheb_filter(ham, to_dev(w.psi), 3, w.a, w.b, w.a0)
    parts = to_dev(w.psi)
    for b0 in range(0, w.nband, 48):
        gpu.cheb_filter(ham, parts[b0:b0 + 48], 3, w.a, w.b, w.a0)
    assert relerr(parts.cpu().numpy(), full.cpu().numpy()) <= 1e-14
    ham.destroy()


def test_error_codes(gpu, cfg1):
    import torch
    w = cfg1
    with pytest.raises(gpu.PwhamError, match="prime factors"):
        gpu.ham_setup(w.lattice, w.kpt, (14, 16, 16), w.gvec, np.zeros((16, 16, 14)), w.proj, w.dij)
    bad = w.gvec.copy()
    bad[1] = bad[0] + np.array([16, 0, 0])      # wraps onto plane wave 0
    with pytest.raises(gpu.PwhamError, match="collides"):
        gpu.ham_setup(w.lattice, w.kpt, w.fft_dims, bad, w.vloc, w.proj, w.dij)
    ham = setup(gpu, w)
    psi = to_dev(w.psi)
    with pytest.raises(gpu.PwhamError, match="b > a"):
        gpu.cheb_filter(ham, psi, 3, 2.0, 1.0, 0.0)
    with pytest.raises(gpu.PwhamError, match="a0 < a"):
        gpu.cheb_filter(ham, psi, 3, 1.0, 2.0, 1.5)
    with pytest.raises(gpu.PwhamError, match="degree"):
        gpu.cheb_filter(ham, psi, -1, 1.0, 2.0, 0.0)
    L = gpu.load_library()
    ws = torch.empty(1024, dtype=torch.uint8, device="cuda")
    rc = L.pwh_apply_h(ham.handle, w.nband, psi.data_ptr(), w.npw, psi.data_ptr(), w.npw, ws.data_ptr(), 16, None)
    assert rc == -1 and b"workspace" in L.pwh_last_error()
    rc = L.pwh_apply_h(ham.handle, w.nband, psi.data_ptr(), w.npw - 1, psi.data_ptr(), w.npw, ws.data_ptr(), 16, None)
    assert rc == -1
    assert L.pwh_apply_h(ham.handle, 0, None, 0, None, 0, None, 0, None) == 0      # nband == 0: no-op
    ham.destroy()


def test_host_entry_points(gpu, cfg2):
    """The end-to-end calls bench.py times: host buffers in, host buffers out, same kernels."""
    import torch
    w = cfg2
    ham = setup(gpu, w)
    psi_h = torch.from_numpy(w.psi.copy()).pin_memory()
    hpsi_h = torch.empty_like(psi_h).pin_memory()
    gpu.apply_h_host(ham, psi_h, hpsi_h)
    ref_h = oracle.apply_h(*ham_args(w), w.psi)
    assert relerr(hpsi_h.numpy(), ref_h) <= TOL_H
    y_h = torch.from_numpy(w.psi.copy()).pin_memory()
    gpu.cheb_filter_host(ham, y_h, 4, w.a, w.b, w.a0, block=40)
    ref_y = oracle.cheb_filter(*ham_args(w), w.psi, 4, w.a, w.b, w.a0)
    assert relerr(y_h.numpy(), ref_y) <= TOL_F
    z_h = torch.from_numpy(w.psi.copy()).pin_memory()
    g_h = torch.empty((w.nband, w.nband), dtype=torch.complex128).pin_memory()
    hz_h = torch.empty_like(z_h).pin_memory()
    n0 = gpu.launch_count()
    gpu.sweep_host(ham, z_h, 4, w.a, w.b, w.a0, g_h, block=64, hpsi_host=hz_h)
    assert gpu.launch_count() > n0
    assert relerr(z_h.numpy(), ref_y) <= TOL_F
    ref_hy = oracle.apply_h(*ham_args(w), ref_y)
    assert relerr(hz_h.numpy(), ref_hy) <= TOL_F
    assert relerr(g_h.numpy().T, oracle.gram(ref_y, ref_hy)) <= TOL_F
    ham.destroy()


# ----------------------------------------------------------------------------------------------------------------
# BASELINE.json's full sizes, in the launch configuration bench.py times
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_size_sampled_bands(gpu, cfg):
    """Configs 3-5 with ALL their bands, driven exactly as bench.py's step drives them (filter of the config's degree in
    column blocks of `block`, H.Psi in the same blocks, Hermitian Gram of the whole block), checked on sampled outputs the
    oracle can compute one by one: bands never interact before gram, so the oracle filters the
    16 sampled bands alone; a Gram entry is one dot product of two such bands.  The samples cover the
    first and last band, both sides of every column-block boundary and random bands in between, i.e. different band
    groups of the local kernels, different column blocks and both ends of the ZGEMM tiles."""
    import torch
    w = synth.make_workload(cfg, qr="torch-cuda")
    spec = w.spec
    M = spec.nband
    assert w.npw == synth.EXPECTED_NPW[cfg] and w.psi.shape[0] == M
    rng = np.random.default_rng(7000 + cfg)
    fixed = {0, M - 1, 127, 128, spec.block - 1, spec.block % M, M // 2}
    extra = [int(i) for i in rng.permutation(M) if int(i) not in fixed]
    idx = sorted(fixed) + extra[:16 - len(fixed)]
    assert len(idx) == 16
    rows = np.sort(rng.choice(M, size=64, replace=False))
    cols = np.sort(rng.choice(M, size=64, replace=False))
    ham = setup(gpu, w)
    psi = to_dev(w.psi)
    hpsi = torch.empty_like(psi)
    for b0 in range(0, M, spec.block):
        gpu.cheb_filter(ham, psi[b0:b0 + spec.block], spec.degree, w.a, w.b, w.a0)
    for b0 in range(0, M, spec.block):
        gpu.apply_h(ham, psi[b0:b0 + spec.block], hpsi[b0:b0 + spec.block])
    g = gpu.gram(psi, hpsi, hermitian=True)
    g_full = gpu.gram(psi[:256], hpsi[:192])               # general (non-Hermitian) product on a ragged sub-block
    torch.cuda.synchronize()
    y_gpu = psi[idx].cpu().numpy()
    hy_gpu = hpsi[idx].cpu().numpy()
    g_gpu = g[idx][:, idx].cpu().numpy()
    g_scale = float(g.abs().max())
    herm_defect = float((g - g.conj().T).abs().max())
    g_blk = g[rows][:, cols].cpu().numpy()
    y_rows = psi[rows].cpu().numpy()
    hy_cols = hpsi[cols].cpu().numpy()
    g_sub = g_full.cpu().numpy()
    g_sub_ref_in = (psi[:256:17].cpu().numpy(), hpsi[:192:13].cpu().numpy())
    ham.destroy()
    del psi, hpsi, g, g_full

    # the whole Gram matrix is Hermitian (H is), including across the mirrored blocks
    assert herm_defect <= 1e-12 * g_scale
    # a 64 x 64 block of random rows and columns: every entry against the oracle's dot product of the GPU's own bands
    assert relerr(g_blk, oracle.gram(y_rows, hy_cols)) <= TOL_H
    assert relerr(g_sub[::17][:, ::13], oracle.gram(*g_sub_ref_in)) <= TOL_H

    y_ref = oracle.cheb_filter(*ham_args(w), w.psi[idx], spec.degree, w.a, w.b, w.a0)
    hy_ref = oracle.apply_h(*ham_args(w), y_ref)
    g_ref = oracle.gram(y_ref, hy_ref)
    for k in range(len(idx)):                     # band by band, each against its own norm
        assert relerr(y_gpu[k], y_ref[k]) <= TOL_F
        assert relerr(hy_gpu[k], hy_ref[k]) <= TOL_F      # H applied to the filtered band inherits the filter's error
    # H alone at TOL_H: the GPU's H applied to the GPU's filtered bands against the oracle's H applied to the same input
    assert relerr(hy_gpu, oracle.apply_h(*ham_args(w), y_gpu)) <= TOL_H
    assert relerr(g_gpu, oracle.gram(y_gpu, hy_gpu)) <= TOL_H
    assert np.abs(g_gpu - g_ref).max() <= TOL_F * g_scale


# ----------------------------------------------------------------------------------------------------------------
# the rest of the ABI's input space: general lattices, arbitrary G order, non-convex G sets, padded projectors
# ----------------------------------------------------------------------------------------------------------------
def check_all(gpu, w, gvec=None, psi=None, proj=None, degrees=(1, 2, 5)):
    """apply_h, gram and cheb_filter of workload `w` against the oracle at the north_star tolerances."""
    ham = setup(gpu, w)
    x = to_dev(w.psi)
    hx = gpu.apply_h(ham, x)
    ref_h = oracle.apply_h(*ham_args(w), w.psi)
    assert relerr(hx.cpu().numpy(), ref_h) <= TOL_H
    assert relerr(gpu.gram(x, hx).cpu().numpy(), oracle.gram(w.psi, ref_h)) <= TOL_H
    for m in degrees:
        y = gpu.cheb_filter(ham, x.clone(), m, w.a, w.b, w.a0).cpu().numpy()
        assert relerr(y, oracle.cheb_filter(*ham_args(w), w.psi, m, w.a, w.b, w.a0)) <= TOL_F, m
    return ham


HEX = [[6.0, 0.0, 0.0], [-3.0, 3.0 * math.sqrt(3.0), 0.0], [0.0, 0.0, 9.0]]           # hexagonal, 120 degrees
TRICLINIC = [[7.0, 0.3, -0.5], [1.1, 6.5, 0.4], [-0.8, 1.2, 8.0]]
FCC = [[0.0, 4.0, 4.0], [4.0, 0.0, 4.0], [4.0, 4.0, 0.0]]                             # primitive fcc: B is bcc-like


@pytest.mark.parametrize("name,seed,lattice,dims,kpt,ecut", [
    ("hexagonal", 101, HEX, (24, 24, 30), (1.0 / 3.0, 1.0 / 3.0, 0.25), 14.0),
    ("triclinic", 102, TRICLINIC, (20, 24, 30), (0.1, -0.2, 0.3), 9.0),
    ("fcc", 103, FCC, (24, 24, 24), (0.5, 0.0, 0.5), 10.0),
    ("triclinic48", 104, TRICLINIC, (48, 48, 40), (0.0, 0.0, 0.0), 20.0),     # the size-specialised plane kernel, skewed disc
])
def test_general_lattice(gpu, name, seed, lattice, dims, kpt, ecut):
    """Non-orthogonal lattices (the kinetic term 1/2|k+G|^2 needs the full reciprocal metric): every
    off-diagonal cofactor of the library's reciprocal-lattice construction is exercised, and the sphere is an oblique
    ellipsoid in index space (skewed discs, x-line ranges that differ per row)."""
    w = synth.random_problem(dims, np.asarray(lattice), kpt, ecut, 6, 5, seed=seed)
    assert np.abs(w.lattice - np.diag(np.diag(w.lattice))).max() > 0.1
    kin_gpu_check = oracle.kinetic(w.lattice, w.kpt, w.gvec)
    assert kin_gpu_check.max() <= ecut * (1 + 1e-12)
    ham = check_all(gpu, w)
    # kinetic term alone, element-wise: H with V_loc = 0 and no projectors applied to unit-modulus vectors
    ham0 = gpu.ham_setup(w.lattice, w.kpt, w.fft_dims, w.gvec, np.zeros_like(w.vloc), None, None)
    ones = np.ones((1, w.npw), dtype=np.complex128)
    kin_gpu = gpu.apply_h(ham0, to_dev(ones)).cpu().numpy()[0]
    assert np.abs(kin_gpu.imag).max() == 0.0
    assert np.abs(kin_gpu.real - kin_gpu_check).max() <= 1e-13 * kin_gpu_check.max()
    ham0.destroy()
    ham.destroy()


@pytest.mark.parametrize("which", ["cfg2", "box"])
def test_shuffled_gvec_order(gpu, cfg2, which):
    """include/pwham.h accepts the plane waves in ANY order: a random permutation of gvec (and of the rows of Psi and P
    with it) must give the permuted result."""
    if which == "cfg2":
        w0 = cfg2
        nb = 24
    else:
        w0 = synth.random_problem((30, 20, 24), (11.0, 8.0, 9.0), (0.25, 0.125, -0.375), 5.0, 9, 6, seed=77)
        nb = 6
    perm = np.random.default_rng(123).permutation(w0.npw)
    import dataclasses
    w = dataclasses.replace(w0, gvec=np.ascontiguousarray(w0.gvec[perm]), proj=np.ascontiguousarray(w0.proj[:, perm]),
                            psi=np.ascontiguousarray(w0.psi[:nb][:, perm]))
    ham = check_all(gpu, w, degrees=(3,))
    # and against the unpermuted problem: same numbers, permuted
    ref = oracle.apply_h(*ham_args(w0), w0.psi[:nb])
    out = gpu.apply_h(ham, to_dev(w.psi)).cpu().numpy()
    assert relerr(out, ref[:, perm]) <= TOL_H
    ham.destroy()


@pytest.mark.parametrize("hole", ["x_slab", "centre", "random_columns", "random_half"])
def test_nonconvex_gset(gpu, hole):
    """A collision-free G set that is not a convex sphere (include/pwham.h promises any such set): a sphere with a slab of
    x removed (touched x-lines not contiguous), with its centre removed (disc rows with gaps), with a random half of its
    z-columns removed, and a random half of its points (which still touches every column of the disc, so the specialised
    kernel remains valid).  The first three violate the preconditions of the size-specialised plane kernels, which
    pwh_ham_setup must detect by itself (no environment switch) and fall back to the generic-size plane kernel."""
    base = synth.random_problem((48, 48, 36), (20.0, 20.0, 15.0), (0.0, 0.0, 0.0), 7.0, 5, 4, seed=90)
    g = base.gvec
    if hole == "x_slab":
        keep = np.abs(g[:, 0]) >= 3
    elif hole == "centre":
        keep = (np.abs(g[:, 0]) >= 2) | (np.abs(g[:, 1]) >= 2)
    elif hole == "random_columns":
        col_keep = np.random.default_rng(6).random((64, 64)) < 0.5
        keep = col_keep[g[:, 0] + 32, g[:, 1] + 32]
    else:
        keep = np.random.default_rng(5).random(g.shape[0]) < 0.5
    w = synth.random_problem((48, 48, 36), (20.0, 20.0, 15.0), (0.0, 0.0, 0.0), 7.0, 5, 4, seed=91,
                             gvec=g[keep])
    assert 0 < w.npw < base.npw
    ham = check_all(gpu, w, degrees=(2,))
    if hole != "random_half":
        assert "kf_plane" in ham.kernels() and "kv2_plane" not in ham.kernels()
    ham.destroy()
    # the convex sphere on the same box does take the specialised kernel
    ham_b = setup(gpu, base)
    assert "kv2_plane" in ham_b.kernels()
    ham_b.destroy()


def test_padded_projector_leading_dimension(gpu, cfg2):
    """ldp > npw (include/pwham.h: 'ldp >= npw'): the projector matrix is borrowed with padded columns; it changes the
    tensor-map stride of operand A in both ZGEMMs.  The padding holds NaNs, which must never be read."""
    import torch
    w = cfg2
    ldp = w.npw + 5
    pbuf = torch.full((w.nproj, ldp), complex(float("nan"), float("nan")), dtype=torch.complex128, device="cuda")
    pbuf[:, : w.npw] = to_dev(w.proj)
    ham = gpu.ham_setup(w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, pbuf[:, : w.npw], w.dij)
    psi = w.psi[:70]
    out = gpu.apply_h(ham, to_dev(psi)).cpu().numpy()
    assert relerr(out, oracle.apply_h(*ham_args(w), psi)) <= TOL_H
    y = gpu.cheb_filter(ham, to_dev(psi), 3, w.a, w.b, w.a0).cpu().numpy()
    assert relerr(y, oracle.cheb_filter(*ham_args(w), psi, 3, w.a, w.b, w.a0)) <= TOL_F
    ham.destroy()


@pytest.mark.parametrize("n,npw", [(1, 5), (64, 300), (130, 4099), (257, 1031), (512, 2500)])
def test_gram_hermitian_variant(gpu, n, npw):
    """pwh_gram_herm: G = X^H (D X) with a real diagonal D is Hermitian; half of the tiles are computed, the rest
    mirrored -- every entry against the oracle's dot products (H_Psi = Psi^H (H Psi))."""
    rng = np.random.default_rng(n * 7 + npw)
    x = rng.standard_normal((n, npw)) + 1j * rng.standard_normal((n, npw))
    y = x * rng.uniform(-2.0, 3.0, size=npw)[None, :]
    g = gpu.gram(to_dev(x), to_dev(y), hermitian=True).cpu().numpy()
    ref = oracle.gram(x, y)
    assert relerr(g, ref) <= TOL_H
    assert np.abs(g - ref).max() <= 1e-11 * np.abs(ref).max() * math.sqrt(npw)
    assert np.abs(g - g.conj().T).max() <= 1e-12 * np.abs(ref).max()


def test_two_handles_alive(gpu):
    """Two handles with different shared-memory needs alive at once (two k-points on different boxes): the handle made
    first must still work after the second one has been set up, and the other way round."""
    wa = synth.random_problem((48, 48, 180), (14.0, 14.0, 50.0), (0.0, 0.0, 0.0), 5.0, 4, 3, seed=60)
    wb = synth.random_problem((48, 48, 30), (14.0, 14.0, 9.0), (0.25, 0.25, 0.25), 5.0, 4, 3, seed=61)
    wc = synth.random_problem((96, 96, 12), (28.0, 28.0, 4.0), (0.0, 0.0, 0.0), 5.0, 4, 3, seed=62)
    ha, hb, hc = setup(gpu, wa), setup(gpu, wb), setup(gpu, wc)
    for w, h in ((wa, ha), (wb, hb), (wc, hc), (wa, ha)):
        out = gpu.apply_h(h, to_dev(w.psi)).cpu().numpy()
        assert relerr(out, oracle.apply_h(*ham_args(w), w.psi)) <= TOL_H
    for h in (ha, hb, hc):
        h.destroy()


def test_ragged_last_block_through_host_entry(gpu, cfg2):
    """392 bands in column blocks of 200: the ragged 192-band tail picks a different split-K count than the 200-band
    block the workspace was sized for (pwh_workspace_bytes must cover every nband <= nband_max)."""
    import torch
    w = cfg2
    rng = np.random.default_rng(392)
    psi = (rng.standard_normal((392, w.npw)) + 1j * rng.standard_normal((392, w.npw))) / math.sqrt(2.0 * w.npw)
    ham = setup(gpu, w)
    L = gpu.load_library()
    sizes = [int(L.pwh_workspace_bytes(ham.handle, n)) for n in range(1, 401)]
    assert all(b >= a for a, b in zip(sizes, sizes[1:])), "pwh_workspace_bytes must be monotone in nband"
    y_h = torch.from_numpy(psi.copy()).pin_memory()
    gpu.cheb_filter_host(ham, y_h, 3, w.a, w.b, w.a0, block=200)
    idx = [0, 199, 200, 391]
    ref = oracle.cheb_filter(*ham_args(w), psi[idx], 3, w.a, w.b, w.a0)
    assert relerr(y_h.numpy()[idx], ref) <= TOL_F
    ham.destroy()


def test_apply_h_rejects_overlapping_blocks(gpu, cfg1):
    w = cfg1
    ham = setup(gpu, w)
    psi = to_dev(w.psi)
    L = gpu.load_library()
    ws = ham.workspace(w.nband)
    rc = L.pwh_apply_h(ham.handle, w.nband, psi.data_ptr(), w.npw, psi.data_ptr() + 16 * w.npw, w.npw, ws.data_ptr(),
                       ws.numel(), None)
    assert rc == -1 and b"overlap" in L.pwh_last_error()
    ham.destroy()

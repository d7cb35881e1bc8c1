"""Seeded synthetic plane-wave workloads (the five BASELINE.json configs).

This module is the ONLY code shared by the CPU oracle side (tests, bench cpu_baseline) and the
CUDA side.  It holds input generation only -- crystals, G-spheres, V_loc(r), projectors, D, the
starting block Psi and the filter bounds -- and none of the method's arithmetic (no H application,
no FFT, no recurrence, no Gram product).  It imports neither `oracle/` nor the CUDA binding.

The paper's own workloads (255-atom Ti interface, 320-atom Ga2O3; section 5.1) need
ABINIT inputs and PAW datasets that are not available; these seeded crystals stand in for them with the
same object shapes (N plane waves x M bands, M a few % of N as in PAPER.md:165; ~8 projectors per atom;
E_cut ~ 7-8 Ha).  Recipe and every reading of BASELINE.json's config text: DESIGN.md section 3.

Array conventions (used everywhere in this repo):
  * a block of wavefunctions is a C-contiguous complex128 array of shape (nband, npw): row b is band b,
    i.e. the paper's N x M matrix Psi stored column-major with ld = npw;
  * projectors: (nproj, npw) complex128, row i = <G|p_i>, i.e. column-major npw x nproj;
  * V_loc: float64 array of shape (n3, n2, n1), element [i3, i2, i1] at flat index i1 + n1*(i2 + n2*i3);
  * gvec: int32 (npw, 3) reduced integer G components (n1-, n2-, n3-direction).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

SEED_ROOT = (2604, 11139)


@dataclasses.dataclass(frozen=True)
class ConfigSpec:
    """Static description of one BASELINE.json config (no arrays)."""
    cfg_id: int
    name: str
    cell: tuple            # orthorhombic cell edges in bohr
    kpt: tuple             # reduced coordinates
    fft_dims: tuple        # (n1, n2, n3)
    sphere: tuple          # ("grid", R) : |k+n| <= R in units of 2*pi/a (cubic);  ("ecut", E) : |q|^2/2 <= E Ha
    nband: int
    block: int             # bands per cheb_filter call
    natom: int
    lmax_set: str          # "sp" = l=0,1 (4 projectors); "spd-" = l=0,1,2 minus m=+2 (8 projectors)
    depth_range: tuple     # Gaussian well depths U(lo, hi) in Ha
    degree: int
    with_gram: bool


CONFIGS = {
    1: ConfigSpec(1, "cfg1_cubic10.26_16^3_G4_nb16", (10.26,) * 3, (0.0, 0.0, 0.0), (16, 16, 16), ("grid", 4),
                  16, 16, 2, "sp", (-2.0, -0.5), 4, False),
    2: ConfigSpec(2, "cfg2_cubic20_48^3_G12_nb128", (20.0,) * 3, (0.0, 0.0, 0.0), (48, 48, 48), ("grid", 12),
                  128, 128, 8, "spd-", (-2.0, -0.5), 8, False),
    3: ConfigSpec(3, "cfg3_cubic40_k.25_96^3_G24_nb512", (40.0,) * 3, (0.25, 0.25, 0.25), (96, 96, 96), ("grid", 24),
                  512, 512, 64, "spd-", (-2.0, -0.5), 10, True),
    4: ConfigSpec(4, "cfg4_cubic54_128^3_G32_nb1024", (54.0,) * 3, (0.0, 0.0, 0.0), (128, 128, 128), ("grid", 32),
                  1024, 1024, 128, "spd-", (-3.0, -0.5), 12, True),
    5: ConfigSpec(5, "cfg5_ortho50x50x75_k.25_120x120x180_ecut8_nb2048", (50.0, 50.0, 75.0), (0.25, 0.25, 0.25),
                  (120, 120, 180), ("ecut", 8.0), 2048, 512, 216, "spd-", (-2.0, -0.5), 16, True),
}

# exact plane-wave counts (recorded; checked by tests/test_synth.py for the ones cheap to build)
EXPECTED_NPW = {1: 257, 2: 7153, 3: 57925, 4: 137065, 5: 202625}


@dataclasses.dataclass
class Workload:
    spec: ConfigSpec
    lattice: np.ndarray        # (3,3) float64, row i = a_i (bohr)
    kpt: np.ndarray            # (3,) float64 reduced
    fft_dims: np.ndarray       # (3,) int32
    gvec: np.ndarray           # (npw,3) int32
    vloc: np.ndarray           # (n3,n2,n1) float64, Ha
    proj: np.ndarray           # (nproj,npw) complex128
    dij: np.ndarray            # (nproj,) float64, Ha
    psi: Optional[np.ndarray]  # (nband,npw) complex128 or None (when only operators were requested)
    atoms: np.ndarray          # (natom,3) reduced positions
    depths: np.ndarray         # (natom,) Ha
    degree: int
    a: float                   # lower edge of the damped interval
    b: float                   # upper bound of the spectrum
    a0: float                  # normalisation point (filter == 1 there)

    @property
    def npw(self) -> int:
        return int(self.gvec.shape[0])

    @property
    def nproj(self) -> int:
        return int(self.proj.shape[0])

    @property
    def nband(self) -> int:
        return self.spec.nband


def reciprocal(lattice: np.ndarray) -> np.ndarray:
    """B = 2*pi*(A^-1)^T, rows b_i, so that a_i . b_j = 2*pi*delta_ij."""
    return 2.0 * math.pi * np.linalg.inv(lattice).T


def gsphere(spec: ConfigSpec) -> np.ndarray:
    """Integer G vectors inside the cutoff, order: n3 outer, n2, n1 inner, each ascending."""
    n1, n2, n3 = spec.fft_dims
    kind, val = spec.sphere
    k = np.asarray(spec.kpt, dtype=np.float64)
    if kind == "grid":
        R = int(val)
        rng_ = [np.arange(-R - 1, R + 2, dtype=np.int64)] * 3
        # exact integer test: |k+n| <= R with k a multiple of 1/4  ->  sum (4n+4k)^2 <= 16 R^2
        k4 = np.rint(4 * k).astype(np.int64)
        assert np.allclose(4 * k, k4), "grid-unit spheres need k on the 1/4 mesh"
        i3, i2, i1 = np.meshgrid(rng_[2], rng_[1], rng_[0], indexing="ij")
        s = (4 * i1 + k4[0]) ** 2 + (4 * i2 + k4[1]) ** 2 + (4 * i3 + k4[2]) ** 2
        keep = s <= 16 * R * R
    else:
        ecut = float(val)
        lat = np.diag(np.asarray(spec.cell, dtype=np.float64))
        B = reciprocal(lat)
        m = [int(math.ceil(math.sqrt(2 * ecut) / B[i, i])) + 2 for i in range(3)]
        rng_ = [np.arange(-m[i], m[i] + 1, dtype=np.int64) for i in range(3)]
        i3, i2, i1 = np.meshgrid(rng_[2], rng_[1], rng_[0], indexing="ij")
        q1 = (i1 + k[0]) * B[0, 0]
        q2 = (i2 + k[1]) * B[1, 1]
        q3 = (i3 + k[2]) * B[2, 2]
        keep = 0.5 * (q1 * q1 + q2 * q2 + q3 * q3) <= ecut
    g = np.stack([i1[keep], i2[keep], i3[keep]], axis=1).astype(np.int32)
    # the sphere must fit the box without wrap collisions
    for ax, n in enumerate((n1, n2, n3)):
        span = int(g[:, ax].max()) - int(g[:, ax].min()) + 1
        assert span <= n, f"sphere does not fit the FFT box along axis {ax}"
    return np.ascontiguousarray(g)


def real_ylm(lmax_set: str, q: np.ndarray) -> np.ndarray:
    """Real orthonormal spherical harmonics Y_lm(q^), order m=-l..l; at q=0: Y_00 only.  -> (nlm, npw)."""
    qn = np.linalg.norm(q, axis=1)
    safe = np.where(qn > 0, qn, 1.0)
    x, y, z = (q[:, 0] / safe, q[:, 1] / safe, q[:, 2] / safe)
    nz = (qn > 0).astype(np.float64)
    out = [np.full(q.shape[0], 1.0 / math.sqrt(4 * math.pi))]
    c1 = math.sqrt(3.0 / (4 * math.pi))
    out += [c1 * y * nz, c1 * z * nz, c1 * x * nz]
    if lmax_set == "spd-":
        c2 = 0.5 * math.sqrt(15.0 / math.pi)
        c20 = 0.25 * math.sqrt(5.0 / math.pi)
        out += [c2 * x * y * nz, c2 * y * z * nz, c20 * (3 * z * z - 1.0) * nz, c2 * x * z * nz]  # m=+2 dropped
    elif lmax_set != "sp":
        raise ValueError(lmax_set)
    return np.stack(out, axis=0)


def _orthonormalise(psi_bn: np.ndarray, qr: str) -> np.ndarray:
    """Orthonormalise the bands (rows) of psi_bn.  Input preparation only."""
    if qr == "numpy":
        qmat, _ = np.linalg.qr(psi_bn.T)          # (npw, nband) Householder QR
        return np.ascontiguousarray(qmat.T)
    if qr == "torch-cuda":
        import torch
        t = torch.from_numpy(psi_bn).cuda()
        qmat, _ = torch.linalg.qr(t.T.contiguous())
        out = qmat.T.contiguous().cpu().numpy()
        del t, qmat
        torch.cuda.empty_cache()
        return out
    if qr == "none":
        return psi_bn
    raise ValueError(qr)


def make_workload(cfg_id: int, *, with_psi: bool = True, qr: str = "numpy",
                  nband: Optional[int] = None) -> Workload:
    """Build config `cfg_id`.  `nband` (optional) overrides the number of bands drawn (the first `nband`
    columns of the same random stream are NOT guaranteed to equal the full draw after orthonormalisation; use it
    only for self-contained smaller problems).  `qr` selects where the one-off orthonormalisation runs."""
    spec = CONFIGS[cfg_id]
    if nband is not None:
        spec = dataclasses.replace(spec, nband=int(nband), block=min(spec.block, int(nband)))
    ss = np.random.SeedSequence(list(SEED_ROOT) + [cfg_id])
    s_atoms, s_depth, s_d, s_psi = ss.spawn(4)

    lattice = np.diag(np.asarray(spec.cell, dtype=np.float64))
    B = reciprocal(lattice)
    omega = abs(np.linalg.det(lattice))
    kpt = np.asarray(spec.kpt, dtype=np.float64)
    n1, n2, n3 = spec.fft_dims
    gvec = gsphere(spec)
    npw = gvec.shape[0]
    q = (gvec.astype(np.float64) + kpt[None, :]) @ B        # (npw,3) Cartesian k+G (rows b_i)
    q2 = np.einsum("ij,ij->i", q, q)

    atoms = np.random.default_rng(s_atoms).random((spec.natom, 3))
    lo, hi = spec.depth_range
    depths = np.random.default_rng(s_depth).uniform(lo, hi, size=spec.natom)

    # V_loc(r) = 0.5 + sum_a depth_a exp(-d^2/2), d = minimum-image distance (orthorhombic => separable)
    def axis_gauss(n, length, frac):
        r = np.arange(n, dtype=np.float64)[None, :] / n - frac[:, None]
        r -= np.rint(r)
        return np.exp(-0.5 * (r * length) ** 2)              # (natom, n)
    g1 = axis_gauss(n1, spec.cell[0], atoms[:, 0])
    g2 = axis_gauss(n2, spec.cell[1], atoms[:, 1])
    g3 = axis_gauss(n3, spec.cell[2], atoms[:, 2])
    g12 = (g2[:, :, None] * g1[:, None, :]).reshape(spec.natom, n2 * n1)
    vloc = 0.5 + ((g3 * depths[:, None]).T @ g12).reshape(n3, n2, n1)
    vloc = np.ascontiguousarray(vloc)

    # projectors beta_{a,lm}(G) = (4 pi / sqrt(Omega)) exp(-|q|^2 r_c^2 / 2) Y_lm(q^) exp(-i q.tau_a), r_c = 1 bohr
    ylm = real_ylm(spec.lmax_set, q)
    nlm = ylm.shape[0]
    radial = (4 * math.pi / math.sqrt(omega)) * np.exp(-0.5 * q2)
    flm = ylm * radial[None, :]
    nproj = spec.natom * nlm
    proj = np.empty((nproj, npw), dtype=np.complex128)
    kg = gvec.astype(np.float64) + kpt[None, :]
    for ia in range(spec.natom):
        phase = np.exp(-2j * math.pi * (kg @ atoms[ia]))
        np.multiply(flm, phase[None, :], out=proj[ia * nlm:(ia + 1) * nlm])
    dij = np.random.default_rng(s_d).uniform(-5.0, 5.0, size=nproj)

    # filter bounds (BASELINE.json: a = median diag, b = max kin + max V + sum |D| ||beta||^2; a0 = min diag)
    kin = 0.5 * q2
    p2 = (proj.real ** 2 + proj.imag ** 2)
    diag = kin + vloc.mean() + dij @ p2
    a = float(np.median(diag))
    b = float(kin.max() + vloc.max() + np.abs(dij) @ p2.sum(axis=1))
    a0 = float(diag.min())
    del p2

    psi = None
    if with_psi:
        rng = np.random.default_rng(s_psi)
        psi = np.empty((spec.nband, npw), dtype=np.complex128)
        scale = 1.0 / (math.sqrt(2.0) * (1.0 + q2))
        chunk = 64
        for b0 in range(0, spec.nband, chunk):
            b1 = min(spec.nband, b0 + chunk)
            z = rng.standard_normal((b1 - b0, npw, 2))
            psi[b0:b1] = (z[..., 0] + 1j * z[..., 1]) * scale[None, :]
        psi = _orthonormalise(psi, qr)

    return Workload(spec=spec, lattice=lattice, kpt=kpt, fft_dims=np.asarray(spec.fft_dims, dtype=np.int32),
                    gvec=gvec, vloc=vloc, proj=proj, dij=dij, psi=psi, atoms=atoms, depths=depths,
                    degree=spec.degree, a=a, b=b, a0=a0)


def gsphere_general(lattice: np.ndarray, kpt, dims, ecut: float) -> np.ndarray:
    """Integer G with 1/2 |B (k + n)|^2 <= ecut for a general (non-orthogonal) lattice, order n3 outer, n1 inner."""
    B = reciprocal(np.asarray(lattice, dtype=np.float64))
    k = np.asarray(kpt, dtype=np.float64)
    rng_ = [np.arange(-(int(n) // 2) - 1, int(n) // 2 + 2, dtype=np.int64) for n in dims]
    i3, i2, i1 = np.meshgrid(rng_[2], rng_[1], rng_[0], indexing="ij")
    c = np.stack([i1 + k[0], i2 + k[1], i3 + k[2]], axis=-1) @ B
    keep = 0.5 * np.einsum("...i,...i->...", c, c) <= float(ecut)
    g = np.stack([i1[keep], i2[keep], i3[keep]], axis=1).astype(np.int32)
    for ax, n in enumerate(dims):
        span = int(g[:, ax].max()) - int(g[:, ax].min()) + 1
        assert span <= n, f"sphere does not fit the FFT box along axis {ax}"
    return np.ascontiguousarray(g)


def random_problem(dims, cell, kpt, ecut, nproj, nband, seed, gvec: Optional[np.ndarray] = None) -> Workload:
    """A small unstructured problem for parity edge cases (odd radices, non-cubic boxes, k-shifts, general lattices):
    the plane waves with 1/2|k+G|^2 <= ecut (or the given `gvec` set), random V_loc, random dense projectors, random
    (not orthonormal) Psi.  `cell` is either three orthorhombic edge lengths or a full 3x3 lattice (row i = a_i).
    Inputs only; the filter bounds are crude brackets (a0 < a < b) that keep the recurrence well-conditioned."""
    rng = np.random.default_rng(np.random.SeedSequence(list(SEED_ROOT) + [1000 + int(seed)]))
    cell_arr = np.asarray(cell, dtype=np.float64)
    general = cell_arr.shape == (3, 3)
    edges = tuple(float(np.linalg.norm(cell_arr[i])) for i in range(3)) if general else tuple(float(c) for c in cell_arr)
    spec = ConfigSpec(1000 + int(seed), f"random_{dims[0]}x{dims[1]}x{dims[2]}", edges,
                      tuple(float(k) for k in kpt), tuple(int(d) for d in dims), ("ecut", float(ecut)), int(nband),
                      int(nband), 0, "sp", (0.0, 0.0), 3, False)
    lattice = cell_arr.copy() if general else np.diag(cell_arr)
    B = reciprocal(lattice)
    k = np.asarray(spec.kpt, dtype=np.float64)
    if gvec is None:
        gvec = gsphere_general(lattice, k, spec.fft_dims, ecut) if general else gsphere(spec)
    gvec = np.ascontiguousarray(gvec, dtype=np.int32)
    npw = gvec.shape[0]
    q = (gvec.astype(np.float64) + k[None, :]) @ B
    kin = 0.5 * np.einsum("ij,ij->i", q, q)
    n1, n2, n3 = spec.fft_dims
    vloc = rng.uniform(-1.0, 1.0, size=(n3, n2, n1))
    proj = (rng.standard_normal((nproj, npw)) + 1j * rng.standard_normal((nproj, npw))) * (0.5 / math.sqrt(npw))
    dij = rng.uniform(-5.0, 5.0, size=nproj)
    psi = (rng.standard_normal((nband, npw)) + 1j * rng.standard_normal((nband, npw))) / math.sqrt(2.0 * npw)
    p2 = proj.real ** 2 + proj.imag ** 2
    b = float(kin.max() + vloc.max() + (np.abs(dij) @ p2.sum(axis=1) if nproj else 0.0))
    lo = float(kin.min() + vloc.min() - (np.abs(dij) @ p2.sum(axis=1) if nproj else 0.0))
    a = lo + 0.5 * (b - lo)
    a0 = lo - 0.05 * (b - lo)
    return Workload(spec=spec, lattice=lattice, kpt=k, fft_dims=np.asarray(spec.fft_dims, dtype=np.int32), gvec=gvec,
                    vloc=np.ascontiguousarray(vloc), proj=np.ascontiguousarray(proj), dij=dij,
                    psi=np.ascontiguousarray(psi), atoms=np.zeros((0, 3)), depths=np.zeros((0,)), degree=3, a=a, b=b,
                    a0=a0)


def paw_blocks(nproj: int, dij: np.ndarray, seed: int, block_sizes=None):
    """Per-atom dense blocks for the PAW-style generalised problem: the projector
    index is cut into consecutive blocks (one per atom; 8 projectors per atom in the BASELINE.json configs, an uneven mix
    for the random test problems), D^R = diag(the config's D_i) + a seeded Hermitian off-diagonal part of relative size
    0.3, Q^R = B B^H / (2 n_R) + a small indefinite Hermitian part (positive enough that S = I + P Q P^H stays positive
    definite).  Returns (offsets int32 [nblocks + 1], [D^R], [Q^R]).  Inputs only."""
    rng = np.random.default_rng(np.random.SeedSequence(list(SEED_ROOT) + [5000 + int(seed)]))
    if block_sizes is None:
        block_sizes = [8] * (nproj // 8) if nproj % 8 == 0 and nproj > 0 else []
        rest = nproj - sum(block_sizes)
        cyc = [4, 1, 5, 3, 8, 2]
        i = 0
        while rest > 0:
            b = min(rest, cyc[i % len(cyc)])
            block_sizes.append(b)
            rest -= b
            i += 1
    assert sum(block_sizes) == nproj
    offsets = np.concatenate([[0], np.cumsum(block_sizes)]).astype(np.int32)
    dblocks, qblocks = [], []
    for r, n in enumerate(block_sizes):
        lo = int(offsets[r])
        a = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
        d = np.diag(np.asarray(dij[lo:lo + n], dtype=np.float64)).astype(np.complex128) + 0.3 * (a + a.conj().T) / 2
        bm = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
        c = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
        q = bm @ bm.conj().T / (2.0 * n) + 0.02 * (c + c.conj().T) / 2
        dblocks.append(np.ascontiguousarray((d + d.conj().T) / 2))
        qblocks.append(np.ascontiguousarray((q + q.conj().T) / 2))
    return offsets, dblocks, qblocks

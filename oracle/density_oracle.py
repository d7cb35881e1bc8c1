"""CPU oracle for the electronic density accumulation and for the band-sharded (multi-GPU) data movement of SURVEY.md
section 8f row f4 -- TEST INFRASTRUCTURE, not the product.  Plain numpy on top of the C oracle's unnormalised 3-D DFT
(oracle/pw_oracle.c orc_dft3d, itself pinned against the DFT definition and numpy.fft in tests/test_oracle_pins.py).

Density (Algorithm 3 step 10: "Accumulate electronic density from f, Psi for current k-point (FFT on GPU)";
PAPER.md:110: "The electronic density is then computed from the occupations and the converged wave function coefficients
for every k-point, using an FFT operation on GPU"):

    u_i(r) = sum_G psi_i(G) exp(+2 pi i sum_a n_G,a r_a / n_a)          (the unnormalised inverse DFT of DESIGN.md reading R6)
    rho(r) += weight * sum_i f_i |u_i(r)|^2

The paper prints no formula; `weight` carries whatever the caller's convention needs (k-point weight, 1/Omega): with
weight = w_k / Omega and orthonormal bands, sum_r rho(r) Omega / F = sum_k w_k sum_i f_i (Parseval) -- DESIGN.md reading R17.

Band sharding (section 2.3, Figure 1; section 3.5): the "column-distributed" layout gives
every process a contiguous range of bands with all plane waves, the "row-distributed" layout a contiguous range of plane
waves with all bands, "to distribute plane-wave indices as uniformly as possible"; the all-to-all (mpi-A) switches
between them, and A^H B over row-distributed data is the sum of the per-process products (mpi-R).
"""
from __future__ import annotations

import numpy as np

from . import pw_oracle


def scatter_box(fft_dims, gvec, coeff) -> np.ndarray:
    """The (n3, n2, n1) box holding coeff[g] at wrap(n_G) and zero elsewhere (SURVEY.md 8c definition 2)."""
    n1, n2, n3 = (int(v) for v in fft_dims)
    box = np.zeros((n3, n2, n1), dtype=np.complex128)
    g = np.asarray(gvec, dtype=np.int64)
    box[g[:, 2] % n3, g[:, 1] % n2, g[:, 0] % n1] = coeff
    return box


def realspace(fft_dims, gvec, psi_band) -> np.ndarray:
    """u(r) on the (n3, n2, n1) grid for one band (unnormalised inverse DFT, sign +)."""
    return pw_oracle.dft3d(scatter_box(fft_dims, gvec, psi_band), +1)


def density(fft_dims, gvec, psi, occ, weight: float = 1.0, rho=None) -> np.ndarray:
    """rho (n3, n2, n1) float64 += weight * sum_i occ[i] |u_i(r)|^2 for the block psi (nband, npw); band by band, in order."""
    n1, n2, n3 = (int(v) for v in fft_dims)
    out = np.zeros((n3, n2, n1), dtype=np.float64) if rho is None else np.array(rho, dtype=np.float64, copy=True)
    psi = np.asarray(psi, dtype=np.complex128).reshape(-1, np.shape(gvec)[0])
    occ = np.asarray(occ, dtype=np.float64)
    assert occ.shape == (psi.shape[0],)
    acc = np.zeros_like(out)
    for i in range(psi.shape[0]):
        u = realspace(fft_dims, gvec, psi[i])
        acc += occ[i] * (u.real * u.real + u.imag * u.imag)
    return out + weight * acc


def density_kpoints(fft_dims, kpoints, rho=None) -> np.ndarray:
    """Sum over k-points (Algorithm 3 steps 9-10): kpoints = iterable of (gvec, psi, occ, weight)."""
    n1, n2, n3 = (int(v) for v in fft_dims)
    out = np.zeros((n3, n2, n1), dtype=np.float64) if rho is None else np.array(rho, dtype=np.float64, copy=True)
    for gvec, psi, occ, weight in kpoints:
        out = density(fft_dims, gvec, psi, occ, weight, out)
    return out


# ---------------------------------------------------------------------------------------------------------------
# band sharding: ownership ranges and the two layouts (pure index bookkeeping, bit-exact)
# ---------------------------------------------------------------------------------------------------------------
def split_range(n: int, p: int, r: int):
    """[lo, hi) of part r when n items are cut into p contiguous parts "as uniformly as possible":
    the first n % p parts have one item more."""
    q, rem = divmod(int(n), int(p))
    lo = r * q + min(r, rem)
    return lo, lo + q + (1 if r < rem else 0)


def column_shard(psi, p: int, r: int) -> np.ndarray:
    """psi is (nband, npw): the bands [lo, hi) of rank r with all plane waves (column-distributed)."""
    lo, hi = split_range(psi.shape[0], p, r)
    return psi[lo:hi]


def row_shard(psi, p: int, r: int) -> np.ndarray:
    """The plane waves [lo, hi) of rank r for all bands (row-distributed)."""
    lo, hi = split_range(psi.shape[1], p, r)
    return psi[:, lo:hi]


def gram_row_distributed(x, y, p: int) -> np.ndarray:
    """X^H Y as the sum over the p row shards of the per-shard products, summed in rank order (mpi-R)."""
    g = None
    for r in range(p):
        part = pw_oracle.gram(np.ascontiguousarray(row_shard(x, p, r)), np.ascontiguousarray(row_shard(y, p, r)))
        g = part if g is None else g + part
    return g

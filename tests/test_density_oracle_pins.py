"""Pins of the density / band-sharding oracle (oracle/density_oracle.py): closed forms for one and two
plane waves, Parseval, the autocorrelation form of the density's Fourier coefficients by brute force, numpy's ifftn as a
library special case, hand-written ownership ranges.  CPU only; nothing here compares the oracle with itself."""
import itertools

import numpy as np
import pytest

from oracle import density_oracle as dn

DIMS = (12, 10, 8)                      # n1, n2, n3 all different: an axis mix-up cannot pass


def small_sphere(rmax2=5):
    g = [(a, b, c) for a, b, c in itertools.product(range(-2, 3), repeat=3) if a * a + b * b + c * c <= rmax2]
    return np.asarray(g, dtype=np.int32)


def grid(dims):
    n1, n2, n3 = dims
    r3, r2, r1 = np.meshgrid(np.arange(n3), np.arange(n2), np.arange(n1), indexing="ij")
    return r1, r2, r3


def test_single_plane_wave_gives_a_constant_density():
    g = small_sphere()
    for j in (0, 7, len(g) - 1):
        psi = np.zeros((1, len(g)), dtype=np.complex128)
        psi[0, j] = 0.6 - 0.8j
        rho = dn.density(DIMS, g, psi, [1.7])
        assert rho.shape == (DIMS[2], DIMS[1], DIMS[0])
        assert np.abs(rho - 1.7).max() <= 1e-14


@pytest.mark.parametrize("ga,gb", [((1, 0, 0), (-1, 0, 0)), ((0, 2, 0), (0, 0, -1)), ((1, -1, 2), (0, 1, 1))])
def test_two_plane_waves_closed_form(ga, gb):
    """|a e^{i Ga.r} + b e^{i Gb.r}|^2 = |a|^2 + |b|^2 + 2 Re(conj(a) b e^{i (Gb-Ga).r}) on the grid, per axis."""
    g = small_sphere(6)
    ia = int(np.where((g == ga).all(axis=1))[0][0])
    ib = int(np.where((g == gb).all(axis=1))[0][0])
    a, b = 0.3 + 0.4j, -0.5 + 0.2j
    psi = np.zeros((1, len(g)), dtype=np.complex128)
    psi[0, ia], psi[0, ib] = a, b
    r1, r2, r3 = grid(DIMS)
    d = np.asarray(gb) - np.asarray(ga)
    phase = 2 * np.pi * (d[0] * r1 / DIMS[0] + d[1] * r2 / DIMS[1] + d[2] * r3 / DIMS[2])
    ref = 2.5 * (abs(a) ** 2 + abs(b) ** 2 + 2 * (np.conj(a) * b * np.exp(1j * phase)).real)
    rho = dn.density(DIMS, g, psi, [2.5])
    assert np.abs(rho - ref).max() <= 1e-13


def test_parseval_and_positivity():
    rng = np.random.default_rng(5)
    g = small_sphere()
    psi = rng.standard_normal((4, len(g))) + 1j * rng.standard_normal((4, len(g)))
    occ = np.asarray([2.0, 1.0, 0.5, 0.0])
    rho = dn.density(DIMS, g, psi, occ, weight=0.25)
    f = DIMS[0] * DIMS[1] * DIMS[2]
    want = 0.25 * f * float((occ * (np.abs(psi) ** 2).sum(axis=1)).sum())
    assert abs(rho.sum() - want) <= 1e-12 * want
    assert rho.min() >= 0.0


def test_fourier_coefficients_are_the_autocorrelation_by_brute_force():
    """(1/F) sum_r rho(r) e^{-2 pi i m.r/n} = sum_i f_i sum_G conj(psi_i(G)) psi_i(G + m): plain loops over the G set; the box
    is large enough (n > 4 max|G|) that no difference G' - G aliases."""
    rng = np.random.default_rng(6)
    g = small_sphere(5)                                  # |n_a| <= 2, box sides 12, 10, 9 > 8
    dims = (12, 10, 9)
    psi = rng.standard_normal((3, len(g))) + 1j * rng.standard_normal((3, len(g)))
    occ = np.asarray([1.0, 0.75, 0.3])
    rho = dn.density(dims, g, psi, occ)
    rhat = np.fft.fftn(rho) / rho.size                    # axes (n3, n2, n1); e^{-i}: the analysis transform
    index = {tuple(v): j for j, v in enumerate(g.tolist())}
    worst = 0.0
    for m in itertools.product(range(-4, 5), repeat=3):
        s = 0.0j
        for j, v in enumerate(g.tolist()):
            k = index.get((v[0] + m[0], v[1] + m[1], v[2] + m[2]))
            if k is not None:
                s += (occ * np.conj(psi[:, j]) * psi[:, k]).sum()
        worst = max(worst, abs(rhat[m[2] % dims[2], m[1] % dims[1], m[0] % dims[0]] - s))
    assert worst <= 1e-13


def test_numpy_ifftn_special_case_and_wraparound():
    rng = np.random.default_rng(7)
    g = small_sphere()
    psi = rng.standard_normal((2, len(g))) + 1j * rng.standard_normal((2, len(g)))
    occ = np.asarray([1.0, 2.0])
    ref = np.zeros((DIMS[2], DIMS[1], DIMS[0]))
    for i in range(2):
        box = np.zeros((DIMS[2], DIMS[1], DIMS[0]), dtype=np.complex128)
        for j, (a, b, c) in enumerate(g.tolist()):
            box[c % DIMS[2], b % DIMS[1], a % DIMS[0]] = psi[i, j]       # negative components wrap to n - |n|
        u = np.fft.ifftn(box) * box.size
        ref += occ[i] * np.abs(u) ** 2
    assert np.abs(dn.density(DIMS, g, psi, occ) - ref).max() <= 1e-12 * ref.max()


def test_accumulation_band_blocks_and_kpoints():
    rng = np.random.default_rng(8)
    g = small_sphere()
    g2 = small_sphere(3)
    psi = rng.standard_normal((5, len(g))) + 1j * rng.standard_normal((5, len(g)))
    psi2 = rng.standard_normal((2, len(g2))) + 1j * rng.standard_normal((2, len(g2)))
    occ, occ2 = rng.uniform(0, 2, 5), rng.uniform(0, 2, 2)
    whole = dn.density(DIMS, g, psi, occ, 0.5)
    parts = dn.density(DIMS, g, psi[3:], occ[3:], 0.5, dn.density(DIMS, g, psi[:3], occ[:3], 0.5))
    assert np.abs(whole - parts).max() <= 1e-13 * whole.max()
    assert np.abs(dn.density(DIMS, g, psi, 3.0 * occ, 0.5) - 3.0 * whole).max() <= 1e-12 * whole.max()
    both = dn.density_kpoints(DIMS, [(g, psi, occ, 0.5), (g2, psi2, occ2, 1.5)])
    assert np.abs(both - (whole + dn.density(DIMS, g2, psi2, occ2, 1.5))).max() <= 1e-13 * both.max()


def test_split_range_hand_values_and_cover():
    assert [dn.split_range(10, 4, r) for r in range(4)] == [(0, 3), (3, 6), (6, 8), (8, 10)]
    assert [dn.split_range(3, 4, r) for r in range(4)] == [(0, 1), (1, 2), (2, 3), (3, 3)]
    for n, p in [(257, 2), (7153, 8), (16, 3), (5, 5)]:
        parts = [dn.split_range(n, p, r) for r in range(p)]
        assert parts[0][0] == 0 and parts[-1][1] == n
        assert all(parts[r][1] == parts[r + 1][0] for r in range(p - 1))
        sizes = [hi - lo for lo, hi in parts]
        assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)


def test_shards_tile_the_block_and_row_distributed_gram_is_the_product():
    rng = np.random.default_rng(9)
    x = rng.standard_normal((7, 61)) + 1j * rng.standard_normal((7, 61))
    y = rng.standard_normal((5, 61)) + 1j * rng.standard_normal((5, 61))
    for p in (1, 2, 3, 4):
        assert np.array_equal(np.concatenate([dn.column_shard(x, p, r) for r in range(p)], axis=0), x)
        assert np.array_equal(np.concatenate([dn.row_shard(x, p, r) for r in range(p)], axis=1), x)
        g = dn.gram_row_distributed(x, y, p)
        ref = np.conj(x) @ y.T                                           # G[i, j] = sum_g conj(x[i, g]) y[j, g]
        assert np.abs(g - ref).max() <= 1e-13 * np.abs(ref).max()

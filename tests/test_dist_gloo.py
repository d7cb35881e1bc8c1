"""The band-sharded multi-GPU layer (paper_2604_11139_b200/dist.py) on CPU: world sizes 2 and 3 over gloo.
The transpositions are pure data movement and must be bit-exact against the oracle's ownership slices; the products over
row-distributed data are checked with the oracle's Gram / numpy injected as the local kernels (libpwham has no CPU path -- on a
GPU the same code calls pwh_gram / pwh_rotate / pwh_density_accumulate, tests/test_gpu_dist.py)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

NBAND, NPW = 7, 61                         # neither divides by 2 or 3: ragged shards in both layouts
DIMS = (12, 10, 8)


def _blocks():
    rng = np.random.default_rng(42)
    x = rng.standard_normal((NBAND, NPW)) + 1j * rng.standard_normal((NBAND, NPW))
    y = rng.standard_normal((NBAND, NPW)) + 1j * rng.standard_normal((NBAND, NPW))
    q = rng.standard_normal((NBAND, NBAND)) + 1j * rng.standard_normal((NBAND, NBAND))
    return x, y, q


def _gvec():
    import itertools
    g = [v for v in itertools.product(range(-2, 3), repeat=3) if sum(c * c for c in v) <= 6]
    return np.asarray(g[:NPW], dtype=np.int32)


def _worker(rank, world, port):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from oracle import density_oracle as dn
        from paper_2604_11139_b200.dist import BandSharded, split_range
        x, y, q = _blocks()
        sh = BandSharded(NBAND, NPW)
        assert (sh.world, sh.rank) == (world, rank)
        assert sh.bands == dn.split_range(NBAND, world, rank) == split_range(NBAND, world, rank)
        assert sh.rows == dn.split_range(NPW, world, rank)
        xc = torch.from_numpy(np.ascontiguousarray(dn.column_shard(x, world, rank)))
        yc = torch.from_numpy(np.ascontiguousarray(dn.column_shard(y, world, rank)))

        # mpi-A: bit-exact against the oracle's slices, and the round trip is the identity
        xr = sh.to_rows(xc)
        assert np.array_equal(xr.numpy(), dn.row_shard(x, world, rank))
        assert torch.equal(sh.to_cols(xr), xc)
        assert sh.alltoall_bytes() == 16 * sh.nband_local * (NPW - sh.nrow_local)

        # mpi-R: Gram over row shards (oracle's plain double loop as the local product), replicated result
        def local_gram(a, b):
            return torch.from_numpy(oracle.gram(a.numpy(), b.numpy()))
        g = sh.gram(xc, yc, local_gram=local_gram).numpy()
        ref = np.conj(x) @ y.T
        assert np.abs(g - ref).max() <= 1e-13 * np.abs(ref).max()

        # rotation Psi <- Psi Q on the row shards: new band j = sum_i Q[i, j] old band i
        def local_rotate(rows, qq):
            return torch.from_numpy(qq.numpy().T @ rows.numpy())
        rot = sh.rotate(xc, torch.from_numpy(q), local_rotate=local_rotate).numpy()
        assert np.abs(rot - dn.column_shard(q.T @ x, world, rank)).max() <= 1e-13 * np.abs(x).max() * NBAND

        # mpi-sR
        lo, hi = sh.bands
        lam = np.linspace(-1.0, 2.0, NBAND)
        mn, mx = sh.minmax(lam[lo:hi].min() if hi > lo else np.inf, lam[lo:hi].max() if hi > lo else -np.inf)
        assert (mn, mx) == (-1.0, 2.0)
        assert np.array_equal(sh.gather_band_values(torch.from_numpy(lam[lo:hi].copy())).numpy(), lam)

        # density: private partial arrays, one all-reduce
        gv = _gvec()
        occ = np.linspace(2.0, 0.0, NBAND)

        def local_density(ham, psi, f, rho, weight):
            rho += torch.from_numpy(dn.density(DIMS, gv, psi.numpy(), f.numpy(), weight))
            return rho
        rho = torch.zeros((DIMS[2], DIMS[1], DIMS[0]), dtype=torch.float64)
        sh.density(None, xc, torch.from_numpy(occ), rho, 0.5, local_density=local_density)
        sh.reduce_density(rho)
        ref_rho = dn.density(DIMS, gv, x, occ, 0.5)
        assert np.abs(rho.numpy() - ref_rho).max() <= 1e-12 * ref_rho.max()
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,port", [(2, 29641), (3, 29643)])
def test_band_sharded_layer_gloo(world, port):
    mp.spawn(_worker, args=(world, port), nprocs=world, join=True)


def test_more_ranks_than_bands_gives_empty_shards():
    from paper_2604_11139_b200.dist import split_range
    assert [split_range(2, 4, r) for r in range(4)] == [(0, 1), (1, 2), (2, 2), (2, 2)]


def test_single_process_needs_no_process_group():
    from paper_2604_11139_b200.dist import BandSharded
    sh = BandSharded(5, 11)
    x = torch.arange(55, dtype=torch.float64).view(5, 11).to(torch.complex128)
    assert sh.world == 1 and sh.bands == (0, 5) and sh.rows == (0, 11)
    assert torch.equal(sh.to_rows(x), x) and torch.equal(sh.to_cols(x), x)
    assert sh.minmax(1.0, 2.0) == (1.0, 2.0)

"""The band-sharded layer (paper_2604_11139_b200/dist.py) on one GPU: a single-rank NCCL group, so that
the default local kernels (pwh_gram, pwh_rotate, pwh_density_accumulate, pwh_cheb_filter) are the ones that run; the
multi-rank data movement itself is covered on CPU by tests/test_dist_gloo.py.  Needs a B200 (`-m gpu`)."""
import os

import numpy as np
import pytest

import oracle
from oracle import density_oracle as dn

pytestmark = pytest.mark.gpu


def relerr(x, ref):
    return float(np.linalg.norm(np.asarray(x) - np.asarray(ref)) / max(np.linalg.norm(ref), 1e-300))


@pytest.fixture(scope="module")
def group():
    import torch
    import torch.distributed as dist
    assert torch.cuda.is_available()
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT="29655", RANK="0", WORLD_SIZE="1")
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    yield dist
    dist.destroy_process_group()


def test_single_rank_nccl_group_runs_the_cuda_kernels(group, cfg2):
    import torch
    from paper_2604_11139_b200 import binding
    from paper_2604_11139_b200.dist import BandSharded
    w = cfg2
    ham = binding.ham_setup(w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, w.proj, w.dij)
    sh = BandSharded(w.nband, w.npw)
    assert sh.world == 1 and sh.bands == (0, w.nband)
    psi = torch.from_numpy(w.psi).cuda()
    n0 = binding.launch_count()
    hpsi = sh.apply_h(ham, psi)
    g = sh.gram(psi, hpsi).cpu().numpy()
    ref_h = oracle.apply_h(w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, w.proj, w.dij, w.psi)
    assert relerr(g, oracle.gram(w.psi, ref_h)) <= 1e-11
    lam, x, _ = binding.heev(torch.from_numpy(oracle.gram(w.psi, ref_h)).cuda())
    rot = sh.rotate(psi, x).cpu().numpy()
    assert relerr(rot, x.cpu().numpy().T @ w.psi) <= 1e-11
    occ = np.linspace(2.0, 0.0, w.nband)
    n1, n2, n3 = (int(v) for v in w.fft_dims)
    rho = torch.zeros((n3, n2, n1), dtype=torch.float64, device="cuda")
    sh.reduce_density(sh.density(ham, psi, torch.from_numpy(occ).cuda(), rho, 0.5))
    assert relerr(rho.cpu().numpy(), dn.density(w.fft_dims, w.gvec, w.psi, occ, 0.5)) <= 1e-11
    mn, mx = sh.minmax(float(lam.min()), float(lam.max()), device="cuda")
    assert (mn, mx) == (float(lam.min()), float(lam.max()))
    assert binding.launch_count() > n0
    ham.destroy()

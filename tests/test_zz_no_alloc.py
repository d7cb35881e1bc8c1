"""pwh_gram_static -- the Gram product for callers that may not allocate (split-K scratch in a static device array of
PWH_GRAM_STATIC_MAX_ENTRIES complex128, include/pwham.h) -- against the existing path pwh_gram on the same inputs, at the
tolerance of the other Gram tests (relative Frobenius error 1e-11), on two calls in a row.  Collected last on purpose (the file
name sorts after every other test file).  Needs a B200 (`-m gpu`)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_H = 1e-11


def relerr(x, ref):
    return float(np.linalg.norm(np.asarray(x) - np.asarray(ref)) / max(np.linalg.norm(ref), 1e-300))


@pytest.fixture(scope="module")
def gpu():
    import torch
    from paper_2604_11139_b200 import binding
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    binding.load_library()
    return binding


def blocks(nx, ny, npw, seed):
    import torch
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((nx, npw)) + 1j * rng.standard_normal((nx, npw))
    y = rng.standard_normal((ny, npw)) + 1j * rng.standard_normal((ny, npw))
    return torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()


def test_gram_static_matches_gram_on_two_calls_in_a_row(gpu):
    """First a large product whose partial sums fill most of the static array (700 x 700: the split count is capped at 2),
    then -- at once, on the same stream -- a small ragged one that reuses the array while it still holds the first call's
    partial sums; then the first one again.  Each result against pwh_gram and against the plain product."""
    import torch
    xa, ya = blocks(700, 700, 3001, 1)
    xb, yb = blocks(37, 130, 4099, 2)
    out_a = torch.empty((700, 700), dtype=torch.complex128, device="cuda")
    out_b = torch.empty((130, 37), dtype=torch.complex128, device="cuda")
    n0 = gpu.launch_count()
    ga = gpu.gram_static(xa, ya, out=out_a).clone()
    gb = gpu.gram_static(xb, yb, out=out_b).clone()
    ga2 = gpu.gram_static(xa, ya, out=out_a).clone()
    torch.cuda.synchronize()
    assert gpu.launch_count() - n0 == 6                           # two kernels per call, nothing else
    ref_a, ref_b = gpu.gram(xa, ya), gpu.gram(xb, yb)             # the existing path (caller-provided workspace)
    assert relerr(ga.cpu().numpy(), ref_a.cpu().numpy()) <= TOL_H
    assert relerr(gb.cpu().numpy(), ref_b.cpu().numpy()) <= TOL_H
    assert torch.equal(ga, ga2)                                   # deterministic: fixed-order second-stage sum
    assert relerr(ga.cpu().numpy(), (xa.conj() @ ya.T).cpu().numpy()) <= TOL_H
    assert relerr(gb.cpu().numpy(), (xb.conj() @ yb.T).cpu().numpy()) <= TOL_H


def test_gram_static_small_shapes_and_padded_leading_dimensions(gpu):
    import torch
    for nx, ny, npw, seed in [(1, 1, 1, 3), (3, 5, 17, 4), (128, 128, 7153, 5), (1024, 1024, 900, 6)]:
        x, y = blocks(nx, ny, npw, seed)
        g = gpu.gram_static(x, y)
        assert relerr(g.cpu().numpy(), gpu.gram(x, y).cpu().numpy()) <= TOL_H, (nx, ny, npw)
    big = torch.full((16, 300 + 9), float("nan"), dtype=torch.complex128, device="cuda")
    x, y = blocks(16, 16, 300, 7)
    big[:, :300] = x
    g = gpu.gram_static(big[:, :300], y)
    assert relerr(g.cpu().numpy(), gpu.gram(x, y).cpu().numpy()) <= TOL_H


def test_gram_static_allocates_nothing_and_rejects_sizes_beyond_the_array(gpu):
    import torch
    x, y = blocks(256, 256, 2000, 8)
    out = torch.empty((256, 256), dtype=torch.complex128, device="cuda")
    gpu.gram_static(x, y, out=out)                                # first call: module load, attribute set-up
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        gpu.gram_static(x, y, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                  # the device's free memory did not move
    assert gpu.GRAM_STATIC_MAX_ENTRIES == 1048576
    xl, yl = blocks(1025, 1024, 8, 9)                             # 1025 * 1024 entries: one row too many
    with pytest.raises(gpu.PwhamError, match="exceeds the static scratch"):
        gpu.gram_static(xl, yl)
    assert relerr(gpu.gram_static(x, y, out=out).cpu().numpy(), gpu.gram(x, y).cpu().numpy()) <= TOL_H   # still usable

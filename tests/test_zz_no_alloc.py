"""gsr_distortion_static (include/gsr.h): the allocation-free variant of gsr_distortion — per-(state, tile) partials in
a file-scope device array of the library instead of a caller workspace — against the existing path, on two calls in a
row that share the array.  Collected last on purpose (the suite runs with pytest -x).  Tolerances: those of
tests/test_gpu_parity.py for the same quantities (MSE rtol 2e-4 / atol 1e-12, PSNR 1e-3 dB); the kernels and the
reduction tree are the same, so the values are also expected to be bitwise equal, which is checked too."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

DB_TOL = 1e-3


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def gsr(torch_mod):
    from paper_2606_17212_b200 import gsr as G
    G.lib()
    return G


def _batch(torch, seed, B, H, W):
    gen = torch.Generator(device="cuda").manual_seed(seed)
    ref = torch.rand((H, W, 3), generator=gen, device="cuda", dtype=torch.float32)
    noise = torch.randn((B, H, W, 3), generator=gen, device="cuda", dtype=torch.float32)
    scale = torch.linspace(0.0, 0.2, B, device="cuda").view(B, 1, 1, 1)          # state 0 equals the reference
    return (ref[None] + scale * noise).clamp(0.0, 1.0).contiguous(), ref


def _check(gsr, torch, imgs, ref):
    B = imgs.shape[0]
    want_mse, want_psnr = gsr.distortion(imgs, ref)                               # existing path: caller workspace
    mse = torch.full((B,), -1.0, dtype=torch.float64, device="cuda")
    psnr = torch.full((B,), -1.0, dtype=torch.float32, device="cuda")
    gsr.distortion_static(imgs, ref, mse, psnr)
    torch.cuda.synchronize()
    assert np.allclose(mse.cpu().numpy(), want_mse.cpu().numpy(), rtol=2e-4, atol=1e-12)
    assert np.max(np.abs(psnr.cpu().numpy() - want_psnr.cpu().numpy())) <= DB_TOL
    assert torch.equal(mse, want_mse) and torch.equal(psnr, want_psnr)           # same kernels, same tree
    return mse


def test_two_calls_in_a_row_match_the_workspace_path(gsr, torch_mod):
    """Call 1: 7 states of 150 x 100 (ragged tiles; 70 tiles each).  Call 2, straight after, on the same array: 3 states
    of 64 x 48 — fewer partials than call 1 left behind, so stale contents would show if they were read."""
    torch = torch_mod
    imgs, ref = _batch(torch, 1, 7, 100, 150)
    m1 = _check(gsr, torch, imgs, ref)
    assert float(m1[0]) == 0.0 and bool((m1[1:] > 0).all())
    imgs2, ref2 = _batch(torch, 2, 3, 48, 64)
    _check(gsr, torch, imgs2, ref2)
    # and the first batch once more: the array's contents from call 2 do not matter either
    m3 = _check(gsr, torch, imgs, ref)
    assert torch.equal(m1, m3)


def test_allocates_nothing_and_rejects_sizes_beyond_the_built_in_scratch(gsr, torch_mod):
    torch = torch_mod
    L = gsr.lib()
    imgs, ref = _batch(torch, 3, 4, 40, 56)
    mse = torch.empty(4, dtype=torch.float64, device="cuda")
    psnr = torch.empty(4, dtype=torch.float32, device="cuda")
    gsr.distortion_static(imgs, ref, mse, psnr)                                   # set-up for this device done
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        gsr.distortion_static(imgs, ref, mse, psnr)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                                         # no device memory taken by the calls
    # the limit: B * tiles <= 2^20; one more state than fits is refused before anything is launched or read
    cap = int(L.gsr_distortion_static_max_partials())
    assert cap == 1 << 20
    H = W = 16 * 64                                                               # 4096 tiles
    B_max = cap // 4096                                                           # 256 states fit exactly
    rc = L.gsr_distortion_static(imgs.data_ptr(), ref.data_ptr(), B_max + 1, H, W, mse.data_ptr(), psnr.data_ptr(), None)
    assert rc == -3                                                               # GSR_E_WORKSPACE_TOO_SMALL
    assert b"exceeds the built-in scratch" in L.gsr_last_error()
    # and a size that fits is still served afterwards
    gsr.distortion_static(imgs, ref, mse, psnr)
    torch.cuda.synchronize()
    assert bool((mse >= 0).all())

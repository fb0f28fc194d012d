"""GPU parity of the richer-distortion / risk-reduction calls (include/gsr.h) against
oracle/metrics.py through the C ABI.

Tolerances: SSIM is computed from fp32 pixels with DOUBLE window moments (fp32 moments left a
systematic 4e-5 on flat images: the variance terms E[x^2] - mu^2 cancel against C2 = 9e-4), in another
summation order than the oracle: 1e-9 is the bar.  The reductions over
states are exact selections plus double sums in a different order than the oracle's sorted sum: 1e-12
relative.  Flicker: fp32 differences of fp32 inputs are exact-rounded once; 1e-6 relative."""
import numpy as np
import pytest

from oracle import metrics as M
from paper_2606_17212_b200 import synth

pytestmark = pytest.mark.gpu

SSIM_TOL = 1e-9


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


def _dev(torch, a, dtype=np.float32):
    return torch.from_numpy(np.ascontiguousarray(a, dtype)).cuda()


@pytest.mark.parametrize("H,W,B", [(16, 16, 1), (37, 53, 3), (5, 7, 2), (64, 48, 2)])
def test_ssim_random_images(gsr, torch_mod, H, W, B):
    rng = np.random.default_rng(H * W + B)
    ref = rng.uniform(size=(H, W, 3)).astype(np.float32)
    imgs = np.clip(ref[None] + rng.normal(0, 0.08, (B, H, W, 3)), 0, 1).astype(np.float32)
    imgs[0] = ref                                                     # SSIM(x, x) = 1
    mse = ((imgs.astype(np.float64) - ref) ** 2).mean(axis=(1, 2, 3))
    want = M.ssim(imgs, ref)
    ssim, dmix = gsr.distortion_ssim(_dev(torch_mod, imgs), _dev(torch_mod, ref), mse=_dev(torch_mod, mse, np.float64))
    got = ssim.cpu().numpy()
    assert np.abs(got - want).max() <= SSIM_TOL, (got, want)
    assert abs(got[0] - 1.0) <= SSIM_TOL
    assert np.abs(dmix.cpu().numpy() - M.mixed_distortion(mse, want)).max() <= 0.2 * SSIM_TOL + 1e-15


def test_ssim_constant_images_closed_form(gsr, torch_mod):
    a, b = 0.3, 0.7
    H, W = 48, 40
    x, y = np.full((1, H, W, 3), a, np.float32), np.full((H, W, 3), b, np.float32)
    ssim, _ = gsr.distortion_ssim(_dev(torch_mod, x), _dev(torch_mod, y))
    assert abs(float(ssim[0]) - M.ssim(x, y)[0]) <= SSIM_TOL


def test_ssim_and_flicker_on_rendered_states(gsr, torch_mod, oracle_mod):
    """The real use: rendered partial states against the full-state render, at two times."""
    torch = torch_mod
    wl = synth.scaled_object_workload(9, C=5, per_cluster=250, W=72, H=56, fov=40.0, n_frames=2, B=6)
    scene = gsr.Scene(wl.scene)
    lv = wl.levels[0]
    dlv = torch.from_numpy(np.ascontiguousarray(lv)).cuda()
    full = torch.full((1, wl.scene.C), 3, dtype=torch.int8, device="cuda")
    outs, refs = [], []
    for cam, t in wl.frames:                                       # same camera class, two times
        cam0 = wl.frames[0][0]
        ws = scene.new_workspace(cam0, lv.shape[0])
        r, _, _ = scene.render_states(cam0, t, full, workspace=ws)
        o, _, _ = scene.render_states(cam0, t, dlv, workspace=ws)
        scene.status(ws)
        outs.append(o.contiguous())
        refs.append(r[0].contiguous())
    o_np, r_np = [o.cpu().numpy() for o in outs], [r.cpu().numpy() for r in refs]
    mse, _ = gsr.distortion(outs[0], refs[0])
    ssim, dmix = gsr.distortion_ssim(outs[0], refs[0], mse=mse)
    want = M.ssim(o_np[0], r_np[0])
    assert np.abs(ssim.cpu().numpy() - want).max() <= SSIM_TOL
    want_mix = M.mixed_distortion(mse.cpu().numpy(), want)
    assert np.abs(dmix.cpu().numpy() - want_mix).max() <= 0.2 * SSIM_TOL + 1e-12
    fl = gsr.flicker(outs[0], outs[1], refs[0], refs[1]).cpu().numpy()
    want_fl = M.flicker(o_np[0], o_np[1], r_np[0], r_np[1])
    assert np.allclose(fl, want_fl, rtol=1e-6, atol=1e-14)
    # a state equal to the reference at both times does not flicker
    z = gsr.flicker(refs[0][None].contiguous(), refs[1][None].contiguous(), refs[0], refs[1])
    assert float(z[0]) == 0.0


@pytest.mark.parametrize("n", [1, 2, 19, 20, 21, 257, 8197])
def test_risk_reduce(gsr, torch_mod, n):
    rng = np.random.default_rng(n)
    v = rng.normal(25, 4, n).round(2)                               # ties
    for alpha in (0.05, 0.10, 1.0):
        for upper in (False, True):
            want = M.risk_reduce(v, alpha, upper)
            got = gsr.risk_reduce(_dev(torch_mod, v, np.float64), alpha, upper)
            for f in ("mean", "cvar", "quantile"):
                assert got[f] == pytest.approx(want[f], rel=1e-12, abs=1e-12), (f, alpha, upper)
            assert got["worst"] == want["worst"] and got["count"] == n
    v32 = v.astype(np.float32)
    want = M.risk_reduce(v32.astype(np.float64), 0.10, False)        # the p10 PSNR use: float input
    got = gsr.risk_reduce(_dev(torch_mod, v32, np.float32), 0.10, False)
    assert got["quantile"] == pytest.approx(want["quantile"], rel=1e-12)
    assert got["cvar"] == pytest.approx(want["cvar"], rel=1e-12)


def test_risk_reduce_hand_worked_on_gpu(gsr, torch_mod):
    got = gsr.risk_reduce(_dev(torch_mod, [1, 2, 3, 4, 5, 6, 7, 8, 9, 10], np.float64), 0.25, True)
    assert (got["mean"], got["cvar"], got["quantile"], got["worst"]) == (5.5, 9.0, 7.75, 10.0)
    got = gsr.risk_reduce(_dev(torch_mod, [21.41, 25.17, 27.48, 27.70], np.float64), 0.10, False)
    assert got["cvar"] == 21.41 and got["quantile"] == pytest.approx(22.538, abs=1e-12)


def test_prefix_monotonicity(gsr, torch_mod):
    torch = torch_mod
    psnr = np.array([21.41, 25.17, 27.48, 27.70])
    prev, nxt = _dev(torch, [0, 1, 2], np.int32), _dev(torch, [1, 2, 3], np.int32)
    assert gsr.prefix_monotonicity(_dev(torch, -psnr, np.float64), prev, nxt) == (0.0, 0)
    m, v = gsr.prefix_monotonicity(_dev(torch, -psnr[[0, 2, 1, 3]], np.float64), prev, nxt)
    assert v == 1 and m == pytest.approx(2.31, abs=1e-12)
    rng = np.random.default_rng(0)
    d = rng.normal(size=500)
    a, b = rng.integers(0, 500, 3000).astype(np.int32), rng.integers(0, 500, 3000).astype(np.int32)
    wm, wv = M.prefix_monotonicity(d, a, b)
    gm, gv = gsr.prefix_monotonicity(_dev(torch, d, np.float64), _dev(torch, a, np.int32), _dev(torch, b, np.int32))
    assert gv == wv and gm == pytest.approx(wm, rel=1e-12)

"""GPU parity of gsr_distortion_backward (include/gsr.h) against oracle/metrics.py distortion_backward,
and the whole gradient chain objective -> images -> records -> scene parameters against central differences of the
GPU's own forward objective."""
import dataclasses

import numpy as np
import pytest

from oracle import metrics as M
from paper_2606_17212_b200 import synth

pytestmark = pytest.mark.gpu


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


def _images(seed, B, H, W):
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:H, 0:W]
    ref = np.stack([0.5 + 0.4 * np.sin(0.3 * xx + 0.2 * yy + k) for k in range(3)], -1).astype(np.float32)
    imgs = np.clip(ref[None] + 0.08 * rng.standard_normal((B, H, W, 3)), 0.0, 1.0).astype(np.float32)
    return imgs, ref


@pytest.mark.parametrize("H,W", [(37, 53), (16, 16), (4, 7), (64, 33)])
def test_against_the_oracle(gsr, torch_mod, H, W):
    """Sizes with ragged tiles, one exact tile, an image smaller than the window; weights incl. 0; lambda 0.2, 1, 0.
    Double moments on both sides, fp32 output: 2e-6 of the largest entry."""
    torch = torch_mod
    imgs, ref = _images(H * 100 + W, 3, H, W)
    w = np.array([0.7, 0.0, 1.9])
    di, dr, dw = torch.from_numpy(imgs).cuda(), torch.from_numpy(ref).cuda(), torch.from_numpy(w).cuda()
    for lam in (0.20, 1.0, 0.0):
        got = gsr.distortion_backward(di, dr, dw, lam).cpu().numpy().astype(np.float64)
        want = M.distortion_backward(imgs, ref, w, lam)
        assert np.abs(got - want).max() <= 2e-6 * np.abs(want).max(), (lam, np.abs(got - want).max(), np.abs(want).max())
        assert np.all(got[1] == 0.0)
    got = gsr.distortion_backward(di, dr, None, 0.20).cpu().numpy().astype(np.float64)
    want = M.distortion_backward(imgs, ref, np.ones(3), 0.20)
    assert np.abs(got - want).max() <= 2e-6 * np.abs(want).max()
    # at the reference itself the gradient vanishes
    z = gsr.distortion_backward(dr[None].contiguous(), dr, None, 0.20)
    assert float(z.abs().max()) <= 1e-9


def test_full_size_sampled_pixels_and_directional_derivative(gsr, torch_mod):
    """800 x 800, 8 states (the resolution bench.py times): (1) the directional derivative of the GPU's own forward
    D = MSE + 0.2 (1 - SSIM) (gsr_distortion / gsr_distortion_ssim, double sums) along a random direction equals
    <gradient, direction>; (2) a 64 x 64 crop far from the border is an image of its own for the 21 x 21 support of the
    gradient at its centre: the centre pixels against the oracle on the crop, rescaled by the pixel counts."""
    torch = torch_mod
    H = W = 800
    B = 8
    gen = torch.Generator(device="cuda").manual_seed(5)
    yy, xx = torch.meshgrid(torch.arange(H, device="cuda"), torch.arange(W, device="cuda"), indexing="ij")
    ref = torch.stack([0.5 + 0.4 * torch.sin(0.03 * xx + 0.02 * yy + k) for k in range(3)], -1).float().contiguous()
    imgs = (ref[None] + 0.05 * torch.randn((B, H, W, 3), generator=gen, device="cuda")).clamp(0, 1).float().contiguous()
    w = torch.full((B,), 1.0 / B, dtype=torch.float64, device="cuda")
    g = gsr.distortion_backward(imgs, ref, w, 0.20)

    def D(im):
        mse, _ = gsr.distortion(im, ref)
        _, dmix = gsr.distortion_ssim(im, ref, mse=mse)
        return float((w * dmix).sum())

    # along the gradient itself (plus noise): a random direction in 15 M dimensions gives a derivative that is a
    # cancelling sum, below the differences' own noise
    u = g / g.abs().max() + 0.1 * torch.randn(imgs.shape, generator=gen, device="cuda")
    h = 1e-3                                                   # fp32 images: the step must survive their rounding
    ip, im_ = (imgs + h * u).float(), (imgs - h * u).float()
    fd = D(ip) - D(im_)
    pred = float((g.double() * (ip.double() - im_.double())).sum())
    assert abs(fd - pred) <= 2e-4 * abs(pred) + 1e-12, (fd, pred)
    # (2)
    y0, x0 = 300, 420
    crop = imgs[2:3, y0:y0 + 64, x0:x0 + 64].cpu().numpy()
    want = M.distortion_backward(crop, ref[y0:y0 + 64, x0:x0 + 64].cpu().numpy(), np.ones(1), 0.20)[0]
    got = g[2, y0:y0 + 64, x0:x0 + 64].double().cpu().numpy() * B * (H * W) / (64 * 64)
    c = slice(22, 42)                                          # 10 + 10 pixels from the crop's border and more
    assert np.abs(got[c, c] - want[c, c]).max() <= 5e-6 * np.abs(want[c, c]).max()


def test_objective_to_parameters_against_differences_of_the_gpu_forward(gsr, torch_mod):
    """L = mean_b D_b, D = MSE + 0.2 (1 - SSIM) against the full-state render: gsr_distortion_backward ->
    gsr_render_backward -> gsr_project_backward, compared with (L(theta + h u) - L(theta - h u)) where L is evaluated
    by the FORWARD calls alone (render, gsr_distortion, gsr_distortion_ssim) on perturbed scenes.  The reference
    image is held fixed (it is a target, not a function of the parameters)."""
    torch = torch_mod
    wl = synth.scaled_object_workload(61, C=3, per_cluster=150.0, W=96, H=80, fov=40.0, n_frames=1, B=6)
    cam, t = wl.frames[0]
    scn = wl.scene
    lv = wl.levels[0].copy()
    lv[0] = 3
    dlv = torch.from_numpy(np.ascontiguousarray(lv, np.int8)).cuda()
    B = lv.shape[0]
    w = torch.full((B,), 1.0 / B, dtype=torch.float64, device="cuda")
    rng = np.random.default_rng(61)
    # the target: the full-state render of a scene with perturbed colours and positions (so that D > 0 at full state)
    tgt_scn = dataclasses.replace(scn, mean=(scn.mean + 0.01 * rng.standard_normal(scn.mean.shape)).astype(np.float32),
                                  sh_base=(scn.sh_base + 0.05 * rng.standard_normal(scn.sh_base.shape)).astype(np.float32))
    s0 = gsr.Scene(tgt_scn)
    full = torch.full((1, scn.C), 3, dtype=torch.int8, device="cuda")
    ref = s0.render_states(cam, t, full)[0][0].contiguous()
    s0.close()

    def objective(sc_np):
        s = gsr.Scene(sc_np)
        ws = s.new_workspace(cam, B)
        out, _, _ = s.render_states(cam, t, dlv, workspace=ws)
        mse, _ = gsr.distortion(out, ref)
        _, dmix = gsr.distortion_ssim(out, ref, mse=mse)
        return float((w * dmix).sum()), s, ws, out

    L0, scene, ws, out = objective(scn)
    gimg = gsr.distortion_backward(out, ref, w, 0.20)
    grec = scene.render_backward(ws, out, gimg)
    gp = scene.project_backward(cam, t, grec)
    gg = gp["gauss"].double().cpu().numpy()
    grads = {"mean": gg[:, 0:3], "log_scale": gg[:, 6:9], "quat": gg[:, 9:13], "opacity_logit": gg[:, 13],
             "sh_base": gp["sh_base"].double().cpu().numpy(), "sh_res": gp["sh_res"].double().cpu().numpy()}
    scene.close()
    for field, h in (("mean", 2e-3), ("log_scale", 1e-2), ("quat", 1e-2), ("opacity_logit", 2e-2), ("sh_base", 1e-2),
                     ("sh_res", 2e-2)):
        theta = np.asarray(getattr(scn, field), np.float32)
        u = rng.standard_normal(theta.shape)
        if field == "mean":
            # parallel to the image plane: a step along the viewing axis swaps the depth order of neighbouring
            # Gaussians (their depths are ~4e-3 apart), at which the composite jumps — the sort is a constant of the
            # differentiation, so that direction is not one along which differences test the gradient
            Rw = np.asarray(cam.R_wc, np.float64).reshape(3, 3)
            u = rng.standard_normal((scn.N, 1)) * Rw[0] + rng.standard_normal((scn.N, 1)) * Rw[1]
        tp = (theta.astype(np.float64) + h * u).astype(np.float32)
        tm = (theta.astype(np.float64) - h * u).astype(np.float32)
        Lp, s1, _, _ = objective(dataclasses.replace(scn, **{field: tp}))
        s1.close()
        Lm, s2, _, _ = objective(dataclasses.replace(scn, **{field: tm}))
        s2.close()
        delta = tp.astype(np.float64) - tm.astype(np.float64)
        pred = float((grads[field].reshape(theta.shape) * delta).sum())
        mag = float(np.abs(grads[field].reshape(theta.shape) * delta).sum())
        # the image is piecewise smooth in the parameters (tile rectangles, cut, cap, stop, depth order are discrete):
        # finite steps cross a few of those, hence a percent-level bar; a wrong chain is off by O(1)
        assert abs((Lp - Lm) - pred) <= 3e-2 * mag + 2e-2 * abs(pred), (field, Lp - Lm, pred, mag)


def test_argument_checks(gsr, torch_mod):
    """Workspace too small -> GSR_E_WORKSPACE_TOO_SMALL (not needed when lambda = 0); misaligned gradient rows of
    gsr_render_backward / gsr_project_backward -> GSR_E_INVALID_ARG."""
    torch = torch_mod
    imgs, ref = _images(9, 2, 20, 24)
    di, dr = torch.from_numpy(imgs).cuda(), torch.from_numpy(ref).cuda()
    small = torch.empty(64, dtype=torch.uint8, device="cuda")
    with pytest.raises(gsr.GsrError):
        gsr.distortion_backward(di, dr, None, 0.20, workspace=small)
    g = gsr.distortion_backward(di, dr, None, 0.0, workspace=small)            # the MSE term alone needs none
    assert np.allclose(g.cpu().numpy(), 2.0 * (imgs - ref[None]) / ref.size, rtol=1e-6, atol=1e-12)
    wl = synth.scaled_object_workload(29, C=2, per_cluster=40.0, W=64, H=48, fov=40.0, n_frames=1, B=2)
    cam, t = wl.frames[0]
    scene = gsr.Scene(wl.scene)
    ws = scene.new_workspace(cam, 2)
    lv = torch.from_numpy(np.ascontiguousarray(wl.levels[0])).cuda()
    out, _, _ = scene.render_states(cam, t, lv, workspace=ws)
    buf = torch.zeros(scene.num_records() * 12 + 1, dtype=torch.float32, device="cuda")
    off = buf[1:]                                                               # 4 bytes past a 16-byte boundary
    assert off.data_ptr() % 16 != 0
    C = gsr.C
    rc = gsr.lib().gsr_render_backward(scene.handle, ws.data_ptr(), out.data_ptr(), out.data_ptr(), 2, off.data_ptr(), None)
    assert rc == -1
    rc = gsr.lib().gsr_project_backward(scene.handle, C.byref(gsr.camera_struct(cam)), float(t), off.data_ptr(),
                                        buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), None)
    assert rc == -1
    scene.close()


def test_objective_weights_and_flicker_gradient_against_the_oracle(gsr, torch_mod):
    """gsr_objective_weights (double, exact selection: 1e-15) incl. ties at the CVaR threshold, n = 1, the paper's
    weights (1, 0.30 at alpha 0.05, lambda_m = 2.0); refused pair indices; gsr_flicker_backward (fp32 differences)."""
    torch = torch_mod
    rng = np.random.default_rng(21)
    for n, alpha in ((96, 0.05), (40, 0.05), (7, 0.2), (1, 0.05), (300, 0.5), (8197, 0.05)):
        d = rng.uniform(0.01, 0.2, n)
        if n >= 7:
            d[3] = d[5] = np.sort(d)[-max(1, int(np.ceil(alpha * n)))]           # ties exactly at the threshold
        prev = rng.integers(0, n, 16).astype(np.int32)
        nxt = rng.integers(0, n, 16).astype(np.int32)
        want = M.objective_weights(d, 1.0, 0.30, alpha, prev, nxt, 2.0)
        got = gsr.objective_weights(torch.from_numpy(d).cuda(), 1.0, 0.30, alpha, torch.from_numpy(prev).cuda(),
                                    torch.from_numpy(nxt).cuda(), 2.0).cpu().numpy()
        assert np.abs(got - want).max() <= 1e-15 * max(1.0, np.abs(want).max()), (n, alpha)
        assert abs(got.sum() - 1.30) <= 1e-12                                    # mean and CVaR weights sum to 1 each; M's cancel
    got = gsr.objective_weights(torch.from_numpy(np.array([0.3, 0.2])).cuda(), 1.0, 0.0, 0.05,
                                torch.tensor([0, 5], dtype=torch.int32, device="cuda"),
                                torch.tensor([1, 1], dtype=torch.int32, device="cuda"), 2.0).cpu().numpy()
    assert np.array_equal(got, [0.5, 0.5])                                        # no violation; the pair (5, 1) is refused
    with pytest.raises(gsr.GsrError):
        gsr.index_status()                                                       # the refusal is latched and reported
    a, b = rng.uniform(0, 1, (2, 3, 21, 17, 3)).astype(np.float32)
    r1, r2 = rng.uniform(0, 1, (2, 21, 17, 3)).astype(np.float32)
    wgt = np.array([0.3, 0.0, 1.7])
    g1, g2 = gsr.flicker_backward(*(torch.from_numpy(x).cuda() for x in (a, b, r1, r2)), torch.from_numpy(wgt).cuda())
    w1, w2 = M.flicker_backward(a, b, r1, r2, wgt)
    assert np.abs(g2.cpu().numpy() - w2).max() <= 2e-7 * np.abs(w2).max()
    assert torch.equal(g1, -g2)


def test_image_space_objective_of_eq2_end_to_end(gsr, torch_mod):
    """L = mean_b D_b + 0.30 CVaR_0.05(D) + 2.0 M(D), D = MSE + 0.20 (1 - SSIM) (Eq. (2) with the paper's weights,
    PAPER.md:68-72; lambda_r R has no image gradient, lambda_t F is a separate call): forward by gsr_distortion,
    gsr_distortion_ssim, gsr_risk_reduce, gsr_prefix_monotonicity; gradient by gsr_objective_weights ->
    gsr_distortion_backward -> gsr_render_backward -> gsr_project_backward; against central differences of the forward
    along the SH coefficients of both colour payloads."""
    torch = torch_mod
    wl = synth.scaled_object_workload(62, C=4, per_cluster=120.0, W=96, H=80, fov=40.0, n_frames=1, B=12)
    cam, t = wl.frames[0]
    scn = wl.scene
    lv = wl.levels[0].copy()
    dlv = torch.from_numpy(np.ascontiguousarray(lv, np.int8)).cuda()
    B = lv.shape[0]
    rng = np.random.default_rng(62)
    prev = torch.from_numpy(np.arange(0, B - 1, dtype=np.int32)).cuda()
    nxt = torch.from_numpy(np.arange(1, B, dtype=np.int32)).cuda()
    tgt = dataclasses.replace(scn, sh_base=(scn.sh_base + 0.05 * rng.standard_normal(scn.sh_base.shape)).astype(np.float32))
    s0 = gsr.Scene(tgt)
    ref = s0.render_states(cam, t, torch.full((1, scn.C), 3, dtype=torch.int8, device="cuda"))[0][0].contiguous()
    s0.close()

    def forward(sc_np):
        s = gsr.Scene(sc_np)
        ws = s.new_workspace(cam, B)
        out, _, _ = s.render_states(cam, t, dlv, workspace=ws)
        mse, _ = gsr.distortion(out, ref)
        _, D = gsr.distortion_ssim(out, ref, mse=mse)
        r = gsr.risk_reduce(D, 0.05, True)
        M_, viol = gsr.prefix_monotonicity(D, prev, nxt)
        return float(r["mean"]) + 0.30 * float(r["cvar"]) + 2.0 * M_, s, ws, out, D, viol

    L0, scene, ws, out, D, viol = forward(scn)
    assert viol >= 2                                           # the monotonicity term is active
    w = gsr.objective_weights(D, 1.0, 0.30, 0.05, prev, nxt, 2.0)
    gimg = gsr.distortion_backward(out, ref, w, 0.20)
    gp = scene.project_backward(cam, t, scene.render_backward(ws, out, gimg))
    grads = {"sh_base": gp["sh_base"].double().cpu().numpy(), "sh_res": gp["sh_res"].double().cpu().numpy()}
    scene.close()
    # colour coefficients: the image is exactly smooth in them (opacity and scale also move the cut q <= tau and the
    # footprint, which are constants of the differentiation: reading K1)
    for field, h in (("sh_base", 5e-3), ("sh_res", 1e-2)):
        theta = np.asarray(getattr(scn, field), np.float32)
        u = rng.standard_normal(theta.shape)
        tp = (theta.astype(np.float64) + h * u).astype(np.float32)
        tm = (theta.astype(np.float64) - h * u).astype(np.float32)
        Lp, s1, _, _, _, vp = forward(dataclasses.replace(scn, **{field: tp}))
        s1.close()
        Lm, s2, _, _, _, vm = forward(dataclasses.replace(scn, **{field: tm}))
        s2.close()
        assert vp == viol and vm == viol                       # no pair changed sides: L is smooth along the step
        delta = tp.astype(np.float64) - tm.astype(np.float64)
        pred = float((grads[field].reshape(theta.shape) * delta).sum())
        mag = float(np.abs(grads[field].reshape(theta.shape) * delta).sum())
        assert abs((Lp - Lm) - pred) <= 3e-2 * mag + 2e-2 * abs(pred), (field, Lp - Lm, pred, mag)


def test_degenerate_sizes_of_the_backward_calls(gsr, torch_mod):
    """Empty batches and a one-pixel image through the calls added for the backward: nothing launched or all-zero
    results, never an error from the device."""
    torch = torch_mod
    L, C = gsr.lib(), gsr.C
    ref = torch.rand((5, 7, 3), device="cuda")
    e = torch.empty((0, 5, 7, 3), device="cuda")
    assert gsr.distortion_backward(e, ref, None, 0.20).shape == (0, 5, 7, 3)
    assert gsr.objective_weights(torch.empty(0, dtype=torch.float64, device="cuda")).numel() == 0
    one = torch.rand((2, 1, 1, 3), device="cuda")
    r1 = torch.rand((1, 1, 3), device="cuda")
    g = gsr.distortion_backward(one, r1, None, 0.20)
    want = M.distortion_backward(one.cpu().numpy(), r1.cpu().numpy(), np.ones(2), 0.20)
    assert np.abs(g.cpu().numpy() - want).max() <= 2e-6 * np.abs(want).max()
    # a batch of zero states through render_backward: the gradient is defined (all zero)
    wl = synth.scaled_object_workload(29, C=2, per_cluster=30.0, W=48, H=32, fov=40.0, n_frames=1, B=2)
    cam, t = wl.frames[0]
    scene = gsr.Scene(wl.scene)
    ws = scene.new_workspace(cam, 0)
    lv = torch.empty((0, wl.scene.C), dtype=torch.int8, device="cuda")
    out, _, _ = scene.render_states(cam, t, lv, workspace=ws)
    assert out.shape[0] == 0
    grad = scene.render_backward(ws, out, out)
    assert float(grad.abs().max()) == 0.0
    gp = scene.project_backward(cam, t, grad)
    assert float(gp["gauss"].abs().max()) == 0.0 and float(gp["cluster"].abs().max()) == 0.0
    gp = scene.project_backward_full(cam, t, grad)
    assert float(gp["gauss"].abs().max()) == 0.0 and float(gp["delta"].abs().max()) == 0.0
    scene.close()
    torch.cuda.synchronize()

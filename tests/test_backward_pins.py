"""Pins of the backward oracle (oracle/gsr_oracle.c O-8: gradients of a linear functional of one state's image with
respect to the 2-D quantities of its Gaussians).  CPU-only.  Pinned against what does not share its formulas:
central finite differences of the FORWARD oracle on perturbed projection records, the single-Gaussian closed form
evaluated with numpy, and the exact zeros the fixed decisions (cap, stop, cut) imply."""
import numpy as np
import pytest

from tests.helpers import axis_camera, tiny_scene

FIELDS = ["rgb0", "rgb1", "rgb2", "opacity", "qa", "qb", "qc", "mx", "my"]


def _get(p, i, k):
    return p["rgb"][i][k] if k < 3 else p[FIELDS[k]][i]


def _set(p, i, k, v):
    if k < 3:
        p["rgb"][i][k] = v
    else:
        p[FIELDS[k]][i] = v


def smooth_scene():
    """Three large, strongly overlapping Gaussians that cover the whole 64x64 image inside their q <= tau region
    (sigma' >= 16 px, opacity >= 0.8: cut radius > 3.2 sigma' > the image diagonal from the centre), never reach the
    cap (alpha <= opacity < 0.99) nor the stop (T >= 0.1^3): the image is a smooth function of every record field."""
    f, z0 = 100.0, 4.0
    means = [[0.05, -0.03, -0.3], [-0.1, 0.08, 0.0], [0.02, 0.12, 0.4]]
    scales = [[0.7, 0.9, 0.5], [1.0, 0.75, 0.6], [0.8, 0.8, 0.9]]
    quats = [[1, 0.2, -0.1, 0.3], [0.9, -0.3, 0.2, 0.1], [1, 0, 0.4, -0.2]]
    logits = [1.5, 2.0, 1.8]                                   # o = 0.82, 0.88, 0.86
    cols = [(0.9, 0.2, 0.3), (0.1, 0.8, 0.4), (0.3, 0.3, 0.9)]
    scn, _ = tiny_scene(means, scales, quats=quats, logits=logits, colors=cols, background=(0.2, 0.1, 0.05))
    return scn, axis_camera(64, 64, f, z0)


def test_b1_gradients_match_central_differences_of_the_forward_oracle(oracle_mod):
    scn, cam = smooth_scene()
    sc = oracle_mod.OracleScene(scn)
    depth = np.zeros(1, np.int8)
    p0 = sc.project(cam, 0.0, depth)
    assert p0["valid"].tolist() == [1, 1, 1]
    rng = np.random.default_rng(5)
    g = rng.standard_normal((cam.H, cam.W, 3))                # L = sum(g * image): dL/dimage = g
    grad = sc.backward(cam, 0.0, depth, g, proj=p0)
    L = lambda p: float((g * sc.render(cam, 0.0, depth, brute_force=True, proj=p)[0]).sum())
    # every pixel evaluates all three Gaussians (the premise of smoothness): E = 3 W H
    assert sc.render(cam, 0.0, depth, brute_force=True, proj=p0)[1][1] == 3 * cam.W * cam.H
    steps = {"rgb": 1e-3, "opacity": 1e-3, "qa": 2e-6, "qb": 2e-6, "qc": 2e-6, "mx": 2e-2, "my": 2e-2}
    worst = 0.0
    for i in range(3):
        for k in range(9):
            h = steps["rgb" if k < 3 else FIELDS[k]]
            pp, pm = p0.copy(), p0.copy()
            v = float(_get(p0, i, k))
            _set(pp, i, k, v + h)
            _set(pm, i, k, v - h)
            # the perturbed value as the record stores it (fp32 fields): use the step actually taken
            hh = float(_get(pp, i, k)) - float(_get(pm, i, k))
            fd = (L(pp) - L(pm)) / hh
            scale = max(abs(fd), abs(grad[i, k]), 1e-9)
            worst = max(worst, abs(fd - grad[i, k]) / scale)
            # the forward oracle evaluates q in fp32: its noise in L (~1e-6) over the step bounds the agreement;
            # a dropped term, a sign or a factor would be an O(1) relative error
            assert abs(fd - grad[i, k]) <= 1e-3 * scale + 2e-5, (i, FIELDS[k], fd, grad[i, k])
    assert worst < 5e-3


def test_b2_single_gaussian_closed_form(oracle_mod):
    """One isotropic Gaussian on the axis over a background: pixel = a c + (1 - a) bg with a = o exp(-q),
    q = r^2 / (2 sigma'^2) — every gradient is a plain sum over pixels, written here with numpy."""
    f, z0, s, logit = 100.0, 4.0, 0.8, 1.2
    col, bg = np.array([0.8, 0.3, 0.6]), np.array([0.1, 0.2, 0.4])
    scn, _ = tiny_scene([[0, 0, 0]], s, logits=logit, colors=col, background=bg)
    cam = axis_camera(64, 64, f, z0)
    sc = oracle_mod.OracleScene(scn)
    depth = np.zeros(1, np.int8)
    p = sc.project(cam, 0.0, depth)
    rng = np.random.default_rng(8)
    g = rng.standard_normal((cam.H, cam.W, 3))
    grad = sc.backward(cam, 0.0, depth, g, proj=p)[0]
    o = float(p["opacity"][0])
    A, B, Cq = float(p["qa"][0]), float(p["qb"][0]), float(p["qc"][0])
    ys, xs = np.mgrid[0:cam.H, 0:cam.W]
    dx, dy = float(p["mx"][0]) - (xs + 0.5), float(p["my"][0]) - (ys + 0.5)
    q = (A * dx + B * dy) * dx + Cq * dy * dy
    assert q.max() < float(p["tau"][0])                                  # the whole image passes the cut
    e = np.exp(-q)
    a = o * e
    gc = (g * (np.asarray(p["rgb"][0]) - bg)).sum(-1)                    # g . (c - bg): dpixel/da
    expect = np.concatenate([(a[..., None] * g).sum((0, 1)), [(e * gc).sum()],
                             [(-a * gc * dx * dx).sum(), (-a * gc * dx * dy).sum(), (-a * gc * dy * dy).sum()],
                             [(-a * gc * (2 * A * dx + B * dy)).sum(), (-a * gc * (B * dx + 2 * Cq * dy)).sum()]])
    assert np.allclose(grad, expect, rtol=1e-6, atol=1e-9)


def test_b3_cap_stop_and_absent_gaussians_have_exactly_the_zeros_the_decisions_imply(oracle_mod):
    f, z0 = 100.0, 4.0
    cam = axis_camera(32, 32, f, z0, cx=16.5, cy=16.5)
    g = np.ones((cam.H, cam.W, 3))
    # (a) alpha capped over the whole image (logit +12, sigma' = 500 px: o exp(-q) >= 0.998 at the corners): colour
    #     gradient 0.99 per pixel, no gradient to opacity, conic or mean
    scn, _ = tiny_scene([[0, 0, 0]], 20.0, logits=12.0, colors=(0.5, 0.5, 0.5))
    sc = oracle_mod.OracleScene(scn)
    gr = sc.backward(cam, 0.0, np.zeros(1, np.int8), g)[0]
    assert np.allclose(gr[:3], 0.99 * cam.W * cam.H, rtol=1e-12) and np.all(gr[3:] == 0.0)
    # (b) a stack of identical wide Gaussians, alpha = 0.5 each: 13 are accepted, the 14th triggers the stop
    #     (2^-14 < 1e-4): Gaussians 14.. get exactly zero gradient, the first 13 do not
    n = 20
    scn, order = tiny_scene([[0, 0, 0.01 * k] for k in range(n)], 5.0, logits=0.0, colors=(0.7, 0.7, 0.7))
    sc = oracle_mod.OracleScene(scn)
    gr = sc.backward(cam, 0.0, np.zeros(1, np.int8), g)
    p = sc.project(cam, 0.0, np.zeros(1, np.int8))
    by_depth = np.argsort(p["z"], kind="stable")
    assert np.all(gr[by_depth[:13], :3] > 0) and np.all(gr[by_depth[13:]] == 0.0)
    # colour gradient of the k-th accepted Gaussian = sum over pixels of alpha T = ~0.5^(k+1) per pixel
    assert np.allclose(gr[by_depth[0], 0] / (cam.W * cam.H), 0.5, rtol=2e-2)
    assert np.allclose(gr[by_depth[3], 0] / gr[by_depth[2], 0], 0.5, rtol=2e-2)
    # (c) a Gaussian absent from the state (level 1 at depth 0) gets no gradient
    scn, _ = tiny_scene([[0, 0, 0], [0.1, 0, 0.2]], 0.5, logits=1.0, levels=[0, 1])
    sc = oracle_mod.OracleScene(scn)
    gr = sc.backward(cam, 0.0, np.zeros(1, np.int8), g)
    assert np.all(gr[1] == 0.0) and np.any(gr[0] != 0.0)


def test_b4_linearity_in_the_image_gradient_and_mse_chain(oracle_mod):
    """grad is linear in g; and with g = 2 (I - R) / (3 W H) it is the gradient of the MSE against R: checked by a
    finite difference of the oracle's own distortion on one colour field."""
    scn, cam = smooth_scene()
    sc = oracle_mod.OracleScene(scn)
    depth = np.zeros(1, np.int8)
    p0 = sc.project(cam, 0.0, depth)
    rng = np.random.default_rng(2)
    g1, g2 = rng.standard_normal((2, cam.H, cam.W, 3))
    a, b = sc.backward(cam, 0.0, depth, g1, proj=p0), sc.backward(cam, 0.0, depth, g2, proj=p0)
    c = sc.backward(cam, 0.0, depth, 2.0 * g1 - 3.0 * g2, proj=p0)
    assert np.allclose(c, 2.0 * a - 3.0 * b, rtol=1e-10, atol=1e-12)
    # the magnitude the GPU parity bar uses dominates the gradient entry by entry and does not depend on signs
    a2, mag = sc.backward(cam, 0.0, depth, g1, proj=p0, want_abs=True)
    assert np.array_equal(a2, a) and np.all(mag >= np.abs(a))
    assert np.allclose(sc.backward(cam, 0.0, depth, -g1, proj=p0, want_abs=True)[1], mag, rtol=1e-12)
    R = rng.uniform(0, 1, (cam.H, cam.W, 3))
    img = sc.render(cam, 0.0, depth, brute_force=True, proj=p0)[0]
    grad = sc.backward(cam, 0.0, depth, 2.0 * (img - R) / img.size, proj=p0)
    mse = lambda p: float(oracle_mod.distortion(sc.render(cam, 0.0, depth, brute_force=True, proj=p)[0][None], R)[0][0])
    pp, pm = p0.copy(), p0.copy()
    pp["opacity"][1] += 1e-3
    pm["opacity"][1] -= 1e-3
    fd = (mse(pp) - mse(pm)) / (float(pp["opacity"][1]) - float(pm["opacity"][1]))
    assert abs(fd - grad[1, 3]) <= 1e-4 * abs(fd)

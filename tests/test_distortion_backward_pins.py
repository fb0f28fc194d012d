"""Pins of the distortion-gradient oracle (oracle/metrics.py distortion_backward: d/d(image) of
sum_b weight_b (MSE_b + lambda (1 - SSIM_b))).  CPU-only.  Against central differences of the forward
oracle of D itself (double: agreement to ~1e-7), the exact zero at image = reference, and the MSE-only closed form."""
import numpy as np

from oracle import metrics as M


def _images(seed, B=2, H=23, W=19):
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:H, 0:W]
    ref = np.stack([0.5 + 0.4 * np.sin(0.3 * xx + 0.2 * yy + k) for k in range(3)], -1)
    imgs = np.clip(ref[None] + 0.08 * rng.standard_normal((B, H, W, 3)), 0.0, 1.0)
    return imgs, ref


def _D(imgs, ref, weight, lam):
    mse = ((imgs - ref[None]) ** 2).reshape(imgs.shape[0], -1).mean(1)
    return float((weight * (mse + lam * (1.0 - M.ssim(imgs, ref)))).sum())


def test_d1_central_differences_of_the_forward_oracle():
    imgs, ref = _images(1)
    weight = np.array([0.7, 1.9])
    for lam in (0.20, 1.0, 0.0):
        g = M.distortion_backward(imgs, ref, weight, lam)
        rng = np.random.default_rng(2)
        # single pixels: corners and edges (zero padding), interior, every channel
        H, W = ref.shape[:2]
        picks = [(0, 0, 0, 0), (1, H - 1, W - 1, 2), (0, 0, W // 2, 1), (1, H // 2, 0, 0), (0, H // 2, W // 2, 2),
                 (1, 3, 4, 1), (0, H - 2, 1, 0)]
        h = 1e-5
        for (b, yy, xx, ch) in picks:
            ip, im = imgs.copy(), imgs.copy()
            ip[b, yy, xx, ch] += h
            im[b, yy, xx, ch] -= h
            fd = (_D(ip, ref, weight, lam) - _D(im, ref, weight, lam)) / (2 * h)
            assert abs(fd - g[b, yy, xx, ch]) <= 1e-6 * abs(g[b, yy, xx, ch]) + 1e-10, (lam, b, yy, xx, ch, fd, g[b, yy, xx, ch])
        # random directions
        for _ in range(3):
            u = rng.standard_normal(imgs.shape)
            fd = (_D(imgs + h * u, ref, weight, lam) - _D(imgs - h * u, ref, weight, lam)) / (2 * h)
            assert abs(fd - float((g * u).sum())) <= 1e-6 * float(np.abs(g * u).sum())


def test_d2_zero_at_the_reference_and_mse_only_closed_form():
    imgs, ref = _images(3, B=1)
    # image = reference: MSE and 1 - SSIM are both at their minimum 0
    g = M.distortion_backward(ref[None], ref, np.ones(1), 0.20)
    assert np.abs(g).max() <= 1e-15
    # lambda = 0: 2 (x - y) / (3 H W) times the weight
    g = M.distortion_backward(imgs, ref, np.array([2.5]), 0.0)
    assert np.allclose(g[0], 2.5 * 2.0 * (imgs[0] - ref) / ref.size, rtol=1e-15, atol=0.0)
    # the SSIM part alone pulls the image towards the reference: moving along -g lowers D
    g = M.distortion_backward(imgs, ref, np.ones(1), 1.0)
    assert _D(imgs - 1e-2 * g / np.abs(g).max(), ref, np.ones(1), 1.0) < _D(imgs, ref, np.ones(1), 1.0)


def test_d3_weights_and_linearity():
    imgs, ref = _images(4, B=3)
    g1 = M.distortion_backward(imgs, ref, np.array([1.0, 0.0, 0.0]))
    g2 = M.distortion_backward(imgs, ref, np.array([0.0, 2.0, 0.0]))
    g = M.distortion_backward(imgs, ref, np.array([1.0, 2.0, 0.0]))
    assert np.array_equal(g[2], np.zeros_like(g[2]))
    assert np.allclose(g, g1 + g2, rtol=1e-15, atol=0.0)
    # smaller than the 11 x 11 window: zero padding everywhere, still consistent with differences
    imgs, ref = _images(5, B=1, H=4, W=7)
    g = M.distortion_backward(imgs, ref, np.ones(1))
    h = 1e-5
    ip, im = imgs.copy(), imgs.copy()
    ip[0, 2, 3, 1] += h
    im[0, 2, 3, 1] -= h
    fd = (_D(ip, ref, np.ones(1), 0.20) - _D(im, ref, np.ones(1), 0.20)) / (2 * h)
    assert abs(fd - g[0, 2, 3, 1]) <= 1e-6 * abs(fd) + 1e-10

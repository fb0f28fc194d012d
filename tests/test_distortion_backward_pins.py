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


def _L(d, w_mean, w_cvar, alpha, prev, nxt, w_mono):
    r = M.risk_reduce(d, alpha, upper_tail=True)
    return w_mean * r["mean"] + w_cvar * r["cvar"] + w_mono * M.prefix_monotonicity(d, prev, nxt)[0]


def test_d4_objective_weights_are_the_differences_of_the_forward_reductions():
    """L(D) = w_mean mean + w_cvar CVaR_0.05 + w_mono M is piecewise linear in D: away from ties and from
    D[next] = D[prev] a small step in one coordinate changes L by exactly weight * step."""
    rng = np.random.default_rng(11)
    for n, alpha in ((40, 0.05), (96, 0.05), (7, 0.2), (1, 0.05), (23, 0.5)):
        d = rng.uniform(0.01, 0.2, n)
        prev = rng.integers(0, n, 12)
        nxt = rng.integers(0, n, 12)
        w = M.objective_weights(d, 1.0, 0.30, alpha, prev, nxt, 2.0)
        h = 1e-7
        for i in range(n):
            dp, dm = d.copy(), d.copy()
            dp[i] += h
            dm[i] -= h
            fd = (_L(dp, 1.0, 0.30, alpha, prev, nxt, 2.0) - _L(dm, 1.0, 0.30, alpha, prev, nxt, 2.0)) / (2 * h)
            assert abs(fd - w[i]) <= 1e-6 * max(1.0, abs(w[i])), (n, alpha, i, fd, w[i])
    # hand values: n = 4, alpha = 0.5 -> k = 2: the two largest get 1/2 each; mean 1/4 each
    w = M.objective_weights([0.1, 0.4, 0.2, 0.3], 1.0, 1.0, 0.5)
    assert np.allclose(w, [0.25, 0.75, 0.25, 0.75], rtol=0, atol=1e-15)
    # ties at the threshold share what is left: values (3, 2, 2, 2, 1), k = 2: one above, one slot for three ties
    w = M.objective_weights([3.0, 2.0, 2.0, 2.0, 1.0], 0.0, 1.0, 0.4)
    assert np.allclose(w, [0.5, 1 / 6, 1 / 6, 1 / 6, 0.0], rtol=0, atol=1e-15) and abs(w.sum() - 1.0) < 1e-15
    # monotonicity: only violated pairs (D[next] > D[prev]) count
    w = M.objective_weights([0.3, 0.2, 0.25], 0.0, 0.0, 0.05, [0, 1], [1, 2], 2.0)
    assert np.array_equal(w, [0.0, -2.0, 2.0])


def test_d5_flicker_gradient_against_differences():
    rng = np.random.default_rng(12)
    a, b = rng.uniform(0, 1, (2, 2, 9, 7, 3))
    r1, r2 = rng.uniform(0, 1, (2, 9, 7, 3))
    wgt = np.array([0.3, 1.7])
    g1, g2 = M.flicker_backward(a, b, r1, r2, wgt)
    F = lambda a_, b_: float((wgt * M.flicker(a_, b_, r1, r2)).sum())
    h = 1e-6
    for (s_, y, x, c) in ((0, 0, 0, 0), (1, 8, 6, 2), (1, 4, 3, 1)):
        for arr, g, which in ((a, g1, 0), (b, g2, 1)):
            p, m = arr.copy(), arr.copy()
            p[s_, y, x, c] += h
            m[s_, y, x, c] -= h
            fd = (F(p, b) - F(m, b)) / (2 * h) if which == 0 else (F(a, p) - F(a, m)) / (2 * h)
            assert abs(fd - g[s_, y, x, c]) <= 1e-7 * abs(g[s_, y, x, c]) + 1e-12
    assert np.array_equal(g1, -g2)

"""Pins of oracle/metrics.py (SSIM, mixed distortion, CVaR / quantile reductions, flicker, prefix
monotonicity) against closed forms, a library route (scipy.ndimage), hand-worked numbers and the
paper's printed prefix points.  CPU-only."""
from pathlib import Path

import numpy as np
import pytest

from oracle import metrics as M

GOLD = Path(__file__).resolve().parent / "golden"


# ------------------------------------------------------------------------------------------ SSIM
def test_window_is_normalised_symmetric_and_has_the_textbook_ratio():
    g = M.gaussian_window()
    assert g.shape == (11,) and abs(g.sum() - 1.0) < 1e-15
    assert np.allclose(g, g[::-1], rtol=0, atol=0)
    # neighbour ratio of a sigma = 1.5 Gaussian at the centre: exp(-1/(2*2.25))
    assert abs(g[6] / g[5] - np.exp(-1.0 / 4.5)) < 1e-15


def test_ssim_of_an_image_with_itself_is_one():
    rng = np.random.default_rng(0)
    x = rng.uniform(size=(40, 37, 3))
    m = M.ssim_map(x, x)
    assert np.allclose(m, 1.0, rtol=0, atol=1e-12)
    assert abs(M.ssim(x[None], x)[0] - 1.0) < 1e-12


def test_ssim_constant_images_closed_form_in_the_interior():
    """x = a, y = b everywhere: away from the zero-padded border the window sees constants, variances and
    covariance vanish and ssim = (2ab + C1)/(a^2 + b^2 + C1) (the contrast/structure factor is C2/C2 = 1)."""
    a, b = 0.3, 0.7
    x, y = np.full((32, 30, 3), a), np.full((32, 30, 3), b)
    m = M.ssim_map(x, y)
    want = (2 * a * b + M.SSIM_C1) / (a * a + b * b + M.SSIM_C1)
    assert np.allclose(m[5:-5, 5:-5], want, rtol=0, atol=1e-12)
    # at the corner the zero padding lowers both means by the same factor: still a closed form
    g = M.gaussian_window()
    f = g[5:].sum() ** 2                          # weight mass inside the image at pixel (0, 0)
    mx, my = a * f, b * f
    sxx, syy, sxy = a * a * f - mx * mx, b * b * f - my * my, a * b * f - mx * my
    corner = ((2 * mx * my + M.SSIM_C1) * (2 * sxy + M.SSIM_C2)) / ((mx * mx + my * my + M.SSIM_C1) * (sxx + syy + M.SSIM_C2))
    assert abs(m[0, 0, 0] - corner) < 1e-12


def test_ssim_against_scipy_gaussian_filter():
    """Independent library route: scipy.ndimage.gaussian_filter(sigma=1.5, truncate -> radius 5, mode constant)."""
    ndi = pytest.importorskip("scipy.ndimage")
    rng = np.random.default_rng(1)
    x = rng.uniform(size=(45, 52, 3))
    y = np.clip(x + rng.normal(0, 0.1, x.shape), 0, 1)
    blur = lambda p: ndi.gaussian_filter(p, sigma=1.5, truncate=5.0 / 1.5 + 1e-9, mode="constant", cval=0.0)
    out = np.zeros_like(x)
    for ch in range(3):
        mx, my = blur(x[..., ch]), blur(y[..., ch])
        sxx, syy = blur(x[..., ch] ** 2) - mx ** 2, blur(y[..., ch] ** 2) - my ** 2
        sxy = blur(x[..., ch] * y[..., ch]) - mx * my
        out[..., ch] = ((2 * mx * my + 1e-4) * (2 * sxy + 9e-4)) / ((mx ** 2 + my ** 2 + 1e-4) * (sxx + syy + 9e-4))
    assert np.allclose(M.ssim_map(x, y), out, rtol=0, atol=1e-12)


def test_ssim_is_symmetric_and_drops_with_noise():
    rng = np.random.default_rng(2)
    x = rng.uniform(size=(33, 33, 3))
    y1 = np.clip(x + rng.normal(0, 0.02, x.shape), 0, 1)
    y2 = np.clip(x + rng.normal(0, 0.2, x.shape), 0, 1)
    assert abs(M.ssim(x[None], y1)[0] - M.ssim(y1[None], x)[0]) < 1e-14
    assert 1.0 > M.ssim(y1[None], x)[0] > M.ssim(y2[None], x)[0]


def test_mixed_distortion_weights():
    """D = MSE + 0.20 (1 - SSIM)."""
    assert M.mixed_distortion(np.array([0.01]), np.array([0.9]))[0] == pytest.approx(0.01 + 0.2 * 0.1, abs=1e-15)
    assert M.mixed_distortion(np.array([0.0]), np.array([1.0]))[0] == 0.0


# ------------------------------------------------------------------------------------------ risk reductions
def test_risk_reduce_hand_worked():
    for line in (GOLD / "risk_hand.txt").read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        head, vals, want = [p.split() for p in line.split("|")]
        r = M.risk_reduce([float(v) for v in vals], float(head[0]), head[1] == "U")
        got = [r["mean"], r["cvar"], r["quantile"], r["worst"]]
        assert np.allclose(got, [float(w) for w in want], rtol=0, atol=1e-12), line
        assert r["count"] == len(vals)


def test_risk_reduce_against_numpy():
    rng = np.random.default_rng(7)
    for n in (1, 2, 19, 20, 21, 257):
        v = rng.normal(size=n)
        for alpha in (0.05, 0.1, 0.5, 1.0):
            lo, up = M.risk_reduce(v, alpha, False), M.risk_reduce(v, alpha, True)
            k = min(n, max(1, int(np.ceil(alpha * n))))
            s = np.sort(v)
            assert lo["cvar"] == pytest.approx(s[:k].mean(), abs=1e-13)
            assert up["cvar"] == pytest.approx(s[-k:].mean(), abs=1e-13)
            assert lo["quantile"] == pytest.approx(np.quantile(v, alpha, method="linear"), abs=1e-13)
            assert up["quantile"] == pytest.approx(np.quantile(v, 1 - alpha, method="linear"), abs=1e-13)
            assert lo["worst"] == s[0] and up["worst"] == s[-1]
            assert lo["mean"] == pytest.approx(v.mean(), abs=1e-13)
            # the upper tail of v is the lower tail of -v
            neg = M.risk_reduce(-v, alpha, False)
            assert up["cvar"] == pytest.approx(-neg["cvar"], abs=1e-13)
            assert up["quantile"] == pytest.approx(-neg["quantile"], abs=1e-13)


# ------------------------------------------------------------------------------------------ flicker / monotonicity
def test_flicker_closed_forms():
    rng = np.random.default_rng(3)
    r1, r2 = rng.uniform(size=(9, 11, 3)), rng.uniform(size=(9, 11, 3))
    a = rng.uniform(size=(2, 9, 11, 3))
    # a state that changes exactly like the reference has no flicker; a constant extra drift eps gives eps^2
    b = a + (r2 - r1)[None]
    assert np.allclose(M.flicker(a, b, r1, r2), 0.0, atol=1e-30)
    eps = 0.125
    assert np.allclose(M.flicker(a, b + eps, r1, r2), eps * eps, rtol=0, atol=1e-15)
    # a static reference: flicker is the MSE between the two renders
    assert np.allclose(M.flicker(a, b, r1, r1), ((b - a) ** 2).mean(axis=(1, 2, 3)), rtol=0, atol=1e-15)


def test_prefix_monotonicity_on_the_papers_prefix_points():
    """"four monotonic prefix points (21.41, 25.17, 27.48, and 27.70 dB) ... with 0 PSNR
    regressions".  With D = -PSNR a growing prefix never regresses: M = 0, 0 violations."""
    psnr = np.array([21.41, 25.17, 27.48, 27.70])
    m, v = M.prefix_monotonicity(-psnr, [0, 1, 2], [1, 2, 3])
    assert m == 0.0 and v == 0
    # swap two points: one regression of 27.48 - 25.17 = 2.31 dB
    psnr2 = np.array([21.41, 27.48, 25.17, 27.70])
    m, v = M.prefix_monotonicity(-psnr2, [0, 1, 2], [1, 2, 3])
    assert v == 1 and m == pytest.approx(2.31, abs=1e-12)

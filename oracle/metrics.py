"""CPU ORACLE for the richer distortion and the risk reductions.

TEST INFRASTRUCTURE ONLY (same rules as oracle/oracle.py).  Plain numpy in float64, written in the order
of the definitions; no product code is imported.

What it follows (PAPER.md = /root/reference/PAPER.md; DESIGN.md §12 = the written spec of this row):

  SSIM .............. PAPER.md:72 "D = MSE + 0.20(1 - SSIM)".  The paper does not print its SSIM; reading G1 is
                      the splatting-toolchain convention: per channel, 11x11 Gaussian window (sigma 1.5,
                      weights normalised to sum 1, separable), zero padding of 5 pixels, colour range 1,
                      C1 = 0.01^2, C2 = 0.03^2;
                          mu_x = w*x, mu_y = w*y, s_xx = w*(x x) - mu_x^2, s_yy = w*(y y) - mu_y^2, s_xy = w*(x y) - mu_x mu_y
                          ssim = ((2 mu_x mu_y + C1)(2 s_xy + C2)) / ((mu_x^2 + mu_y^2 + C1)(s_xx + s_yy + C2))
                      and SSIM = mean of the map over all H x W x 3 values.
  mixed distortion .. D = MSE + 0.20 (1 - SSIM)
  risk reductions ... PAPER.md:68 "CVaR_0.05(D)", "held-out partial-state p10 PSNR"
                      "worst-10% PSNR".  Reading G2 for n values v and tail fraction a: k = max(1, ceil(a n));
                      CVaR = mean of the k WORST values (largest for a distortion = upper tail, smallest for
                      a PSNR = lower tail); quantile = linear interpolation at position a(n-1) of the ascending
                      order (lower tail) or (1-a)(n-1) (upper tail); worst = the extreme value; mean = plain mean.
  flicker ........... PAPER.md:70 "F penalizes temporal-change error".  Reading G3 for two times t1 < t2:
                          F_b = mean over pixels and channels of ((out_b(t2) - out_b(t1)) - (ref(t2) - ref(t1)))^2
  monotonicity ...... PAPER.md:70 "M penalizes quality regressions as a prefix grows".  Reading G4 for pairs
                      (prev, next) of states where next is a larger prefix: M = sum max(0, D[next] - D[prev]);
                      violations = number of pairs with D[next] > D[prev].

  gradient of D ..... d/d(image) of sum_b weight_b D_b, D = MSE + lambda (1 - SSIM) (the term E_w[D_w] of Eq. (2),
                      PAPER.md:66-72): the chain rule of the definitions above written out (distortion_backward);
                      pins: tests/test_distortion_backward_pins.py (central differences of D itself, the zero
                      at image = reference, the MSE-only closed form)

  objective weights . d/dD_b of  w_mean mean(D) + w_cvar CVaR_alpha(D) + w_mono M(D)  (Eq. (2): the terms
                      of the objective that are functions of the per-state distortions; lambda_c = 0.30,
                      lambda_m = 2.0 in PAPER.md:72): mean -> 1/n each; CVaR (upper tail) -> 1/k for every value
                      strictly above the threshold, and the remaining (k - #above)/k shared equally by the values
                      equal to it (a subgradient; reading L1); M -> +1 on next and -1 on prev of every violated pair
                      (objective_weights); flicker_backward: d F_b/d out_b(t2) = 2 e / (3 H W) = - d F_b/d out_b(t1)
                      pins: tests/test_distortion_backward_pins.py d4, d5 (differences of the forward reductions)

Pins: tests/test_metrics_pins.py (SSIM(x,x) = 1, constant-image closed form, scipy.ndimage Gaussian filtering
as an independent library route, hand-worked CVaR / quantile, constant-shift flicker closed form, the paper's
four monotone prefix points PAPER.md:94).
"""
from __future__ import annotations

import math

import numpy as np

SSIM_C1, SSIM_C2 = 0.01 ** 2, 0.03 ** 2
SSIM_RADIUS, SSIM_SIGMA = 5, 1.5
MIX_WEIGHT = 0.20


def gaussian_window() -> np.ndarray:
    """The 11 normalised 1-D weights exp(-(k-5)^2 / (2 sigma^2)) / sum."""
    g = np.array([math.exp(-((k - SSIM_RADIUS) ** 2) / (2.0 * SSIM_SIGMA ** 2)) for k in range(2 * SSIM_RADIUS + 1)])
    return g / g.sum()


def _blur(a: np.ndarray) -> np.ndarray:
    """w * a for one [H, W] plane: separable, zero padding, rows then columns."""
    g = gaussian_window()
    H, W = a.shape
    pad = np.zeros((H, W + 2 * SSIM_RADIUS))
    pad[:, SSIM_RADIUS:SSIM_RADIUS + W] = a
    h = np.zeros((H, W))
    for k in range(2 * SSIM_RADIUS + 1):
        h += g[k] * pad[:, k:k + W]
    pad = np.zeros((H + 2 * SSIM_RADIUS, W))
    pad[SSIM_RADIUS:SSIM_RADIUS + H, :] = h
    v = np.zeros((H, W))
    for k in range(2 * SSIM_RADIUS + 1):
        v += g[k] * pad[k:k + H, :]
    return v


def ssim_map(img: np.ndarray, ref: np.ndarray) -> np.ndarray:
    """[H, W, 3] x [H, W, 3] -> SSIM map [H, W, 3] (reading G1)."""
    x, y = np.asarray(img, np.float64), np.asarray(ref, np.float64)
    out = np.zeros(x.shape)
    for ch in range(x.shape[2]):
        mx, my = _blur(x[:, :, ch]), _blur(y[:, :, ch])
        sxx = _blur(x[:, :, ch] * x[:, :, ch]) - mx * mx
        syy = _blur(y[:, :, ch] * y[:, :, ch]) - my * my
        sxy = _blur(x[:, :, ch] * y[:, :, ch]) - mx * my
        out[:, :, ch] = ((2 * mx * my + SSIM_C1) * (2 * sxy + SSIM_C2)) / ((mx * mx + my * my + SSIM_C1) * (sxx + syy + SSIM_C2))
    return out


def ssim(imgs: np.ndarray, ref: np.ndarray) -> np.ndarray:
    """[B, H, W, 3] vs [H, W, 3] -> SSIM per state, float64 [B]."""
    return np.array([ssim_map(im, ref).mean() for im in np.asarray(imgs)])


def ssim_backward_map(img: np.ndarray, ref: np.ndarray) -> np.ndarray:
    """d(mean of the SSIM map)/d(img) for one state, [H, W, 3].  With m1 = w*x, m2 = w*(x x), m12 = w*(x y) (the
    three blurred planes that depend on x) and
        N1 = 2 mu_x mu_y + C1, N2 = 2 s_xy + C2, D1 = mu_x^2 + mu_y^2 + C1, D2 = s_xx + s_yy + C2, ssim = N1 N2 / (D1 D2),
        mu_x = m1, s_xx = m2 - m1^2, s_xy = m12 - m1 mu_y:
        d ssim/d s_xx = -N1 N2 / (D1 D2^2)                      (= d ssim/d m2)
        d ssim/d s_xy = 2 N1 / (D1 D2)                          (= d ssim/d m12)
        d ssim/d m1   = 2 mu_y N2 / (D1 D2) - 2 mu_x N1 N2 / (D1^2 D2) - 2 mu_x d ssim/d s_xx - mu_y d ssim/d s_xy
    A blurred plane is linear in x with the symmetric window (zero padding keeps the operator symmetric), so
        d mean/dx = ( w*(d ssim/d m1) + 2 x w*(d ssim/d m2) + y w*(d ssim/d m12) ) / (3 H W)."""
    x, y = np.asarray(img, np.float64), np.asarray(ref, np.float64)
    out = np.zeros(x.shape)
    n = float(x.size)
    for ch in range(x.shape[2]):
        xc, yc = x[:, :, ch], y[:, :, ch]
        mx, my = _blur(xc), _blur(yc)
        sxx = _blur(xc * xc) - mx * mx
        syy = _blur(yc * yc) - my * my
        sxy = _blur(xc * yc) - mx * my
        N1, N2 = 2 * mx * my + SSIM_C1, 2 * sxy + SSIM_C2
        D1, D2 = mx * mx + my * my + SSIM_C1, sxx + syy + SSIM_C2
        d_sxx = -N1 * N2 / (D1 * D2 * D2)
        d_sxy = 2 * N1 / (D1 * D2)
        d_m1 = 2 * my * N2 / (D1 * D2) - 2 * mx * N1 * N2 / (D1 * D1 * D2) - 2 * mx * d_sxx - my * d_sxy
        out[:, :, ch] = (_blur(d_m1) + 2 * xc * _blur(d_sxx) + yc * _blur(d_sxy)) / n
    return out


def distortion_backward(imgs: np.ndarray, ref: np.ndarray, weight, lam: float = MIX_WEIGHT) -> np.ndarray:
    """d/d(imgs) of sum_b weight[b] (MSE_b + lam (1 - SSIM_b)): [B, H, W, 3] float64.
    MSE_b = mean((img_b - ref)^2) over H x W x 3, so d MSE/d img = 2 (img - ref) / (3 H W)."""
    im, rf = np.asarray(imgs, np.float64), np.asarray(ref, np.float64)
    w = np.asarray(weight, np.float64).reshape(-1)
    out = np.zeros(im.shape)
    for b in range(im.shape[0]):
        g = 2.0 * (im[b] - rf) / float(rf.size)
        if lam != 0.0:
            g = g - lam * ssim_backward_map(im[b], rf)
        out[b] = w[b] * g
    return out


def mixed_distortion(mse: np.ndarray, ssim_v: np.ndarray) -> np.ndarray:
    return np.asarray(mse, np.float64) + MIX_WEIGHT * (1.0 - np.asarray(ssim_v, np.float64))


RISK_FIELDS = ("mean", "cvar", "quantile", "worst", "count")


def risk_reduce(values, alpha: float, upper_tail: bool) -> dict:
    """Reading G2.  upper_tail=True: large values are bad (a distortion); False: small values are bad (a PSNR)."""
    v = sorted(float(x) for x in np.asarray(values, np.float64).reshape(-1))
    n = len(v)
    if n == 0:
        return dict(mean=0.0, cvar=0.0, quantile=0.0, worst=0.0, count=0.0)
    k = max(1, int(math.ceil(alpha * n)))
    k = min(k, n)
    if upper_tail:
        tail = v[n - k:]
        pos = (1.0 - alpha) * (n - 1)
        worst = v[-1]
    else:
        tail = v[:k]
        pos = alpha * (n - 1)
        worst = v[0]
    lo = int(math.floor(pos))
    hi = min(lo + 1, n - 1)
    q = v[lo] + (pos - lo) * (v[hi] - v[lo])
    return dict(mean=sum(v) / n, cvar=sum(tail) / k, quantile=q, worst=worst, count=float(n))


def flicker(imgs_t1, imgs_t2, ref_t1, ref_t2) -> np.ndarray:
    """Reading G3.  [B,H,W,3], [B,H,W,3], [H,W,3], [H,W,3] -> float64 [B]."""
    a, b = np.asarray(imgs_t1, np.float64), np.asarray(imgs_t2, np.float64)
    r1, r2 = np.asarray(ref_t1, np.float64), np.asarray(ref_t2, np.float64)
    out = np.zeros(a.shape[0])
    for s in range(a.shape[0]):
        e = (b[s] - a[s]) - (r2 - r1)
        out[s] = (e * e).sum() / e.size
    return out


def prefix_monotonicity(d, idx_prev, idx_next):
    """Reading G4.  Returns (M, violations)."""
    d = np.asarray(d, np.float64).reshape(-1)
    M, viol = 0.0, 0
    for p, q in zip(np.asarray(idx_prev).tolist(), np.asarray(idx_next).tolist()):
        inc = float(d[q]) - float(d[p])
        if inc > 0.0:
            M += inc
            viol += 1
    return M, viol


def objective_weights(d, w_mean: float, w_cvar: float, alpha: float, idx_prev=(), idx_next=(), w_mono: float = 0.0) -> np.ndarray:
    """dL/dD_b for L = w_mean mean(D) + w_cvar CVaR_alpha(D) (upper tail, reading G2) + w_mono M(D) (reading G4)."""
    v = [float(x) for x in np.asarray(d, np.float64).reshape(-1)]
    n = len(v)
    w = [0.0] * n
    if n == 0:
        return np.zeros(0)
    for i in range(n):
        w[i] += w_mean / n
    k = min(max(1, int(math.ceil(alpha * n))), n)
    thr = sorted(v)[n - k]                      # the mildest of the k worst (largest) values
    above = sum(1 for x in v if x > thr)
    ties = sum(1 for x in v if x == thr)
    for i in range(n):
        if v[i] > thr:
            w[i] += w_cvar / k
        elif v[i] == thr:
            w[i] += w_cvar * (k - above) / (ties * k)
    for p, q in zip(np.asarray(idx_prev).tolist(), np.asarray(idx_next).tolist()):
        if v[q] - v[p] > 0.0:
            w[q] += w_mono
            w[p] -= w_mono
    return np.array(w)


def flicker_backward(imgs_t1, imgs_t2, ref_t1, ref_t2, weight):
    """d/d(imgs_t1), d/d(imgs_t2) of sum_b weight[b] F_b (reading G3): ([B,H,W,3], [B,H,W,3]) float64."""
    a, b = np.asarray(imgs_t1, np.float64), np.asarray(imgs_t2, np.float64)
    r1, r2 = np.asarray(ref_t1, np.float64), np.asarray(ref_t2, np.float64)
    w = np.asarray(weight, np.float64).reshape(-1)
    g2 = np.zeros(a.shape)
    for s_ in range(a.shape[0]):
        e = (b[s_] - a[s_]) - (r2 - r1)
        g2[s_] = w[s_] * 2.0 * e / e.size
    return -g2, g2

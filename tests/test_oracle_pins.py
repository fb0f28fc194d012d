"""Pins of the CPU oracle against what the paper and the mathematics fix (SURVEY.md §8(c) P1..P16 + P17).

CPU-only.  None of these re-type the oracle's own formulas: they are hand-enumerated tables,
closed forms of special cases, invariants, or library linear algebra (numpy) on the same inputs.
"""
from pathlib import Path

import numpy as np
import pytest

from paper_2606_17212_b200 import synth
from tests.helpers import Y0, axis_camera, tiny_scene

GOLD = Path(__file__).resolve().parent / "golden"


# ------------------------------------------------------------------------------------------ P1
def test_p1_closure_truth_table(oracle_mod):
    rows = [l.split() for l in (GOLD / "closure_truth_table.txt").read_text().splitlines()
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 16
    mask = np.array([int(r[0], 2) for r in rows], np.uint8)
    depth, closure = oracle_mod.close_levels(mask)
    assert depth.tolist() == [int(r[1]) for r in rows]
    assert closure.tolist() == [int(r[2], 2) for r in rows]


def test_p1_closure_properties(oracle_mod):
    m = np.arange(16, dtype=np.uint8)
    depth, closure = oracle_mod.close_levels(m)
    # idempotent: closing a closed mask changes nothing
    d2, c2 = oracle_mod.close_levels(closure)
    assert np.array_equal(d2, depth) and np.array_equal(c2, closure)
    # closure is a subset of the mask; monotone: setting a bit never lowers depth
    assert np.all((closure & m) == closure)
    for a in range(16):
        for bit in range(4):
            assert depth[a | (1 << bit)] >= depth[a]
    # every mask with bit 0 clear has depth -1
    assert np.all(depth[(m & 1) == 0] == -1)


def test_p1_cfg0_states_are_all_closed_depth_vectors():
    lv = synth.all_closed_states(4)
    assert lv.shape == (625, 4)
    assert len({tuple(r) for r in lv.tolist()}) == 625
    assert lv.min() == -1 and lv.max() == 3
    assert lv[0].tolist() == [-1, -1, -1, -1] and lv[-1].tolist() == [3, 3, 3, 3]
    assert lv[1].tolist() == [-1, -1, -1, 0]          # lexicographic, last cluster fastest


# ------------------------------------------------------------------------------------------ P2
@pytest.mark.parametrize("bg", [(0.0, 0.0, 0.0), (1.0, 1.0, 1.0), (0.25, 0.5, 0.125)])
def test_p2_all_absent_state_is_background_bitwise(oracle_mod, bg):
    wl = synth.workload_cfg0()
    wl.scene.background = np.asarray(bg, np.float32)
    sc = oracle_mod.OracleScene(wl.scene)
    cam, t = wl.frames[0]
    for brute in (False, True):
        img, st = sc.render(cam, t, np.full(4, -1, np.int8), brute_force=brute)
        assert np.array_equal(img, np.broadcast_to(np.asarray(bg, np.float32).astype(np.float64), img.shape))
        assert st.tolist() == [0, 0]


# ------------------------------------------------------------------------------------------ P3
def _closed_form_single(cam, f, s, z0, o, c, bg, rect_px):
    sig2 = (f * s / z0) ** 2 + 0.3
    ys, xs = np.mgrid[0:cam.H, 0:cam.W]
    r2 = (xs + 0.5 - cam.cx) ** 2 + (ys + 0.5 - cam.cy) ** 2
    alpha = np.minimum(0.99, o * np.exp(-r2 / (2 * sig2)))
    inside = (xs >= rect_px[0]) & (xs < rect_px[2]) & (ys >= rect_px[1]) & (ys < rect_px[3])
    alpha = np.where(inside & (alpha >= 1.0 / 255.0), alpha, 0.0)
    return alpha[..., None] * np.asarray(c)[None, None, :] + (1 - alpha[..., None]) * np.asarray(bg)[None, None, :]


@pytest.mark.parametrize("bg", [(0.0, 0.0, 0.0), (1.0, 1.0, 1.0)])
def test_p3_single_isotropic_gaussian_closed_form(oracle_mod, bg):
    f, z0, s, logit = 100.0, 4.0, 0.2, 0.8472979        # sigma' ~ 5 px ; o ~ 0.7
    col = (0.8, 0.3, 0.6)
    scn, _ = tiny_scene([[0, 0, 0]], s, logits=logit, colors=col, background=bg)
    cam = axis_camera(128, 128, f, z0)
    sc = oracle_mod.OracleScene(scn)
    o = 1.0 / (1.0 + np.exp(-logit))
    # by hand: sigma'^2 = 25.3 ; lambda = 25.3 + sqrt(0.1) ; r = ceil(3*sqrt(25.616)) = 16
    # rect: tiles floor((64-16)/16)=3 .. floor((64+16+15)/16)=5 -> pixels [48, 80)
    p = sc.project(cam, 0.0, np.zeros(1, np.int8))
    assert p["valid"][0] == 1 and p["radius"][0] == 16 and p["rect"][0].tolist() == [3, 3, 5, 5]
    expect = _closed_form_single(cam, f, s, z0, o, col, bg, (48, 48, 80, 80))
    for brute in (False, True):
        img, _ = sc.render(cam, 0.0, np.zeros(1, np.int8), brute_force=brute)
        assert np.abs(img - expect).max() < 2e-6
    assert np.abs(img[64, 64] - expect[64, 64]).max() < 2e-6 and abs(expect[64, 64, 0] - bg[0]) > 0.1


# ------------------------------------------------------------------------------------------ P4
def test_p4_transmittance_monotone_and_telescoping(oracle_mod):
    wl = synth.workload_cfg0()
    # all colours exactly 1, black background -> pixel = sum_i alpha_i T_{i-1} = 1 - T_final
    wl.scene.sh_base[:] = 0
    wl.scene.sh_base[:, 0, :] = np.float32(0.5 / Y0)
    wl.scene.sh_res[:] = 0
    wl.scene.log_scale += 1.0                      # bigger splats: long per-pixel sequences
    sc = oracle_mod.OracleScene(wl.scene)
    cam, t = wl.frames[0]
    full = np.full(4, 2, np.int8)
    img, st, Tf = sc.render(cam, t, full, want_T=True)
    c1 = np.float64(np.float32(0.5 / Y0)) * Y0 + 0.5      # the colour actually encoded (~1)
    assert np.all((Tf >= 0) & (Tf <= 1))
    assert np.abs(img[..., 0] - c1 * (1 - Tf)).max() < 1e-12
    rng = np.random.default_rng(0)
    longest = 0
    for _ in range(200):
        x, y = rng.integers(0, cam.W), rng.integers(0, cam.H)
        g, a, T = sc.trace_pixel(cam, t, full, int(x), int(y))
        if len(T) == 0:
            continue
        longest = max(longest, len(T))
        Tprev = np.concatenate([[1.0], T[:-1]])
        assert np.all(T <= Tprev) and np.all(T >= 0) and np.all(T <= 1)
        acc = np.where(a > 0, a, 0.0)
        assert abs((acc * Tprev).sum() + T[-1] - 1.0) < 1e-12
    assert longest >= 10


# ------------------------------------------------------------------------------------------ P5
def test_p5_two_coaxial_gaussians_over_formula(oracle_mod):
    f, z0 = 100.0, 4.0
    c1, c2 = (0.9, 0.1, 0.2), (0.1, 0.8, 0.3)
    cam = axis_camera(64, 64, f, z0, cx=32.5, cy=32.5)     # pixel (32,32) centre exactly on the axis
    def centre(zs, cols, logits):
        scn, order = tiny_scene([[0, 0, zs[0]], [0, 0, zs[1]]], 0.3, logits=logits, colors=cols)
        sc = oracle_mod.OracleScene(scn)
        img, _ = sc.render(cam, 0.0, np.zeros(1, np.int8), brute_force=True)
        return img[32, 32], sc
    o1, o2 = 1 / (1 + np.exp(-0.5)), 1 / (1 + np.exp(0.3))
    # Gaussian 0 in front (smaller z)
    px, _ = centre([-0.5, 0.5], [c1, c2], [0.5, -0.3])
    exp = o1 * np.array(c1) + (1 - o1) * o2 * np.array(c2)
    assert np.abs(px - exp).max() < 1e-6
    # swap depths -> roles swap
    px, _ = centre([0.5, -0.5], [c1, c2], [0.5, -0.3])
    exp = o2 * np.array(c2) + (1 - o2) * o1 * np.array(c1)
    assert np.abs(px - exp).max() < 1e-6
    # equal depth -> ordered by index (Gaussian 0 first)
    px, sc = centre([0.0, 0.0], [c1, c2], [0.5, -0.3])
    exp = o1 * np.array(c1) + (1 - o1) * o2 * np.array(c2)
    assert np.abs(px - exp).max() < 1e-6
    g, a, T = sc.trace_pixel(cam, 0.0, np.zeros(1, np.int8), 32, 32)
    assert g.tolist() == [0, 1]


# ------------------------------------------------------------------------------------------ P6
def test_p6_integer_footprint_by_hand(oracle_mod):
    f, z0 = 100.0, 4.0
    cam = axis_camera(128, 96, f, z0)                      # 8 x 6 tiles
    s = 0.04                                               # sigma'^2 = 1 + 0.3 ; r = ceil(3 sqrt(1.3+0.3162)) = 4
    # world x = (px - cx) z0 / f.  Place 2-D means by hand:
    def world(px, py):
        return [(px - cam.cx) * z0 / f, (py - cam.cy) * z0 / f, 0.0]
    means = [world(40.0, 40.0),      # interior: x in [36,44] -> tiles floor(36/16)=2 .. floor(59/16)=3 -> [2,3) ; same in y
             world(47.0, 16.0),      # x: [43,51] -> floor(43/16)=2 .. floor(66/16)=4 -> [2,4) ; y: [12,20] -> 0..floor(35/16)=2 -> [0,2)
             world(1.0, 94.0),       # corner: x [-3,5] -> clamp(floor(-3/16)=-1)=0 .. floor(20/16)=1 ; y [90,98] -> 5 .. clamp(floor(113/16)=7,6)=6
             world(-20.0, 40.0),     # off-screen left: x [-24,-16] -> tx0 = 0, tx1 = clamp(floor(-1/16) = -1) = 0 -> empty
             world(140.0, 40.0)]     # off-screen right: x [136,144] -> tx0 = clamp(8,8)=8, tx1 = 8 -> empty
    # flat in z (scale 1e-4) so the perspective term of the Jacobian adds nothing off-axis
    scn, _ = tiny_scene(means, [[s, s, 1e-4]] * 5)
    sc = oracle_mod.OracleScene(scn)
    p = sc.project(cam, 0.0, np.zeros(1, np.int8))
    assert p["radius"].tolist() == [4] * 5
    assert p["valid"].tolist() == [1, 1, 1, 0, 0]
    assert p["rect"][0].tolist() == [2, 2, 3, 3] and p["count"][0] == 1
    assert p["rect"][1].tolist() == [2, 0, 4, 2] and p["count"][1] == 4
    assert p["rect"][2].tolist() == [0, 5, 1, 6] and p["count"][2] == 1
    # behind the near plane: culled
    scn, _ = tiny_scene([[0, 0, -3.9]], s)         # z_cam = 0.1 <= znear
    p = oracle_mod.OracleScene(scn).project(cam, 0.0, np.zeros(1, np.int8))
    assert p["valid"][0] == 0


# ------------------------------------------------------------------------------------------ P7
def test_p7_axis_aligned_anisotropic_and_roll(oracle_mod):
    f, z0 = 100.0, 4.0
    cam = axis_camera(128, 128, f, z0)
    sx, sy, sz = 0.2, 0.08, 0.5
    scn, _ = tiny_scene([[0, 0, 0]], [[sx, sy, sz]])
    p = oracle_mod.OracleScene(scn).project(cam, 0.0, np.zeros(1, np.int8))[0]
    a, c = (f * sx / z0) ** 2 + 0.3, (f * sy / z0) ** 2 + 0.3
    assert abs(p["cov2d"][0] - a) < 1e-4 * a and abs(p["cov2d"][2] - c) < 1e-4 * c and abs(p["cov2d"][1]) < 1e-5
    assert abs(p["qa"] - 0.5 / a) < 1e-6 and abs(p["qc"] - 0.5 / c) < 1e-6
    # 90 degree roll about z: quaternion (cos45, 0, 0, sin45) swaps the screen axes
    h = np.sqrt(0.5)
    scn, _ = tiny_scene([[0, 0, 0]], [[sx, sy, sz]], quats=[[h, 0, 0, h]])
    p = oracle_mod.OracleScene(scn).project(cam, 0.0, np.zeros(1, np.int8))[0]
    assert abs(p["cov2d"][0] - c) < 1e-4 * c and abs(p["cov2d"][2] - a) < 1e-4 * a and abs(p["cov2d"][1]) < 1e-4
    # 90 degree rotation about y brings the z scale onto the screen x axis
    scn, _ = tiny_scene([[0, 0, 0]], [[sx, sy, sz]], quats=[[h, 0, h, 0]])
    p = oracle_mod.OracleScene(scn).project(cam, 0.0, np.zeros(1, np.int8))[0]
    az = (f * sz / z0) ** 2 + 0.3
    assert abs(p["cov2d"][0] - az) < 1e-4 * az and abs(p["cov2d"][2] - c) < 1e-4 * c


# ------------------------------------------------------------------------------------------ P8
def test_p8_deformation_special_cases(oracle_mod):
    assert oracle_mod.basis(0.0, 4).tolist() == [1.0, 1.0, 1.0, 1.0]
    assert np.allclose(oracle_mod.basis(1.0, 4), [-1, 1, -1, 1], atol=1e-7)
    assert np.allclose(oracle_mod.basis(0.5, 4), [0, -1, 0, 1], atol=1e-7)
    rng = np.random.default_rng(1)
    N = 6
    means = rng.uniform(-1, 1, (N, 3))
    A0 = np.zeros((1, 3, 4)); A0[0, :, :3] = np.eye(3) + 0.1 * rng.standard_normal((3, 3)); A0[0, :, 3] = [0.1, -0.2, 0.3]
    A1 = 0.05 * rng.standard_normal((1, 3, 4))
    q = rng.integers(-127, 128, (N, 1, 3)).astype(np.int8)
    scn, order = tiny_scene(means, 0.05, A0=A0, A1=A1, motion_q=q, motion_scale=[0.01], R=1,
                            levels=[0, 0, 1, 1, 2, 3])
    sc = oracle_mod.OracleScene(scn)
    cam = axis_camera()
    m = means[order]
    hom = np.concatenate([m, np.ones((N, 1))], axis=1)
    # t = 0: A = A0, depth 0 -> affine only
    p = sc.project(cam, 0.0, np.array([0], np.int8))
    exp0 = hom @ A0[0].T
    present = scn.level_of() <= 0
    assert np.abs(p["mu"][present] - exp0[present]).max() < 1e-6
    # t = 0.25, depth 1: R = 1 single-term residual by hand: s_c * cos(pi t) * q
    t = 0.25
    p = sc.project(cam, t, np.array([1], np.int8))
    expA = hom @ (A0[0] + t * A1[0]).T
    exp1 = expA + 0.01 * np.cos(np.pi * t) * q[order][:, 0, :].astype(np.float64)
    present = scn.level_of() <= 1
    assert np.abs(p["mu"][present] - exp1[present]).max() < 1e-6
    # depth 0 at the same t has no residual
    p0 = sc.project(cam, t, np.array([0], np.int8))
    assert np.abs(p0["mu"][scn.level_of() == 0] - expA[scn.level_of() == 0]).max() < 1e-6
    # q == 0 -> depth 0 and depth 1 geometry identical bit for bit
    scn2, _ = tiny_scene(means, 0.05, A0=A0, A1=A1, motion_scale=[0.01], R=1, levels=[0, 0, 1, 1, 2, 3])
    sc2 = oracle_mod.OracleScene(scn2)
    a, b = sc2.project(cam, t, np.array([0], np.int8)), sc2.project(cam, t, np.array([1], np.int8))
    base = scn2.level_of() == 0
    for fld in ("mu", "mx", "my", "qa", "qb", "qc", "radius", "rect", "depth_bits"):
        assert np.array_equal(a[fld][base], b[fld][base])
    # presence: level l present iff depth >= l
    for d in range(-1, 4):
        p = sc.project(cam, 0.3, np.array([d], np.int8))
        assert np.array_equal(p["valid"] == 1, scn.level_of() <= d)


# ------------------------------------------------------------------------------------------ P9
def test_p9_sh_orthonormal_by_quadrature(oracle_mod):
    # Gauss-Legendre in cos(theta) x uniform phi integrates polynomials of degree <= 6 exactly
    xs, ws = np.polynomial.legendre.leggauss(8)
    nphi = 16
    G = np.zeros((16, 16))
    for ct, w in zip(xs, ws):
        st = np.sqrt(1 - ct * ct)
        for k in range(nphi):
            ph = 2 * np.pi * (k + 0.5) / nphi
            Y = oracle_mod.sh_basis(16, (st * np.cos(ph), st * np.sin(ph), ct))
            G += w * (2 * np.pi / nphi) * np.outer(Y, Y)
    assert np.abs(G - np.eye(16)).max() < 1e-12


def test_p9_colour_special_cases(oracle_mod):
    cam = axis_camera()
    col = (0.2, 0.7, 0.4)
    scn, _ = tiny_scene([[0.3, -0.2, 0.1]], 0.1, colors=col)
    p = oracle_mod.OracleScene(scn).project(cam, 0.0, np.zeros(1, np.int8))[0]
    assert np.abs(p["rgb"] - np.array(col)).max() < 1e-7           # degree 0: Y0*sh0 + 0.5
    # sh_res == 0 -> depth 3 colour == depth 2 colour bitwise; non-zero residual changes only depth 3
    wl = synth.workload_cfg0()
    cam, t = wl.frames[0]
    sc = oracle_mod.OracleScene(wl.scene)
    a, b = sc.project(cam, t, np.full(4, 2, np.int8)), sc.project(cam, t, np.full(4, 3, np.int8))
    both = (a["valid"] == 1)
    assert np.abs(a["rgb"][both] - b["rgb"][both]).max() > 1e-4
    wl.scene.sh_res[:] = 0
    sc = oracle_mod.OracleScene(wl.scene)
    a, b = sc.project(cam, t, np.full(4, 2, np.int8)), sc.project(cam, t, np.full(4, 3, np.int8))
    assert np.array_equal(a["rgb"][both], b["rgb"][both])
    # clamp at zero: a strongly negative DC gives exactly 0
    scn, _ = tiny_scene([[0, 0, 0]], 0.1, colors=(-0.5, 0.5, 2.0))
    p = oracle_mod.OracleScene(scn).project(axis_camera(), 0.0, np.zeros(1, np.int8))[0]
    assert p["rgb"][0] == 0.0 and abs(p["rgb"][2] - 2.0) < 1e-6      # no upper clamp (reading A13)


# ------------------------------------------------------------------------------------------ P10
def test_p10_key_list(oracle_mod):
    wl = synth.workload_cfg0()
    cam, t = wl.frames[0]
    sc = oracle_mod.OracleScene(wl.scene)
    for depth in ([3, 3, 3, 3], [0, 1, 2, 3], [-1, 2, -1, 0]):
        p = sc.project(cam, t, np.array(depth, np.int8))
        tile, dbits, idx = sc.keys(p, cam)
        # independent enumeration with numpy
        TX = (cam.W + 15) // 16
        rows = []
        for i in np.nonzero(p["valid"])[0]:
            x0, y0, x1, y1 = p["rect"][i]
            for ty in range(y0, y1):
                for tx in range(x0, x1):
                    rows.append((ty * TX + tx, int(p["depth_bits"][i]), int(i)))
        rows = np.array(rows, np.int64)
        assert len(rows) == len(tile) == p["count"][p["valid"] == 1].sum()
        order = np.lexsort((rows[:, 2], rows[:, 1], rows[:, 0]))
        assert np.array_equal(rows[order, 0], tile) and np.array_equal(rows[order, 1], dbits)
        assert np.array_equal(rows[order, 2], idx)
        key = (tile.astype(object) << 64) | (dbits.astype(object) << 32) | idx.astype(object)
        assert all(key[k] < key[k + 1] for k in range(len(key) - 1))        # strictly increasing, unique
        # depth bits order == float order for positive z
        z = p["z"][idx]
        same_tile = tile[1:] == tile[:-1]
        assert np.all(z[1:][same_tile] >= z[:-1][same_tile])


# ------------------------------------------------------------------------------------------ P11
def test_p11_brute_force_equals_gaussian_major_bitwise(oracle_mod):
    wl = synth.workload_cfg0()
    wl.scene.log_scale += 0.7                     # enough overlap that order and termination matter
    cam, t = wl.frames[0]
    sc = oracle_mod.OracleScene(wl.scene)
    lv = wl.levels[0][::25]
    a, sa = sc.render_batch(cam, t, lv, brute_force=True)
    b, sb = sc.render_batch(cam, t, lv, brute_force=False)
    assert np.array_equal(a, b)
    assert np.array_equal(sa[:, 0], sb[:, 0])
    assert np.all(sb[:, 1] <= sa[:, 1])           # O2 stops visiting a pixel once it terminated; O1 breaks too
    assert a.std() > 0.05


# ------------------------------------------------------------------------------------------ P12
def test_p12_permutation_within_group_leaves_image_unchanged(oracle_mod):
    wl = synth.workload_cfg0()
    cam, t = wl.frames[0]
    scn = wl.scene
    img0, _ = oracle_mod.OracleScene(scn).render(cam, t, np.full(4, 3, np.int8))
    rng = np.random.default_rng(5)
    perm = np.arange(scn.N)
    for g in range(4 * scn.C):
        a, b = scn.group_off[g], scn.group_off[g + 1]
        perm[a:b] = a + rng.permutation(b - a)
    for name in ("mean", "log_scale", "quat", "opacity_logit", "sh_base", "sh_res", "motion_q"):
        setattr(scn, name, np.ascontiguousarray(getattr(scn, name)[perm]))
    img1, _ = oracle_mod.OracleScene(scn).render(cam, t, np.full(4, 3, np.int8))
    assert np.array_equal(img0, img1)             # random depths: no ties, so the order is unchanged


# ------------------------------------------------------------------------------------------ P13
def test_p13_distortion(oracle_mod):
    rng = np.random.default_rng(2)
    ref = rng.uniform(0, 1, (8, 12, 3))
    eps = 0.01
    imgs = np.stack([ref, ref + eps, ref - 2 * eps])
    mse, psnr = oracle_mod.distortion(imgs, ref)
    assert mse[0] == 0.0 and psnr[0] == 100.0                       # MSE floor 1e-10 -> 100 dB cap
    assert abs(mse[1] - eps ** 2) < 1e-15 and abs(psnr[1] + 20 * np.log10(eps)) < 1e-9
    assert abs(mse[2] - 4 * eps ** 2) < 1e-15
    x = rng.uniform(0, 1, (3, 8, 12, 3))
    mse, psnr = oracle_mod.distortion(x, ref)
    assert np.allclose(mse, ((x - ref[None]) ** 2).mean(axis=(1, 2, 3)), rtol=1e-13)
    assert np.allclose(psnr, 10 * np.log10(1.0 / mse), rtol=1e-13)


# ------------------------------------------------------------------------------------------ P14
def test_p14_eq4_by_hand(oracle_mod):
    for line in (GOLD / "eq4_hand.txt").read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        lhs, rhs = line.split("|")
        v = np.array([float(x) for x in lhs.split()])
        mean, q10, sd, risk = [float(x) for x in rhs.split()]
        n = len(v)
        # feed as pairs: mse_without = v, mse_with = 0
        mse = np.concatenate([v, np.zeros(n)])
        psnr = np.concatenate([np.zeros(n), v])         # delta_db = psnr_with - psnr_without = v
        dm, dd, util = oracle_mod.group_utility(mse, psnr, np.arange(n), np.arange(n, 2 * n), np.zeros(n, int), 1)
        assert np.array_equal(dm, v) and np.array_equal(dd, v)
        for off in (0, 4):
            assert abs(util[0, off + 0] - mean) < 1e-12 and abs(util[0, off + 1] - q10) < 1e-12
            assert abs(util[0, off + 2] - sd) < 1e-12 and abs(util[0, off + 3] - risk) < 1e-9
        assert util[0, 8] == n


def test_p14_aggregates_match_numpy(oracle_mod):
    rng = np.random.default_rng(3)
    n, G = 500, 7
    mse = rng.uniform(0, 0.1, 2 * n)
    psnr = -10 * np.log10(mse)
    gid = rng.integers(0, G - 1, n)                   # last group stays empty
    iw, iwith = np.arange(n), rng.permutation(n) + n
    dm, dd, util = oracle_mod.group_utility(mse, psnr, iw, iwith, gid, G)
    assert np.array_equal(dm, mse[iw] - mse[iwith]) and np.array_equal(dd, psnr[iwith] - psnr[iw])
    for g in range(G - 1):
        for off, v in ((0, dm[gid == g]), (4, dd[gid == g])):
            assert abs(util[g, off] - v.mean()) < 1e-12
            assert abs(util[g, off + 1] - np.quantile(v, 0.1, method="linear")) < 1e-12
            assert abs(util[g, off + 2] - np.std(v)) < 1e-12
            risk = (0.75 * v.mean() + 0.25 * np.quantile(v, 0.1)) / (1 + 0.05 * np.std(v))
            assert abs(util[g, off + 3] - risk) < 1e-12
        assert util[g, 8] == (gid == g).sum()
    assert np.all(util[G - 1] == 0)


def test_p14_offscreen_group_zero_and_disjoint_additive(oracle_mod):
    # cluster 0: left half of the screen, cluster 1: right half (disjoint tile support), cluster 2: off-screen
    rng = np.random.default_rng(4)
    cam = axis_camera(128, 64, 100.0, 4.0)
    n = 40
    def blob(cx_px, spread):
        px = cx_px + spread * rng.uniform(-1, 1, n)
        py = 32 + 14 * rng.uniform(-1, 1, n)
        return np.stack([(px - cam.cx) * 0.04, (py - cam.cy) * 0.04, rng.uniform(-0.3, 0.3, n)], axis=1)
    means = np.concatenate([blob(28, 12), blob(100, 12), blob(400, 10)])
    clusters = np.repeat([0, 1, 2], n)
    levels = np.tile(np.repeat([0, 1], n // 2), 3)
    cols = rng.uniform(0.1, 0.9, (3 * n, 3))
    scn, _ = tiny_scene(means, 0.05, clusters=clusters, levels=levels, colors=cols, logits=rng.standard_normal(3 * n))
    sc = oracle_mod.OracleScene(scn)
    states = np.array([[1, 1, 1],      # 0 full = reference
                       [0, 0, 0],      # 1 context
                       [1, 0, 0],      # 2 + group (0,1)
                       [0, 1, 0],      # 3 + group (1,1)
                       [1, 1, 0],      # 4 + both
                       [0, 0, 1]],     # 5 + off-screen group (2,1)
                      np.int8)
    imgs, stats = sc.render_batch(cam, 0.0, states)
    assert stats[5, 0] == stats[1, 0]                  # the off-screen cluster adds no intersections
    mse, psnr = oracle_mod.distortion(imgs, imgs[0])
    assert np.array_equal(imgs[5], imgs[1]) and mse[5] == mse[1]          # Delta = 0 exactly
    d_a, d_b, d_ab = mse[1] - mse[2], mse[1] - mse[3], mse[1] - mse[4]
    assert d_a > 0 and d_b > 0 and abs(d_ab - (d_a + d_b)) < 1e-15


# ------------------------------------------------------------------------------------------ P15
def test_p15_state_factorisation_mask_vs_depth(oracle_mod):
    wl = synth.workload_cfg0()
    cam, t = wl.frames[0]
    sc = oracle_mod.OracleScene(wl.scene)
    masks = np.array([[0b0111, 0b1011, 0b0001, 0b1110], [0b0011, 0b1101, 0b1111, 0b0101]], np.uint8)
    depth, _ = oracle_mod.close_levels(masks)
    assert depth.tolist() == [[2, 1, 0, -1], [1, 0, 3, 0]]
    other = np.array([[0b0111, 0b0011, 0b1001, 0b0000], [0b1011, 0b0001, 0b1111, 0b1001]], np.uint8)
    d2, _ = oracle_mod.close_levels(other)
    assert np.array_equal(depth, d2)
    a, _ = sc.render_batch(cam, t, depth)
    b, _ = sc.render_batch(cam, t, d2)
    assert np.array_equal(a, b)


# ------------------------------------------------------------------------------------------ P16
def test_p16_termination_count(oracle_mod):
    # 20 identical wide Gaussians stacked on the axis, logit 0 -> alpha = 0.5 at the centre pixel
    f, z0 = 100.0, 4.0
    cam = axis_camera(64, 64, f, z0, cx=32.5, cy=32.5)
    n = 20
    means = [[0, 0, 0.01 * k] for k in range(n)]
    col = (0.6, 0.6, 0.6)
    for bg in ((0.0, 0.0, 0.0), (1.0, 1.0, 1.0)):
        scn, _ = tiny_scene(means, 0.8, colors=col, background=bg)
        sc = oracle_mod.OracleScene(scn)
        g, a, T = sc.trace_pixel(cam, 0.0, np.zeros(1, np.int8), 32, 32)
        # accepted 1..13 (T = 2^-13 = 1.22e-4 >= 1e-4); the 14th would give 2^-14 < 1e-4 -> stop
        assert len(g) == 14 and g.tolist() == list(range(14))
        assert np.all(np.abs(a[:13] - 0.5) < 1e-6) and a[13] == -1.0
        assert abs(T[12] - 2.0 ** -13) < 1e-9 and T[13] == T[12]
        img, _ = sc.render(cam, 0.0, np.zeros(1, np.int8), brute_force=True)
        Tf = 2.0 ** -13
        assert np.abs(img[32, 32] - (np.array(col) * (1 - Tf) + Tf * np.array(bg))).max() < 1e-6
        # with the stop disabled all 20 are accepted and the pixel moves by < 1.3e-4
        img2, _ = sc.render(cam, 0.0, np.zeros(1, np.int8), brute_force=True, t_stop=0.0)
        assert 0 < np.abs(img2[32, 32] - img[32, 32]).max() < 1.3e-4


# ------------------------------------------------------------------------------------------ P17
def test_p17_projection_matches_numpy_linear_algebra(oracle_mod):
    """O-0 + O-3 against textbook matrix formulas evaluated with numpy in double:
    Sigma = R S S^T R^T ; Sigma' = J W Sigma W^T J^T + 0.3 I ; conic = inv(Sigma') ;
    radius from the largest eigenvalue (eigvalsh)."""
    rng = np.random.default_rng(7)
    N = 200
    means = rng.uniform(-1, 1, (N, 3))
    scales = np.exp(rng.normal(-3.0, 0.5, (N, 3)))
    quats = rng.standard_normal((N, 4))
    scn, order = tiny_scene(means, scales, quats=quats, logits=rng.standard_normal(N))
    R, tw = synth.look_at([2.5, -1.5, -3.0])
    cam = synth.make_camera(R, tw, 160, 112, 140.0)
    p = oracle_mod.OracleScene(scn).project(cam, 0.0, np.zeros(1, np.int8))
    Rd, td = R.astype(np.float64), tw.astype(np.float64)
    checked = 0
    for k in range(N):
        i = order[k]
        w, x, y, z = quats[i] / np.linalg.norm(quats[i])
        Rg = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                       [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                       [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])
        # the rotation really is a rotation taking e_k to column k
        assert np.allclose(Rg @ Rg.T, np.eye(3), atol=1e-12) and np.linalg.det(Rg) > 0.999
        Sig = Rg @ np.diag(scales[i] ** 2) @ Rg.T
        pc = Rd @ means[i].astype(np.float32).astype(np.float64) + td
        if pc[2] <= 0.2:
            assert p["valid"][k] == 0
            continue
        limx, limy = 1.3 * 0.5 * cam.W / cam.fx, 1.3 * 0.5 * cam.H / cam.fy
        xt = np.clip(pc[0] / pc[2], -limx, limx) * pc[2]
        yt = np.clip(pc[1] / pc[2], -limy, limy) * pc[2]
        J = np.array([[cam.fx / pc[2], 0, -cam.fx * xt / pc[2] ** 2], [0, cam.fy / pc[2], -cam.fy * yt / pc[2] ** 2]])
        S2 = J @ Rd @ Sig @ Rd.T @ J.T + 0.3 * np.eye(2)
        conic = np.linalg.inv(S2)
        lam = np.linalg.eigvalsh(S2)[1]
        m = np.array([cam.fx * pc[0] / pc[2] + cam.cx, cam.fy * pc[1] / pc[2] + cam.cy])
        if p["valid"][k] == 0:
            continue                                    # off-screen; footprint rules are pinned by P6
        assert np.allclose([p["mx"][k], p["my"][k]], m, atol=2e-3)
        assert np.allclose(p["cov2d"][k], [S2[0, 0], S2[0, 1], S2[1, 1]], rtol=2e-4, atol=1e-4)
        assert np.allclose([2 * p["qa"][k], p["qb"][k], 2 * p["qc"][k]], [conic[0, 0], conic[0, 1], conic[1, 1]],
                           rtol=5e-4, atol=1e-6)
        if lam - (S2[0, 0] + S2[1, 1]) / 2 > np.sqrt(0.1) * 1.05:     # away from the lambda floor (reading A11)
            r = 3 * np.sqrt(lam)
            assert p["radius"][k] in (int(np.ceil(r)), int(np.ceil(r - 1e-3)), int(np.ceil(r + 1e-3)))
        assert abs(p["z"][k] - pc[2]) < 1e-5
        checked += 1
    assert checked > 50


def test_p8_multi_term_basis_residual(oracle_mod):
    """Eq. (1) with R = 4 terms: residual = s_c * sum_{r=1..4} cos(pi r t) q_{i,r}, evaluated with numpy."""
    rng = np.random.default_rng(11)
    N, R = 5, 4
    means = rng.uniform(-1, 1, (N, 3))
    q = rng.integers(-127, 128, (N, R, 3)).astype(np.int8)
    scn, order = tiny_scene(means, 0.05, motion_q=q, motion_scale=[0.003], R=R)
    sc = oracle_mod.OracleScene(scn)
    t = 0.3
    p = sc.project(axis_camera(), t, np.array([1], np.int8))
    b = np.cos(np.pi * np.arange(1, R + 1) * np.float64(np.float32(t)))
    exp = means[order].astype(np.float32).astype(np.float64) + 0.003 * np.einsum("r,nrk->nk", b, q[order].astype(np.float64))
    assert np.abs(p["mu"] - exp).max() < 1e-6
    assert np.abs(exp - means[order]).max() > 0.05          # the residual is not negligible


# ------------------------------------------------------------------------------------------ P18: Eq. (1) residual levels
def test_p18_position_residual_levels(oracle_mod):
    """Eq. (1): mu = A mu_bar + sum_r b_r q_r + delta^(2) + delta^(3); reading I1: the level-l
    residual applies iff the cluster's depth is >= l.  Special cases: no residual arrays == zero arrays ==
    the old result; depth 0/1 ignore them; depth 2 shifts the deformed mean by exactly delta2 (one fp32 add),
    depth 3 by delta2 then delta3; an on-axis Gaussian shifted sideways by delta lands f*delta/z pixels away."""
    import dataclasses
    wl = synth.workload_cfg0()
    sc = wl.scene
    cam, t = wl.frames[0]
    base = oracle_mod.OracleScene(sc)
    zero = oracle_mod.OracleScene(dataclasses.replace(sc, delta2=np.zeros((sc.N, 3), np.float32),
                                                      delta3=np.zeros((sc.N, 3), np.float32)))
    scd = synth.with_position_residuals(sc)
    res = oracle_mod.OracleScene(scd)
    for d in range(-1, 4):
        depth = np.full(sc.C, d, np.int8)
        p0, pz, pr = base.project(cam, t, depth), zero.project(cam, t, depth), res.project(cam, t, depth)
        assert p0.tobytes() == pz.tobytes()
        if d <= 1:
            assert p0.tobytes() == pr.tobytes()
        present = sc.level_of() <= d
        if d == 2:
            want = p0["mu"] + scd.delta2
            assert np.array_equal(pr["mu"][present], want.astype(np.float32)[present])
        if d == 3:
            want = (p0["mu"] + scd.delta2).astype(np.float32) + scd.delta3
            assert np.array_equal(pr["mu"][present], want.astype(np.float32)[present])
    # closed form: one Gaussian on the optical axis, delta2 = (dx, 0, 0): the 2-D mean moves by f dx / z
    f, z0, dx = 100.0, 4.0, 0.25
    one, _ = tiny_scene([[0.0, 0.0, 0.0]], 0.05, levels=[0])
    one = dataclasses.replace(one, delta2=np.array([[dx, 0.0, 0.0]], np.float32))
    camx = axis_camera(W=128, H=128, f=f, z0=z0)
    o = oracle_mod.OracleScene(one)
    m1 = o.project(camx, 0.0, np.array([1], np.int8))
    m2 = o.project(camx, 0.0, np.array([2], np.int8))
    assert m2["mx"][0] - m1["mx"][0] == pytest.approx(f * dx / z0, abs=1e-4) and m2["my"][0] == m1["my"][0]


# ------------------------------------------------------------------------------------------ P19: attribute refinements
def test_p19_attribute_refinement_levels(oracle_mod):
    """"Scale, rotation, opacity, and colour use a base plus three learned refinements"; reading I2:
    additive residuals on log-scale / raw quaternion / opacity logit, level l applied iff depth >= l.
    Pins: zero refinements == none; depth 0 ignores them; a single on-axis isotropic Gaussian follows the P3
    closed form with s_v = s exp(sum dls), o_v = sigmoid(logit + sum dlogit); a quaternion refinement that only
    rescales the quaternion changes nothing (normalisation)."""
    import dataclasses
    wl = synth.workload_cfg0()
    sc, (cam, t) = wl.scene, wl.frames[0]
    base = oracle_mod.OracleScene(sc)
    z3 = lambda *shape: np.zeros((3, sc.N) + shape, np.float32)
    zero = oracle_mod.OracleScene(dataclasses.replace(sc, d_log_scale=z3(3), d_quat=z3(4), d_opacity_logit=z3()))
    ref = oracle_mod.OracleScene(synth.with_attribute_refinements(sc))
    # scaling the quaternion by a positive factor per level: same rotation
    dq = np.stack([0.25 * sc.quat, 0.5 * sc.quat, 1.0 * sc.quat]).astype(np.float32)
    qonly = oracle_mod.OracleScene(dataclasses.replace(sc, d_quat=dq))
    for d in range(-1, 4):
        depth = np.full(sc.C, d, np.int8)
        p0, pz, pr, pq = (o.project(cam, t, depth) for o in (base, zero, ref, qonly))
        assert p0.tobytes() == pz.tobytes()
        if d <= 0:
            assert p0.tobytes() == pr.tobytes()
        else:
            m = p0["valid"] == 1
            assert np.any(pr["cov2d"][m] != p0["cov2d"][m]) and np.any(pr["opacity"][m] != p0["opacity"][m])
        m = (p0["valid"] == 1) & (pq["valid"] == 1)
        assert np.allclose(pq["cov2d"][m], p0["cov2d"][m], rtol=2e-5, atol=1e-6)
    # closed form (P3) per depth for one isotropic Gaussian on the axis
    f, z0, s0, logit = 100.0, 4.0, 0.05, 0.3
    one, _ = tiny_scene([[0.0, 0.0, 0.0]], s0, logits=logit, colors=[0.8, 0.6, 0.4], levels=[0])
    dls = np.array([0.2, -0.1, 0.05], np.float32).reshape(3, 1, 1) * np.ones((3, 1, 3), np.float32)
    dlg = np.array([0.5, -0.25, 1.0], np.float32).reshape(3, 1)
    one = dataclasses.replace(one, d_log_scale=dls, d_opacity_logit=dlg)
    camx = axis_camera(W=64, H=64, f=f, z0=z0, cx=32.5, cy=32.5)   # pixel (32, 32) centre on the axis
    o = oracle_mod.OracleScene(one)
    for d in range(4):
        s_v = s0 * np.exp(float(dls[:d, 0, 0].astype(np.float64).sum())) if d else s0
        o_v = 1.0 / (1.0 + np.exp(-(logit + float(dlg[:d, 0].astype(np.float64).sum()))))
        img, _ = o.render(camx, 0.0, np.array([d], np.int8))
        sig2 = (f * s_v / z0) ** 2 + 0.3
        pr = o.project(camx, 0.0, np.array([d], np.int8))
        assert pr["cov2d"][0][0] == pytest.approx(sig2, rel=1e-5)
        alpha = min(0.99, o_v)                                       # at the centre exp(0) = 1
        assert img[32, 32, 0] == pytest.approx(0.8 * alpha, rel=1e-5)


def test_p19b_colour_refinement_levels(oracle_mod):
    """Reading I3: per-level SH residuals; the colour at depth v uses sh_base + levels 1..v (+ sh_res at 3).
    Degree-0 closed form: rgb = max(0, 0.5 + Y0 (sh0 + sum_{l<=v} d_l)); zero residuals == none."""
    import dataclasses
    one, _ = tiny_scene([[0.0, 0.0, 0.0]], 0.05, colors=[0.5, 0.5, 0.5], levels=[0])
    dsh = np.zeros((3, 1, 1, 3), np.float32)
    dsh[0, 0, 0] = [0.3, 0.0, -0.2]
    dsh[1, 0, 0] = [0.1, 0.2, 0.0]
    dsh[2, 0, 0] = [-3.0, 0.1, 0.1]                   # drives the red channel below zero: clamped
    o = oracle_mod.OracleScene(dataclasses.replace(one, d_sh=dsh))
    cam = axis_camera()
    for d in range(4):
        want = np.maximum(0.0, 0.5 + Y0 * dsh[:d, 0, 0].astype(np.float64).sum(axis=0))
        got = o.project(cam, 0.0, np.array([d], np.int8))["rgb"][0]
        assert np.allclose(got, want, rtol=0, atol=1e-12), (d, got, want)
    wl = synth.workload_cfg0()
    sc, (camw, t) = wl.scene, wl.frames[0]
    z = oracle_mod.OracleScene(dataclasses.replace(sc, d_sh=np.zeros((3, sc.N, sc.K, 3), np.float32)))
    b = oracle_mod.OracleScene(sc)
    for d in range(4):
        dep = np.full(sc.C, d, np.int8)
        assert z.project(camw, t, dep).tobytes() == b.project(camw, t, dep).tobytes()


def test_p20_affine_push_forward_of_covariance(oracle_mod):
    """Reading I4 (optional): Sigma_t = L Sigma L^T with L = the 3x3 part of A_{c,t}.  L = I changes nothing
    (bitwise); L = s I scales the screen variance by s^2 (closed form of P3); a 90-degree roll about the optical
    axis swaps the two screen variances of an axis-aligned anisotropic Gaussian (P7)."""
    import dataclasses
    wl = synth.workload_cfg0()
    sc, (cam, t) = wl.scene, wl.frames[0]
    ident = dataclasses.replace(sc, A1=np.zeros_like(sc.A1), affine_on_covariance=True)
    plain = dataclasses.replace(sc, A1=np.zeros_like(sc.A1))
    for d in (0, 3):
        dep = np.full(sc.C, d, np.int8)
        assert oracle_mod.OracleScene(ident).project(cam, t, dep).tobytes() == \
            oracle_mod.OracleScene(plain).project(cam, t, dep).tobytes()
    f, z0, s0 = 100.0, 4.0, 0.05
    camx = axis_camera(W=64, H=64, f=f, z0=z0)
    for scale in (0.5, 2.0):
        A0 = np.zeros((1, 3, 4)); A0[0, :, :3] = scale * np.eye(3)
        one, _ = tiny_scene([[0.0, 0.0, 0.0]], s0, levels=[0], A0=A0)
        one = dataclasses.replace(one, affine_on_covariance=True)
        pr = oracle_mod.OracleScene(one).project(camx, 0.0, np.array([0], np.int8))
        assert pr["cov2d"][0][0] == pytest.approx((f * scale * s0 / z0) ** 2 + 0.3, rel=1e-5)
    # roll by 90 degrees about z: x' = -y, y' = x
    A0 = np.zeros((1, 3, 4)); A0[0, 0, 1] = -1.0; A0[0, 1, 0] = 1.0; A0[0, 2, 2] = 1.0
    aniso, _ = tiny_scene([[0.0, 0.0, 0.0]], np.array([[0.08, 0.02, 0.05]]), levels=[0], A0=A0)
    p_off = oracle_mod.OracleScene(aniso).project(camx, 0.0, np.array([0], np.int8))
    p_on = oracle_mod.OracleScene(dataclasses.replace(aniso, affine_on_covariance=True)).project(camx, 0.0, np.array([0], np.int8))
    assert p_on["cov2d"][0][0] == pytest.approx(p_off["cov2d"][0][2], rel=1e-5)
    assert p_on["cov2d"][0][2] == pytest.approx(p_off["cov2d"][0][0], rel=1e-5)
    assert abs(p_on["cov2d"][0][1]) < 1e-4


# ------------------------------------------------------------------------------------------ P21-P24
# Pins of four constants / conventions of readings A9 and A11 that no pin above exercises (each chosen so that the
# nearest plausible mistake fails it): the SH view direction, the alpha cap, the Jacobian clamp, the lambda floor.
def pin_scene_sh_view_direction():
    """One Gaussian off the optical axis, SH degree 1 with one pure degree-1 coefficient per channel (R on the x
    term, G on the y term, B on the z term), seen by a camera whose R_wc and t_wc are both non-trivial, so that
    -R^T t (the camera centre) differs from -R t."""
    eye = np.array([1.5, -2.0, -3.0])
    R, tw = synth.look_at(eye, target=(0.2, 0.1, 0.3))
    cam = synth.make_camera(R, tw, 96, 80, 90.0)
    mu = np.array([0.5, 0.4, 0.6])
    k = 0.6
    sh = np.zeros((1, 4, 3))
    sh[0, 3, 0] = k          # basis order (1; y, z, x): index 3 is the x term
    sh[0, 1, 1] = k          # index 1 is the y term
    sh[0, 2, 2] = k          # index 2 is the z term
    scn, _ = tiny_scene([mu], 0.05, sh_degree=1, sh_base=sh)
    return scn, cam, eye, mu, k


def test_p21_sh_view_direction_is_from_the_camera_centre(oracle_mod):
    scn, cam, eye, mu, k = pin_scene_sh_view_direction()
    p = oracle_mod.OracleScene(scn).project(cam, 0.0, np.zeros(1, np.int8))[0]
    assert p["valid"] == 1
    d = mu.astype(np.float32).astype(np.float64) - eye        # Gaussian minus the camera position given to look_at
    d /= np.linalg.norm(d)
    c1 = np.sqrt(3.0 / (4.0 * np.pi))                         # degree-1 constant of the orthonormal real basis
    expect = 0.5 + c1 * k * d                                 # channel R <- x, G <- y, B <- z
    assert np.all(expect > 0.05)                              # away from the clamp at 0
    assert np.abs(p["rgb"] - expect).max() < 2e-6             # eye is exact only to the fp32 rounding of t_wc
    # what the two nearest mistakes would give is far away: centre = -R t, and the direction reversed
    Rd, td = cam.R_wc.astype(np.float64), cam.t_wc.astype(np.float64)
    wrong = mu - (-(Rd @ td))
    wrong /= np.linalg.norm(wrong)
    assert np.abs(0.5 + c1 * k * wrong - expect).max() > 0.05
    assert np.abs((0.5 - c1 * k * d) - expect).max() > 0.05


def pin_scene_alpha_cap(bg):
    col = (0.8, 0.3, 0.6)
    scn, _ = tiny_scene([[0, 0, 0]], 0.2, logits=8.0, colors=col, background=bg)      # o = 0.99966 > 0.99
    cam = axis_camera(64, 64, 100.0, 4.0, cx=32.5, cy=32.5)                           # pixel (32,32) centred on the axis
    return scn, cam, col


@pytest.mark.parametrize("bg", [(0.0, 0.0, 0.0), (1.0, 1.0, 1.0)])
def test_p22_alpha_is_capped_at_0_99(oracle_mod, bg):
    scn, cam, col = pin_scene_alpha_cap(bg)
    sc = oracle_mod.OracleScene(scn)
    for brute in (False, True):
        img, _ = sc.render(cam, 0.0, np.zeros(1, np.int8), brute_force=brute)
        # q = 0 at the centre pixel: alpha = min(0.99, 0.99966) = 0.99; T' = 0.01 >= 1e-4, so it is added
        expect = 0.99 * np.array(col) + 0.01 * np.array(bg)
        assert np.abs(img[32, 32] - expect).max() < 1e-6
        # uncapped (0.99966) or capped at 0.999 the pixel would move by > 3e-3 times |c - bg|
        assert np.abs((0.999 * np.array(col) + 0.001 * np.array(bg)) - expect).max() > 1e-3


def pin_scene_jacobian_clamp():
    """A large isotropic Gaussian at x/z = 2 lim_x (lim_x = 1.3 (W/2)/fx), in front of the near plane; it is big
    enough (3 sigma' ~ 59 px) for its footprint to reach the screen, so the record is valid."""
    W, H, f, z = 64, 64, 50.0, 4.0
    lim = 1.3 * 0.5 * W / f
    s = 1.2
    scn, _ = tiny_scene([[2.0 * lim * z, 0.0, 0.0]], s)
    return scn, axis_camera(W, H, f, z), lim, s, f, z


def test_p23_jacobian_uses_the_clamped_point(oracle_mod):
    scn, cam, lim, s, f, z = pin_scene_jacobian_clamp()
    p = oracle_mod.OracleScene(scn).project(cam, 0.0, np.zeros(1, np.int8))[0]
    assert p["valid"] == 1
    x = float(np.float32(2.0 * lim * z))

    def cov(xt):       # Sigma' = s^2 J J^T + 0.3 I with J = [[f/z, 0, -f xt/z^2], [0, f/z, 0]]  (R_wc = I, Sigma = s^2 I)
        J = np.array([[f / z, 0.0, -f * xt / z ** 2], [0.0, f / z, 0.0]])
        return s * s * J @ J.T + 0.3 * np.eye(2)
    clamped, unclamped = cov(lim * z), cov(x)
    assert unclamped[0, 0] > 2.0 * clamped[0, 0]                       # the two readings are far apart
    assert np.allclose(p["cov2d"], [clamped[0, 0], clamped[0, 1], clamped[1, 1]], rtol=2e-5)
    # the 2-D mean is NOT clamped: it sits at cx + f x / z
    assert abs(p["mx"] - (cam.cx + f * x / z)) < 1e-3
    # a clamp at 1.0 lim instead of 1.3 lim: lim_x = 0.64 gives a visibly different Sigma'_00
    wrong = cov((lim / 1.3) * z)
    assert abs(wrong[0, 0] - clamped[0, 0]) > 0.1 * clamped[0, 0]


def pin_scene_lambda_floor():
    f, z0 = 100.0, 4.0
    s = np.sqrt(1.4) * z0 / f        # sigma'^2 = 1.4 + 0.3 = 1.7, isotropic: mid^2 - det = 0 < 0.1
    scn, _ = tiny_scene([[0, 0, 0]], s)
    return scn, axis_camera(128, 128, f, z0)


def test_p24_lambda_floor_sets_the_radius(oracle_mod):
    scn, cam = pin_scene_lambda_floor()
    p = oracle_mod.OracleScene(scn).project(cam, 0.0, np.zeros(1, np.int8))[0]
    # by hand: lambda = 1.7 + sqrt(0.1) = 2.0162 ; 3 sqrt(lambda) = 4.2598 -> radius 5
    # without the floor: 3 sqrt(1.7) = 3.9115 -> radius 4
    assert np.ceil(3 * np.sqrt(1.7)) == 4 and np.ceil(3 * np.sqrt(1.7 + np.sqrt(0.1))) == 5
    assert p["radius"] == 5
    # rectangle from radius 5 around (64, 64): floor(59/16) = 3 .. floor((69+15)/16) = 5
    assert p["rect"].tolist() == [3, 3, 5, 5]

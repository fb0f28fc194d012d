"""Pins of the projection-backward oracle (oracle/gsr_oracle.c O-9: from the gradient with respect to the 2-D
quantities of a Gaussian in one state to the gradient with respect to the scene's own parameters).
CPU-only.  Pinned against what does not share its formulas: central finite differences of the FORWARD oracle
(O-0 activation + O-2 deformation + O-3 projection and colour, pinned themselves by P1..P24) under perturbed scene
parameters, closed forms for the on-axis isotropic Gaussian, finite differences of the exported SH basis, and the
invariants of the parameterisation (a quaternion's length, an isotropic Gaussian's rotation)."""
import dataclasses

import numpy as np
import pytest

from paper_2606_17212_b200 import synth
from tests.helpers import Y0, axis_camera, tiny_scene

OUT = ["rgb0", "rgb1", "rgb2", "opacity", "qa", "qb", "qc", "mx", "my"]


def outputs(p):
    """[N, 9] double: the nine 2-D quantities O-8 differentiates, from a projection record array."""
    return np.concatenate([np.asarray(p["rgb"], np.float64), np.stack([p[k].astype(np.float64) for k in OUT[3:]], 1)], 1)


def small_workload():
    """The cfg1 recipe at 3 clusters x ~30 Gaussians (SH degree 3, R = 8, time-dependent cluster affine, motion
    residual), a camera off every axis, t = 0.37."""
    wl = synth.scaled_object_workload(41, C=3, per_cluster=30.0, W=96, H=64, fov=40.0, n_frames=1, B=2)
    return wl.scene, wl.frames[0][0], 0.37


def functional(oracle_mod, scn, cam, t, depth, w, valid0=None):
    sc = oracle_mod.OracleScene(scn)
    p = sc.project(cam, t, depth)
    if valid0 is not None:
        assert np.array_equal(p["valid"], valid0)          # the perturbation flips no discrete decision
    v = p["valid"] == 1
    return float((w[v] * outputs(p)[v]).sum()), p


# name of the Scene field, name of the gradient, step (the forward oracle is fp32: steps well above its rounding)
FAMILIES = [("mean", "mean", 4e-3), ("log_scale", "log_scale", 1e-2), ("quat", "quat", 1e-2),
            ("opacity_logit", "opacity_logit", 2e-2), ("sh_base", "sh_base", 2e-2), ("sh_res", "sh_res", 2e-2),
            ("motion_scale", "motion_scale", None), ("A0", "A", 4e-3), ("A1", "A", 4e-3)]


@pytest.mark.parametrize("d", [0, 1, 3])
def test_c1_directional_derivatives_match_central_differences_of_the_forward_oracle(oracle_mod, d):
    scn, cam, t = small_workload()
    depth = np.full(scn.C, d, np.int8)
    rng = np.random.default_rng(100 + d)
    w = rng.standard_normal((scn.N, 9))
    L0, p0 = functional(oracle_mod, scn, cam, t, depth, w)
    valid0 = p0["valid"].copy()
    assert valid0.sum() >= 0.5 * (scn.level_of() <= d).sum() > 10
    sc = oracle_mod.OracleScene(scn)
    g9 = np.where((valid0 == 1)[:, None], w, 0.0)
    grads = sc.project_backward(cam, t, depth, g9)
    assert grads["margin"][valid0 == 1].min() > 1e-3          # every decision is far from its threshold
    for field, gname, h in FAMILIES:
        theta = np.asarray(getattr(scn, field), np.float32)
        for trial in range(3):
            u = rng.standard_normal(theta.shape)
            if h is None:                                     # motion_scale ~ 1e-4: a relative step
                step = 0.05 * theta.astype(np.float64) * u
            else:
                step = h * u
            tp = (theta.astype(np.float64) + step).astype(np.float32)
            tm = (theta.astype(np.float64) - step).astype(np.float32)
            delta = tp.astype(np.float64) - tm.astype(np.float64)    # the step actually taken in fp32
            Lp, _ = functional(oracle_mod, dataclasses.replace(scn, **{field: tp}), cam, t, depth, w, valid0)
            Lm, _ = functional(oracle_mod, dataclasses.replace(scn, **{field: tm}), cam, t, depth, w, valid0)
            g = grads[gname].reshape(theta.shape).copy()
            if field == "A1":
                g = t * g                                      # A_c(t) = A0 + t A1
            pred = float((g * delta).sum())
            fd = Lp - Lm
            mag = float(np.abs(g * delta).sum())
            # fp32 forward: ~1e-7 relative noise on values of size |L| ~ sum |w f|; central differences: O(h^2)
            assert abs(fd - pred) <= 5e-3 * mag + 1e-4 * abs(fd) + 2e-3, (field, trial, fd, pred, mag)
        if d == 0 and field in ("sh_res", "motion_scale"):
            assert np.all(grads[gname] == 0.0)                 # not applied at depth 0
    if d == 0:
        assert np.all(grads["rho"] == 0.0)
    if d < 3:
        assert np.all(grads["sh_res"] == 0.0)


def test_c2_single_coordinates_and_the_motion_residual(oracle_mod):
    """Coordinate by coordinate for three Gaussians (a wrong index or a transposition moves a single entry), and the
    motion residual rho through an int8 step of q: L(q + e) - L(q - e) = 2 s_c b_r g_rho to second order."""
    scn, cam, t = small_workload()
    depth = np.full(scn.C, 2, np.int8)
    rng = np.random.default_rng(7)
    w = rng.standard_normal((scn.N, 9))
    L0, p0 = functional(oracle_mod, scn, cam, t, depth, w)
    valid0 = p0["valid"].copy()
    sc = oracle_mod.OracleScene(scn)
    grads = sc.project_backward(cam, t, depth, np.where((valid0 == 1)[:, None], w, 0.0))
    picks = np.nonzero(valid0 == 1)[0][[0, 7, 19]]
    for field, h in (("mean", 4e-3), ("log_scale", 1e-2), ("quat", 1e-2)):
        theta = np.asarray(getattr(scn, field), np.float32)
        for i in picks:
            for k in range(theta.shape[1]):
                tp, tm = theta.copy(), theta.copy()
                tp[i, k] += h
                tm[i, k] -= h
                hh = float(tp[i, k]) - float(tm[i, k])
                Lp, _ = functional(oracle_mod, dataclasses.replace(scn, **{field: tp}), cam, t, depth, w, valid0)
                Lm, _ = functional(oracle_mod, dataclasses.replace(scn, **{field: tm}), cam, t, depth, w, valid0)
                fd = (Lp - Lm) / hh
                ref = grads[field][i, k]
                scale = np.abs(grads[field][i]).max()
                assert abs(fd - ref) <= 5e-3 * scale + 2e-3 / hh * 1e-2, (field, i, k, fd, ref)
    basis = oracle_mod.basis(t, scn.R).astype(np.float64)
    cl = scn.cluster_of()
    for i in picks:
        for r in (0, 3):
            for k in range(3):
                qp, qm = scn.motion_q.copy(), scn.motion_q.copy()
                qp[i, r, k] = min(127, int(qp[i, r, k]) + 4)
                qm[i, r, k] = max(-127, int(qm[i, r, k]) - 4)
                dq = int(qp[i, r, k]) - int(qm[i, r, k])
                Lp, _ = functional(oracle_mod, dataclasses.replace(scn, motion_q=qp), cam, t, depth, w, valid0)
                Lm, _ = functional(oracle_mod, dataclasses.replace(scn, motion_q=qm), cam, t, depth, w, valid0)
                pred = float(scn.motion_scale[cl[i]]) * basis[r] * dq * grads["rho"][i, k]
                scale = float(scn.motion_scale[cl[i]]) * abs(basis[r]) * abs(dq) * np.abs(grads["rho"][i]).max()
                assert abs((Lp - Lm) - pred) <= 2e-2 * scale + 2e-4, (i, r, k, Lp - Lm, pred)


def test_c3_closed_forms_on_axis_isotropic_gaussian(oracle_mod):
    """One isotropic Gaussian (sigma) at depth z0 on the optical axis, R_wc = I, degree-0 colour: m_x = fx x / z + cx,
    Sigma' = (f sigma / z)^2 I + 0.3 I, A = Cq = 1 / (2 (f^2 sigma^2 / z^2 + 0.3)), B = 0, o = sigmoid(logit),
    rgb = 0.5 + Y0 c.  Their derivatives at x = y = 0, by hand."""
    f, z0, sg, logit = 120.0, 5.0, 0.4, 0.7
    scn, _ = tiny_scene([[0, 0, 0]], sg, logits=logit, colors=(0.8, 0.3, 0.6))
    cam = axis_camera(64, 64, f, z0)
    sc = oracle_mod.OracleScene(scn)
    depth = np.zeros(1, np.int8)
    o = 1.0 / (1.0 + np.exp(-logit))
    s2 = (f * sg / z0) ** 2 + 0.3                              # a = c
    for k, expect in [
        (7, {"mean": [f / z0, 0, 0]}),                         # dm_x/dx = f / z; no dependence on y, z at x = 0
        (8, {"mean": [0, f / z0, 0]}),
        (3, {"opacity_logit": o * (1 - o)}),
        # A = 1 / (2 a), a = f^2 sigma^2 / z^2 + 0.3: dA/dlog sigma_x = -(1 / (2 a^2)) 2 (f sigma / z)^2 (x scale only
        # enters s00), dA/dz = -(1 / (2 a^2)) (-2 f^2 sigma^2 / z^3)
        (4, {"log_scale": [-(f * sg / z0) ** 2 / s2 ** 2, 0, 0], "mean": [0, 0, (f * sg) ** 2 / z0 ** 3 / s2 ** 2]}),
        (6, {"log_scale": [0, -(f * sg / z0) ** 2 / s2 ** 2, 0], "mean": [0, 0, (f * sg) ** 2 / z0 ** 3 / s2 ** 2]}),
        (0, {"sh_base": [[Y0, 0, 0]]}),
    ]:
        g9 = np.zeros((1, 9))
        g9[0, k] = 1.0
        gr = sc.project_backward(cam, 0.0, depth, g9)
        for name, val in expect.items():
            assert np.allclose(np.asarray(gr[name]).reshape(np.shape(val)), val, rtol=1e-5, atol=1e-9), (OUT[k], name, gr[name])
        assert np.allclose(gr["quat"], 0.0, atol=1e-9)         # isotropic: the rotation does not matter
        assert np.all(gr["rho"] == 0.0) and np.all(gr["sh_res"] == 0.0)
    # B = -b / det: db/d(x) at x = 0 is 0 by symmetry, but d(B)/d(mean_x) of an OFF-axis Gaussian is not — covered by c1


def test_c4_sh_basis_gradient_against_finite_differences_of_the_basis(oracle_mod):
    rng = np.random.default_rng(3)
    for _ in range(5):
        v = rng.standard_normal(3)
        G = oracle_mod.sh_basis_grad(16, v)
        h = 1e-6
        for a in range(3):
            e = np.zeros(3)
            e[a] = h
            fd = (oracle_mod.sh_basis(16, v + e) - oracle_mod.sh_basis(16, v - e)) / (2 * h)
            assert np.allclose(G[a], fd, rtol=1e-7, atol=1e-8)
        for K in (1, 4, 9):
            assert np.array_equal(oracle_mod.sh_basis_grad(K, v), G[:, :K])


def test_c5_invariants_of_the_parameterisation(oracle_mod):
    scn, cam, t = small_workload()
    depth = np.array([3, 1, 0], np.int8)
    rng = np.random.default_rng(9)
    sc = oracle_mod.OracleScene(scn)
    p = sc.project(cam, t, depth)
    g9 = np.where((p["valid"] == 1)[:, None], rng.standard_normal((scn.N, 9)), 0.0)
    gr = sc.project_backward(cam, t, depth, g9)
    # scaling a quaternion changes nothing: its gradient is orthogonal to it
    dots = (gr["quat"] * scn.quat.astype(np.float64)).sum(1)
    assert np.all(np.abs(dots) <= 1e-12 * np.abs(gr["quat"]).sum(1) + 1e-18)
    # the translation column of A_c(t) moves every Gaussian of the cluster alike: it collects dL/dp, and so does
    # mean through the linear part: g_mean = L^T dL/dp
    cl = scn.cluster_of()
    A = scn.A0.astype(np.float64) + float(np.float32(t)) * scn.A1.astype(np.float64)   # t travels as binary32
    for c in range(scn.C):
        dp = np.linalg.solve(A[c, :, :3].T, gr["mean"][cl == c].T).T          # dL/dp per Gaussian
        assert np.allclose(dp.sum(0), gr["A"][c, :, 3], rtol=1e-9, atol=1e-12)
        assert np.allclose(dp.T @ scn.mean[cl == c].astype(np.float64), gr["A"][c, :, :3], rtol=1e-9, atol=1e-12)
    # where the residual applies (depth >= 1) rho and p move the mean alike: g_rho = dL/dp; at depth 0 g_rho = 0
    dp1 = np.linalg.solve(A[1, :, :3].T, gr["mean"][cl == 1].T).T
    assert np.allclose(gr["rho"][cl == 1], dp1, rtol=1e-9, atol=1e-12)
    assert np.all(gr["rho"][cl == 2] == 0.0) and gr["motion_scale"][2] == 0.0
    # the SH residual only at depth 3; absent Gaussians (level > depth) get nothing at all
    assert np.any(gr["sh_res"][cl == 0] != 0.0) and np.all(gr["sh_res"][cl != 0] == 0.0)
    gone = scn.level_of() > depth[cl]
    assert gone.any()
    for name in ("mean", "rho", "log_scale", "quat", "opacity_logit", "sh_base", "sh_res"):
        assert np.all(gr[name][gone] == 0.0)
    # linear in g9, and accumulating
    g2 = sc.project_backward(cam, t, depth, 2.0 * g9)
    acc = sc.project_backward(cam, t, depth, g9, into=sc.project_backward(cam, t, depth, g9))
    for name in oracle_mod.OracleScene.PARAM_GRADS:
        assert np.allclose(g2[name], 2.0 * gr[name], rtol=1e-12, atol=1e-300)
        assert np.allclose(acc[name], 2.0 * gr[name], rtol=1e-12, atol=1e-300)


def test_c6_clamped_jacobian_and_clamped_colour_pass_no_gradient(oracle_mod):
    """(a) A Gaussian beyond 1.3 lim_x: x~ = lim_x z no longer depends on x, so dSigma'/dx only has the m_x path —
    finite differences of the forward oracle agree with O-9 there too, and differ from the unclamped formula.
    (b) A colour channel below zero (rgb = max(0, .) = 0) passes nothing to its coefficients nor to the mean."""
    f, z0 = 100.0, 4.0
    cam = axis_camera(64, 64, f, z0)
    limx = 0.5 * 64 / f * 1.3
    xg = 1.5 * limx * z0
    scn, _ = tiny_scene([[xg, 0.1, 0.0]], [0.3, 0.2, 0.25], quats=[[1, 0.2, 0.1, -0.3]], logits=0.5, colors=(0.8, 0.3, 0.6))
    sc = oracle_mod.OracleScene(scn)
    depth = np.zeros(1, np.int8)
    p0 = sc.project(cam, 0.0, depth)
    # the Gaussian is off screen (its rectangle is empty -> valid 0) but O-3 has projected it: use its record fields
    w = np.zeros((1, 9))
    w[0, 4:7] = [1.0, -0.7, 0.4]                                # a functional of the conic only
    gr = sc.project_backward(cam, 0.0, depth, w)
    conic = lambda q: float(w[0, 4] * q["qa"][0] + w[0, 5] * q["qb"][0] + w[0, 6] * q["qc"][0])
    assert p0["qa"][0] != 0.0
    for k, h in ((0, 2e-3), (2, 2e-3)):
        mp, mm = scn.mean.copy(), scn.mean.copy()
        mp[0, k] += h
        mm[0, k] -= h
        qp = oracle_mod.OracleScene(dataclasses.replace(scn, mean=mp)).project(cam, 0.0, depth)
        qm = oracle_mod.OracleScene(dataclasses.replace(scn, mean=mm)).project(cam, 0.0, depth)
        fd = (conic(qp) - conic(qm)) / (float(mp[0, k]) - float(mm[0, k]))
        assert abs(fd - gr["mean"][0, k]) <= 5e-3 * abs(gr["mean"][0]).max() + 1e-7, (k, fd, gr["mean"][0])
    assert abs(gr["mean"][0, 0]) < 1e-12                       # clamped: the conic does not depend on x at all
    # (b)
    scn, _ = tiny_scene([[0.1, 0.07, 0.0]], 0.3, logits=0.5, colors=(0.8, -0.2, 0.6), sh_degree=1,
                        sh_base=np.array([[[0.3 / Y0, -0.7 / Y0, 0.1 / Y0], [0.1, 0.2, 0.3], [0.2, 0.1, 0.1], [0.3, 0.3, 0.2]]]))
    sc = oracle_mod.OracleScene(scn)
    p = sc.project(cam, 0.0, depth)
    assert p["rgb"][0][1] == 0.0 and p["rgb"][0][0] > 0.0
    g9 = np.zeros((1, 9))
    g9[0, 1] = 1.0                                              # the clamped channel only
    gr = sc.project_backward(cam, 0.0, depth, g9)
    assert np.all(gr["sh_base"] == 0.0) and np.all(gr["mean"] == 0.0)
    g9[0, 0] = 1.0
    gr = sc.project_backward(cam, 0.0, depth, g9)
    assert np.all(gr["sh_base"][0, :, 1] == 0.0) and np.all(gr["sh_base"][0, :, 0] != 0.0) and np.any(gr["mean"] != 0.0)


def test_c7_colour_only_functional_isolates_the_view_direction_path(oracle_mod):
    """With weights on rgb only, the mean receives gradient through dir = (mu - centre) / |.| alone (two orders of
    magnitude below the projection path, invisible in c1): SH degree 3 colours against central differences."""
    scn, cam, t = small_workload()
    depth = np.full(scn.C, 3, np.int8)
    rng = np.random.default_rng(21)
    w = np.zeros((scn.N, 9))
    w[:, :3] = rng.standard_normal((scn.N, 3))
    L0, p0 = functional(oracle_mod, scn, cam, t, depth, w)
    valid0 = p0["valid"].copy()
    sc = oracle_mod.OracleScene(scn)
    grads = sc.project_backward(cam, t, depth, np.where((valid0 == 1)[:, None], w, 0.0))
    assert np.all(grads["log_scale"] == 0.0) and np.all(grads["quat"] == 0.0) and np.all(grads["opacity_logit"] == 0.0)
    theta = scn.mean
    for trial in range(4):
        u = rng.standard_normal(theta.shape)
        tp = (theta.astype(np.float64) + 2e-2 * u).astype(np.float32)
        tm = (theta.astype(np.float64) - 2e-2 * u).astype(np.float32)
        delta = tp.astype(np.float64) - tm.astype(np.float64)
        Lp, _ = functional(oracle_mod, dataclasses.replace(scn, mean=tp), cam, t, depth, w, valid0)
        Lm, _ = functional(oracle_mod, dataclasses.replace(scn, mean=tm), cam, t, depth, w, valid0)
        pred = float((grads["mean"] * delta).sum())
        mag = float(np.abs(grads["mean"] * delta).sum())
        assert mag > 1e-3
        assert abs((Lp - Lm) - pred) <= 5e-3 * mag, (trial, Lp - Lm, pred, mag)
    # moving a mean along its own view direction does not change the direction: the gradient is orthogonal to it
    centre = -(cam.R_wc.astype(np.float64).T @ cam.t_wc.astype(np.float64))
    pmu = p0["mu"].astype(np.float64)
    v = pmu - centre
    A = scn.A0.astype(np.float64) + float(np.float32(t)) * scn.A1.astype(np.float64)
    cl = scn.cluster_of()
    for i in np.nonzero(valid0 == 1)[0][:10]:
        dmu = np.linalg.solve(A[cl[i], :, :3].T, grads["mean"][i])
        assert abs(dmu @ v[i]) <= 1e-5 * np.linalg.norm(dmu) * np.linalg.norm(v[i])


FULL_FAMILIES = [("mean", "mean", 4e-3), ("log_scale", "log_scale", 1e-2), ("quat", "quat", 1e-2),
                 ("opacity_logit", "opacity_logit", 2e-2), ("sh_base", "sh_base", 2e-2), ("sh_res", "sh_res", 2e-2),
                 ("A0", "A", 4e-3), ("A1", "A", 4e-3),
                 ("delta2", "delta2", 4e-3), ("delta3", "delta3", 4e-3), ("d_log_scale", "d_log_scale", 1e-2),
                 ("d_quat", "d_quat", 1e-2), ("d_opacity_logit", "d_opacity_logit", 2e-2), ("d_sh", "d_sh", 2e-2)]


@pytest.mark.parametrize("affine", [False, True])
def test_c8_full_representation_against_central_differences(oracle_mod, affine):
    """The rest of the representation: position residual levels, per-level scale / rotation / opacity /
    colour refinements and, optionally, the affine on the covariance — a mixed state (cluster depths 3, 2, 1) so that
    every level's residual is applied by some cluster and skipped by another."""
    base, cam, t = small_workload()
    scn = synth.with_attribute_refinements(synth.with_position_residuals(base))
    scn = dataclasses.replace(scn, affine_on_covariance=affine)
    depth = np.array([3, 2, 1], np.int8)
    rng = np.random.default_rng(300 + int(affine))
    w = rng.standard_normal((scn.N, 9))
    L0, p0 = functional(oracle_mod, scn, cam, t, depth, w)
    valid0 = p0["valid"].copy()
    assert valid0.sum() > 20
    sc = oracle_mod.OracleScene(scn)
    grads = sc.project_backward(cam, t, depth, np.where((valid0 == 1)[:, None], w, 0.0))
    assert grads["margin"][valid0 == 1].min() > 1e-3
    for field, gname, h in FULL_FAMILIES:
        theta = np.asarray(getattr(scn, field), np.float32)
        for trial in range(2):
            u = rng.standard_normal(theta.shape)
            tp = (theta.astype(np.float64) + h * u).astype(np.float32)
            tm = (theta.astype(np.float64) - h * u).astype(np.float32)
            delta = tp.astype(np.float64) - tm.astype(np.float64)
            Lp, _ = functional(oracle_mod, dataclasses.replace(scn, **{field: tp}), cam, t, depth, w, valid0)
            Lm, _ = functional(oracle_mod, dataclasses.replace(scn, **{field: tm}), cam, t, depth, w, valid0)
            g = grads[gname].reshape(theta.shape).copy()
            if field == "A1":
                g = t * g
            pred = float((g * delta).sum())
            mag = float(np.abs(g * delta).sum())
            assert mag > 0.0
            assert abs((Lp - Lm) - pred) <= 5e-3 * mag + 1e-4 * abs(Lp - Lm) + 2e-3, (field, trial, Lp - Lm, pred, mag)
    # which states feed which level: cluster 0 (depth 3) feeds all three levels, cluster 1 (depth 2) levels 1-2,
    # cluster 2 (depth 1) level 1 only; delta3 only from cluster 0, delta2 from clusters 0 and 1
    cl = scn.cluster_of()
    live = valid0 == 1
    for name in ("d_log_scale", "d_quat", "d_opacity_logit", "d_sh"):
        g = grads[name].reshape(3, scn.N, -1)
        assert np.any(g[2][(cl == 0) & live] != 0.0) and np.all(g[2][cl != 0] == 0.0)
        assert np.any(g[1][(cl == 1) & live] != 0.0) and np.all(g[1][cl == 2] == 0.0)
        assert np.any(g[0][(cl == 2) & live] != 0.0)
    assert np.all(grads["delta3"][cl != 0] == 0.0) and np.any(grads["delta3"][cl == 0] != 0.0)
    assert np.all(grads["delta2"][cl == 2] == 0.0) and np.any(grads["delta2"][cl == 1] != 0.0)
    # a residual that is applied moves mu exactly like rho does
    assert np.allclose(grads["delta2"][cl == 1], grads["rho"][cl == 1], rtol=1e-12, atol=0.0)
    # base attribute gradient = the sum over all depths; level-1 residual = the same here (every cluster has depth >= 1)
    assert np.allclose(grads["d_log_scale"][0], grads["log_scale"], rtol=1e-12, atol=0.0)


def test_c9_affine_on_the_covariance_isolated_on_the_conic(oracle_mod):
    """Reading I4 with a cluster affine far from the identity (linear part I + 0.3 N(0,1) + t A1) and a functional
    of the conic alone (values ~0.1, so the forward oracle's fp32 noise is ~1e-6 and the bar has no room for a missing
    4 % term): the covariance path into A (dL/dL = (G + G^T) L Sigma) and into scale / rotation (dL/dSigma = L^T G L)."""
    base, cam, t = small_workload()
    rng = np.random.default_rng(77)
    A0 = base.A0.copy()
    A0[:, :, :3] += (0.3 * rng.standard_normal((base.C, 3, 3))).astype(np.float32)
    scn = dataclasses.replace(synth.with_attribute_refinements(base), A0=A0, affine_on_covariance=True)
    depth = np.array([3, 1, 2], np.int8)
    w = np.zeros((scn.N, 9))
    w[:, 4:7] = rng.standard_normal((scn.N, 3))
    L0, p0 = functional(oracle_mod, scn, cam, t, depth, w)
    valid0 = p0["valid"].copy()
    assert valid0.sum() > 20
    sc = oracle_mod.OracleScene(scn)
    grads = sc.project_backward(cam, t, depth, np.where((valid0 == 1)[:, None], w, 0.0))
    for field, gname, h in (("A0", "A", 2e-3), ("A1", "A", 4e-3), ("log_scale", "log_scale", 5e-3), ("quat", "quat", 5e-3),
                            ("d_log_scale", "d_log_scale", 5e-3), ("d_quat", "d_quat", 5e-3), ("mean", "mean", 2e-3)):
        theta = np.asarray(getattr(scn, field), np.float32)
        for trial in range(3):
            u = rng.standard_normal(theta.shape)
            if field in ("A0", "A1") and trial == 0:
                u[:, :, 3] = 0.0                                # the linear part alone
            tp = (theta.astype(np.float64) + h * u).astype(np.float32)
            tm = (theta.astype(np.float64) - h * u).astype(np.float32)
            delta = tp.astype(np.float64) - tm.astype(np.float64)
            Lp, _ = functional(oracle_mod, dataclasses.replace(scn, **{field: tp}), cam, t, depth, w, valid0)
            Lm, _ = functional(oracle_mod, dataclasses.replace(scn, **{field: tm}), cam, t, depth, w, valid0)
            g = grads[gname].reshape(theta.shape).copy()
            if field == "A1":
                g = t * g
            pred = float((g * delta).sum())
            mag = float(np.abs(g * delta).sum())
            assert abs((Lp - Lm) - pred) <= 5e-3 * mag + 1e-5, (field, trial, Lp - Lm, pred, mag)


def test_c10_colour_refinement_levels_respect_the_clamp_and_the_depth(oracle_mod):
    """One Gaussian with a channel below zero (rgb = max(0, .) = 0) and per-level colour residuals, at depth 2: the
    clamped channel passes nothing to any level; the live channel passes the same row Y_j to sh_base and to the
    residuals of levels 1 and 2 — and nothing to level 3, which this state does not contain, nor to sh_res."""
    cam = axis_camera(64, 64, 100.0, 4.0)
    scn, _ = tiny_scene([[0.1, 0.07, 0.0]], 0.3, logits=0.5, sh_degree=1,
                        sh_base=np.array([[[0.3 / Y0, -0.7 / Y0, 0.1 / Y0], [0.1, 0.2, 0.3], [0.2, 0.1, 0.1], [0.3, 0.3, 0.2]]]))
    dsh = np.zeros((3, 1, 4, 3), np.float32)
    dsh[:, 0, :, :] = 0.002 * np.arange(1, 37, dtype=np.float32).reshape(3, 4, 3)
    scn = dataclasses.replace(scn, d_sh=dsh)
    sc = oracle_mod.OracleScene(scn)
    depth = np.full(1, 2, np.int8)
    p = sc.project(cam, 0.0, depth)
    assert p["rgb"][0][1] == 0.0 and p["rgb"][0][0] > 0.0
    g9 = np.zeros((1, 9))
    g9[0, 1] = 1.0                                              # the clamped channel only
    gr = sc.project_backward(cam, 0.0, depth, g9)
    assert np.all(gr["d_sh"] == 0.0) and np.all(gr["sh_base"] == 0.0) and np.all(gr["mean"] == 0.0)
    g9[0, 0] = 1.0
    gr = sc.project_backward(cam, 0.0, depth, g9)
    assert np.all(gr["sh_base"][0, :, 0] != 0.0) and np.all(gr["sh_base"][0, :, 1] == 0.0)
    assert np.array_equal(gr["d_sh"][0][0], gr["sh_base"][0]) and np.array_equal(gr["d_sh"][1][0], gr["sh_base"][0])
    assert np.all(gr["d_sh"][2] == 0.0) and np.all(gr["sh_res"] == 0.0)
    # the rows are Y_j(dir) g: against the exported basis at the Gaussian's view direction
    centre = -(cam.R_wc.astype(np.float64).T @ cam.t_wc.astype(np.float64))
    v = p["mu"][0].astype(np.float64) - centre
    Y = oracle_mod.sh_basis(4, v / np.linalg.norm(v))
    assert np.allclose(gr["sh_base"][0, :, 0], Y, rtol=1e-12, atol=0.0)

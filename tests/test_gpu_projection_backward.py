"""GPU parity of gsr_project_backward (include/gsr.h) against the projection-backward oracle (O-9)
through the C ABI: from per-record gradients to the gradients with respect to the scene's parameters.
fp32 recomputation of the projection against a double oracle: by tolerance, stated per test."""
import numpy as np
import pytest

from paper_2606_17212_b200 import synth

pytestmark = pytest.mark.gpu

GAUSS = [("mean", 0, 3), ("rho", 3, 6), ("log_scale", 6, 9), ("quat", 9, 13), ("opacity_logit", 13, 14)]


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


def oracle_from_records(oracle_mod, scn, cam, t, grad_rec):
    """grad_rec double [2N, 12] -> the oracle's parameter gradients: the records of a 2-variant scene are three
    pseudo-states of the oracle (it differentiates one state at a time and accumulates): depth 0 (record 2 i: first
    colour and geometry), depth 3 (record 2 i + 1: second colour and geometry — every Gaussian is present) and
    depth 2 (record 2 i + 1: first colour only; a level-3 Gaussian is never composited with the first colour, so
    the callers below zero those entries, as gsr_render_backward leaves them)."""
    osc = oracle_mod.OracleScene(scn)
    N = scn.N
    gA, gB = grad_rec[0::2], grad_rec[1::2]
    out = None
    for d, g9 in ((0, np.concatenate([gA[:, 0:3], gA[:, 6:12]], 1)),
                  (3, np.concatenate([gB[:, 3:6], gB[:, 6:12]], 1)),
                  (2, np.concatenate([gB[:, 0:3], np.zeros((N, 6))], 1))):
        out = osc.project_backward(cam, t, np.full(scn.C, d, np.int8), np.ascontiguousarray(g9), into=out)
    return out


def random_records(scn, rng):
    g = rng.standard_normal((2 * scn.N, 12)).astype(np.float32).astype(np.float64)
    lvl = scn.level_of()
    g[1::2][lvl == 3, 0:3] = 0.0          # see oracle_from_records
    g[0::2][lvl != 0] = 0.0               # record 2 i exists for level-0 Gaussians only
    return g


def compare(scn, got, want, tol=2e-4, floor=0.0):
    """Per Gaussian and parameter block: |gpu - oracle| <= tol * (largest entry of the block) — the kernel recomputes
    the projection in fp32 (~1e-6 per factor through a 2x2 inverse conditioned by the 0.3 dilation) and the blocks'
    entries are of one scale.  Gaussians with a decision within 1e-4 (relative) of its threshold are skipped: the
    two sides take decisions in different precisions there.  Per-cluster sums: against the summed magnitudes.
    floor > 0 (the chain test): plus floor * (the median over Gaussians of the block's largest entry) — the
    compositor's backward leaves ABSOLUTE errors on entries that are small by cancellation."""
    ok = want["margin"] > 1e-4
    assert ok.mean() > 0.97
    gg = got["gauss"].double().cpu().numpy()
    for name, lo, hi in GAUSS:
        w = want[name].reshape(scn.N, -1)
        err = np.abs(gg[:, lo:hi] - w)
        bmax = np.abs(w).max(1, keepdims=True)
        bound = tol * bmax + floor * np.median(bmax[bmax > 0]) + 1e-12
        bad = (err > bound) & ok[:, None]
        assert not bad.any(), (name, np.argwhere(bad)[:4], err[bad][:4], w[bad][:4])
    for name in ("sh_base", "sh_res"):
        g = got[name].double().cpu().numpy()
        err = np.abs(g - want[name])
        bmax = np.abs(want[name]).max((1, 2), keepdims=True)
        bound = tol * bmax + floor * (np.median(bmax[bmax > 0]) if (bmax > 0).any() else 0.0) + 1e-12
        bad = (err > bound) & ok[:, None, None]
        assert not bad.any(), (name, np.argwhere(bad)[:4])
    # clusters: a sum over the cluster's Gaussians (atomics); magnitude of the summed terms from the oracle's rows
    cl = scn.cluster_of()
    gc = got["cluster"].double().cpu().numpy()
    wc = np.concatenate([want["A"].reshape(scn.C, 12), want["motion_scale"][:, None]], 1)
    for c in range(scn.C):
        if not ok[cl == c].all():
            continue
        mag = np.abs(want["mean"][cl == c]).sum() * max(1.0, np.abs(scn.mean[cl == c]).max())
        assert np.all(np.abs(gc[c, :12] - wc[c, :12]) <= tol * mag + 1e-12), (c, gc[c], wc[c])
        assert abs(gc[c, 12] - wc[c, 12]) <= tol * np.abs(want["rho"][cl == c]).sum() * 127.0 * scn.R + 1e-12


def run_gpu(gsr, torch, scn, cam, t, grad_rec):
    scene = gsr.Scene(scn)
    out = scene.project_backward(cam, t, torch.from_numpy(grad_rec.astype(np.float32)).cuda())
    torch.cuda.synchronize()
    scene.close()
    return out


@pytest.mark.parametrize("seed,C,per,deg", [(51, 4, 200.0, 3), (52, 3, 90.0, 3)])
def test_random_record_gradients_against_the_oracle(gsr, torch_mod, oracle_mod, seed, C, per, deg):
    wl = synth.scaled_object_workload(seed, C=C, per_cluster=per, W=120, H=88, fov=40.0, n_frames=2, B=2)
    cam, t = wl.frames[1]
    scn = wl.scene
    rng = np.random.default_rng(seed)
    grad_rec = random_records(scn, rng)
    got = run_gpu(gsr, torch_mod, scn, cam, t, grad_rec)
    want = oracle_from_records(oracle_mod, scn, cam, t, grad_rec)
    assert np.any(want["sh_res"] != 0.0) and np.any(want["rho"] != 0.0) and np.any(want["quat"] != 0.0)
    compare(scn, got, want)


def test_lower_sh_degrees_and_a_clamped_gaussian(gsr, torch_mod, oracle_mod):
    """SH degree 0..2 (other template instances) and Gaussians outside 1.3 lim (clamped Jacobian), behind the camera
    and inside znear (culled: zero gradient)."""
    from tests.helpers import tiny_scene, axis_camera
    rng = np.random.default_rng(5)
    for deg in (0, 1, 2):
        K = (deg + 1) ** 2
        n = 40
        means = rng.uniform(-1.0, 1.0, (n, 3))
        means[0] = [4.5, 0.1, 0.0]      # x/z beyond 1.3 lim_x = 0.78 at z = 4: clamped
        means[1] = [0.0, 0.0, -4.5]     # behind the camera
        means[2] = [0.1, 0.1, -3.9]     # z = 0.1 < znear
        scn, _ = tiny_scene(means, rng.uniform(0.05, 0.3, (n, 3)), quats=rng.standard_normal((n, 4)),
                            logits=rng.standard_normal(n), sh_degree=deg, R=2,
                            sh_base=0.3 * rng.standard_normal((n, K, 3)), sh_res=0.1 * rng.standard_normal((n, K, 3)),
                            motion_q=rng.integers(-100, 100, (n, 2, 3)), motion_scale=np.array([2e-4]),
                            levels=rng.integers(0, 4, n))
        cam = axis_camera(96, 64, 80.0, 4.0)
        grad_rec = random_records(scn, rng)
        got = run_gpu(gsr, torch_mod, scn, cam, 0.3, grad_rec)
        want = oracle_from_records(oracle_mod, scn, cam, 0.3, grad_rec)
        compare(scn, got, want)
        gg = got["gauss"].cpu().numpy()
        # culled Gaussians: exactly zero
        culled = [i for i in range(n) if not (scn.mean[i, 2] + 4.0 > 0.2)]
        assert len(culled) >= 2
        for i in culled:
            assert np.all(gg[i] == 0.0) and np.all(got["sh_base"][i].cpu().numpy() == 0.0)


def test_chain_from_images_to_parameters_against_the_oracle(gsr, torch_mod, oracle_mod):
    """render -> gsr_render_backward -> gsr_project_backward against O-5 -> O-8 -> O-9 state by state: the full
    gradient of sum_b <g_b, image_b> with respect to the scene's parameters."""
    torch = torch_mod
    wl = synth.scaled_object_workload(53, C=4, per_cluster=120.0, W=96, H=72, fov=40.0, n_frames=1, B=6)
    cam, t = wl.frames[0]
    scn = wl.scene
    lv = wl.levels[0].copy()
    lv[0] = 3
    lv[1] = 0
    scene = gsr.Scene(scn)
    ws = scene.new_workspace(cam, lv.shape[0])
    dlv = torch.from_numpy(np.ascontiguousarray(lv, np.int8)).cuda()
    out, _, _ = scene.render_states(cam, t, dlv, workspace=ws)
    scene.status(ws)
    rng = np.random.default_rng(53)
    g = rng.standard_normal(tuple(out.shape)).astype(np.float32)
    grad_rec = scene.render_backward(ws, out, torch.from_numpy(g).cuda())
    got = scene.project_backward(cam, t, grad_rec)
    torch.cuda.synchronize()
    scene.close()
    osc = oracle_mod.OracleScene(scn)
    want = None
    for b in range(lv.shape[0]):
        g9 = osc.backward(cam, t, lv[b], g[b].astype(np.float64))
        want = osc.project_backward(cam, t, lv[b], g9, into=want)
    # the compositor's backward carries cancellation-bounded absolute errors (tests/test_gpu_backward.py): the
    # chain is compared at 2e-3 of each block's largest entry plus 2e-3 of a typical block
    compare(scn, got, want, tol=2e-3, floor=2e-3)


def test_full_size_cfg1_properties(gsr, torch_mod):
    """configs[1] at full size: properties that hold at any size.  (1) the gradient of a raw quaternion is
    orthogonal to it; (2) the translation column of A_c(t) collects dL/dp of the cluster's Gaussians, which is also
    L^-T g_mean (L = the linear part of A_c(t)); (3) linear in the record gradients."""
    torch = torch_mod
    wl = synth.workload_cfg1(n_frames=1)
    cam, t = wl.frames[0]
    scn = wl.scene
    scene = gsr.Scene(scn)
    gen = torch.Generator(device="cuda").manual_seed(3)
    gr = torch.randn((scene.num_records(), 12), generator=gen, device="cuda", dtype=torch.float32)
    a = scene.project_backward(cam, t, gr)
    b = scene.project_backward(cam, t, 2.0 * gr)
    for k in ("gauss", "sh_base", "sh_res"):
        assert torch.equal(b[k], 2.0 * a[k])                  # a factor 2 is exact in binary32, thread by thread
    # the per-cluster sums are float atomics over ~3 k Gaussians: equal up to summation order
    assert bool(((b["cluster"] - 2.0 * a["cluster"]).abs() <= 1e-4 * a["cluster"].abs().amax(1, keepdim=True)).all())
    gq = a["gauss"][:, 9:13].double()
    q = torch.from_numpy(scn.quat.astype(np.float64)).cuda()
    dots = (gq * q).sum(1).abs()
    # (the unprojected gradient, of which the kernel removes the component along q, is of the size of the
    # log-scale gradient: both come from dL/d(Rm diag(s)); the rounding of the removal is relative to THAT size)
    size = (gq.abs() * q.abs()).sum(1) + a["gauss"][:, 6:9].double().abs().sum(1) * q.norm(dim=1)
    assert bool((dots <= 2e-5 * size + 1e-30).all()), float((dots / size).max())
    cl = torch.from_numpy(scn.cluster_of().astype(np.int64)).cuda()
    A = torch.from_numpy(scn.A0.astype(np.float64) + float(np.float32(t)) * scn.A1.astype(np.float64)).cuda()
    Linv_T = torch.linalg.inv(A[:, :, :3]).transpose(1, 2)                      # [C,3,3]
    dp = torch.einsum("nab,nb->na", Linv_T[cl], a["gauss"][:, 0:3].double())
    col = torch.zeros((scn.C, 3), dtype=torch.float64, device="cuda").index_add_(0, cl, dp)
    mag = torch.zeros((scn.C, 3), dtype=torch.float64, device="cuda").index_add_(0, cl, dp.abs())
    got = a["cluster"][:, [3, 7, 11]].double()
    assert bool(((got - col).abs() <= 2e-5 * mag + 1e-30).all())
    scene.close()


def test_refuses_scenes_it_does_not_cover(gsr, torch_mod):
    wl = synth.scaled_object_workload(29, C=2, per_cluster=40.0, W=64, H=48, fov=40.0, n_frames=1, B=2)
    scn = synth.with_position_residuals(wl.scene)
    scene = gsr.Scene(scn)
    gr = torch_mod.zeros((scene.num_records(), 12), device="cuda")
    with pytest.raises(gsr.GsrError):
        scene.project_backward(wl.frames[0][0], 0.5, gr)
    scene.close()


def oracle_from_records4(oracle_mod, scn, cam, t, grad_rec):
    """grad_rec double [4N, 12] of a scene with four records per Gaussian (record 4 i + delivered depth v, one colour in
    columns 0..2) -> the oracle's parameter gradients: pseudo-state v = every cluster at depth v, with the rows of
    record v (the oracle skips the Gaussians whose level is above v, as the GPU skips the records that do not exist)."""
    osc = oracle_mod.OracleScene(scn)
    out = None
    for v in range(4):
        r = grad_rec[v::4]
        g9 = np.ascontiguousarray(np.concatenate([r[:, 0:3], r[:, 6:12]], 1))
        out = osc.project_backward(cam, t, np.full(scn.C, v, np.int8), g9, into=out)
    return out


def compare_full(scn, got, want, tol=2e-4):
    compare(scn, got, want, tol)
    ok = want["margin"] > 1e-4

    def block(name, g, w):
        g, w = g.reshape(scn.N, -1), w.reshape(scn.N, -1)
        bmax = np.abs(w).max(1, keepdims=True)
        bad = (np.abs(g - w) > tol * bmax + 1e-12) & ok[:, None]
        assert not bad.any(), (name, np.argwhere(bad)[:4], g[bad][:4], w[bad][:4])

    d = got["delta"].double().cpu().numpy()
    block("delta2", d[:, 0:3], want["delta2"])
    block("delta3", d[:, 3:6], want["delta3"])
    at = got["attr"].double().cpu().numpy()
    dsh = got["d_sh"].double().cpu().numpy()
    for l in range(3):
        block(f"d_log_scale[{l}]", at[l][:, 0:3], want["d_log_scale"][l])
        block(f"d_quat[{l}]", at[l][:, 3:7], want["d_quat"][l])
        block(f"d_opacity_logit[{l}]", at[l][:, 7:8], want["d_opacity_logit"][l])
        block(f"d_sh[{l}]", dsh[l], want["d_sh"][l])


@pytest.mark.parametrize("what", ["all", "all+affine", "delta_only", "attr_only"])
def test_full_representation_against_the_oracle(gsr, torch_mod, oracle_mod, what):
    """Four records per Gaussian: position residual levels, per-level attribute and colour refinements, optionally the
    affine on the covariance (with a cluster affine far from the identity) — random record gradients against O-9."""
    import dataclasses
    torch = torch_mod
    wl = synth.scaled_object_workload(57, C=4, per_cluster=150.0, W=120, H=88, fov=40.0, n_frames=2, B=2)
    cam, t = wl.frames[1]
    scn = wl.scene
    rng = np.random.default_rng(57)
    if what in ("all", "all+affine"):
        scn = synth.with_attribute_refinements(synth.with_position_residuals(scn))
    elif what == "delta_only":
        scn = synth.with_position_residuals(scn)
    else:
        scn = synth.with_attribute_refinements(scn)
    if what == "all+affine":
        A0 = scn.A0.copy()
        A0[:, :, :3] += (0.2 * rng.standard_normal((scn.C, 3, 3))).astype(np.float32)
        scn = dataclasses.replace(scn, A0=A0, affine_on_covariance=True)
    lvl = scn.level_of()
    grad_rec = rng.standard_normal((4 * scn.N, 12)).astype(np.float32).astype(np.float64)
    grad_rec[:, 3:6] = 0.0                                  # one colour per record
    for v in range(4):
        grad_rec[v::4][lvl > v] = 0.0                       # a level-l Gaussian has the records v >= l only
    scene = gsr.Scene(scn)
    assert scene.num_records() == 4 * scn.N
    got = scene.project_backward_full(cam, t, torch.from_numpy(grad_rec.astype(np.float32)).cuda())
    torch.cuda.synchronize()
    scene.close()
    want = oracle_from_records4(oracle_mod, scn, cam, t, grad_rec)
    compare_full(scn, got, want)
    if what == "delta_only":
        assert float(got["attr"].abs().max()) == 0.0 and float(got["d_sh"].abs().max()) == 0.0
    if what in ("all", "all+affine"):
        assert np.any(want["d_quat"][2] != 0.0) and np.any(want["delta3"] != 0.0) and np.any(want["d_sh"][2] != 0.0)


def test_full_entry_serves_two_record_scenes_and_the_chain(gsr, torch_mod, oracle_mod):
    """(1) A scene with two records per Gaussian through gsr_project_backward_full: the same numbers as
    gsr_project_backward, zeros for the refinement outputs.  (2) The whole chain on the full representation:
    render -> gsr_render_backward -> gsr_project_backward_full against O-5 -> O-8 -> O-9 state by state."""
    torch = torch_mod
    wl = synth.scaled_object_workload(58, C=4, per_cluster=110.0, W=96, H=72, fov=40.0, n_frames=1, B=6)
    cam, t = wl.frames[0]
    scene = gsr.Scene(wl.scene)
    gen = torch.Generator(device="cuda").manual_seed(4)
    gr = torch.randn((scene.num_records(), 12), generator=gen, device="cuda", dtype=torch.float32)
    a, b = scene.project_backward(cam, t, gr), scene.project_backward_full(cam, t, gr)
    for k in ("gauss", "sh_base", "sh_res"):
        assert torch.equal(a[k], b[k])
    assert torch.allclose(a["cluster"], b["cluster"], rtol=1e-4, atol=1e-6)
    assert float(b["delta"].abs().max()) == 0.0 and float(b["attr"].abs().max()) == 0.0 and float(b["d_sh"].abs().max()) == 0.0
    scene.close()
    # (2)
    scn = synth.with_attribute_refinements(synth.with_position_residuals(wl.scene))
    lv = wl.levels[0].copy()
    lv[0], lv[1], lv[2] = 3, 2, 1
    scene = gsr.Scene(scn)
    ws = scene.new_workspace(cam, lv.shape[0])
    dlv = torch.from_numpy(np.ascontiguousarray(lv, np.int8)).cuda()
    out, _, _ = scene.render_states(cam, t, dlv, workspace=ws)
    scene.status(ws)
    rng = np.random.default_rng(58)
    g = rng.standard_normal(tuple(out.shape)).astype(np.float32)
    grad_rec = scene.render_backward(ws, out, torch.from_numpy(g).cuda())
    got = scene.project_backward_full(cam, t, grad_rec)
    torch.cuda.synchronize()
    scene.close()
    osc = oracle_mod.OracleScene(scn)
    want = None
    for s_ in range(lv.shape[0]):
        g9 = osc.backward(cam, t, lv[s_], g[s_].astype(np.float64))
        want = osc.project_backward(cam, t, lv[s_], g9, into=want)
    compare(scn, got, want, tol=2e-3, floor=2e-3)
    at = got["attr"].double().cpu().numpy()
    for l in range(3):
        w = want["d_log_scale"][l]
        scale = np.median(np.abs(w).max(1)[np.abs(w).max(1) > 0])
        assert np.all(np.abs(at[l][:, 0:3] - w) <= 2e-3 * np.abs(w).max(1, keepdims=True) + 2e-3 * scale + 1e-12)

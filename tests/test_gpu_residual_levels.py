"""GPU parity for scenes WITH the level-2 / level-3 position residuals delta^(2), delta^(3) of Eq. (1)
(DESIGN.md §14 reading I1): four projected records per Gaussian (one per delivered depth).
Same bars as the core path: integer work bit-exact, decision-feeding fp32 bit-exact, pixels <= 2e-4,
PSNR <= 1e-3 dB, batched == serial bitwise, dedup-neutral."""
import numpy as np
import pytest

from paper_2606_17212_b200 import synth

pytestmark = pytest.mark.gpu

PIX_TOL, DB_TOL = 2e-4, 1e-3


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


def _workload(seed, attrs=False, **kw):
    wl = synth.scaled_object_workload(seed, **kw)
    wl.scene = synth.with_position_residuals(wl.scene, seed_cfg=seed)
    if attrs:   # + per-level scale / rotation / opacity refinements (reading I2)
        wl.scene = synth.with_attribute_refinements(wl.scene, seed_cfg=seed)
    return wl


def _render(torch, scene, cam, t, lv, **kw):
    ws = scene.new_workspace(cam, lv.shape[0])
    out, mse, psnr = scene.render_states(cam, t, torch.from_numpy(np.ascontiguousarray(lv, np.int8)).cuda(),
                                         workspace=ws, **kw)
    scene.status(ws)
    return out, mse, psnr, ws


@pytest.mark.parametrize("attrs", [False, True])
def test_projection_bit_exact_per_depth(gsr, torch_mod, oracle_mod, attrs):
    wl = _workload(21, attrs=attrs, C=5, per_cluster=700.0, W=168, H=120, fov=40.0, n_frames=2, B=8)
    sc = wl.scene
    for cam, t in wl.frames:
        scene = gsr.Scene(sc)
        assert scene.V == 4
        osc = oracle_mod.OracleScene(sc)
        lv = np.stack([np.full(sc.C, d, np.int8) for d in range(-1, 4)])
        _, _, _, ws = _render(torch_mod, scene, cam, t, lv)
        P = scene.debug_projection(ws)
        level = sc.level_of()
        checked = 0
        for d in range(0, 4):
            op = osc.project(cam, t, np.full(sc.C, d, np.int8))
            rid = 4 * np.arange(sc.N) + d                        # variant v = d
            present = level <= d
            m = op["valid"] == 1
            assert np.array_equal((P["valid"][rid] == 1) & present, m), f"valid mismatch at depth {d}"
            checked += int(m.sum())
            for name in ("radius", "rect", "depth_bits", "count"):
                assert np.array_equal(P[name][rid][m], op[name][m]), (name, d)
            assert np.array_equal(P["mean2d"][rid][m].view(np.uint32),
                                  np.stack([op["mx"], op["my"]], 1)[m].view(np.uint32))
            assert np.array_equal(P["conic"][rid][m].view(np.uint32),
                                  np.stack([op["qa"], op["qb"], op["qc"]], 1)[m].view(np.uint32))
            assert np.max(np.abs(P["rgb_base"][rid][m] - op["rgb"][m])) < 2e-6
        assert checked > 0
        # the residuals really move things: depth-2 and depth-1 geometry differ
        v1, v2 = 4 * np.arange(sc.N) + 1, 4 * np.arange(sc.N) + 2
        both = (P["valid"][v1] == 1) & (P["valid"][v2] == 1)
        assert np.any(P["mean2d"][v1][both] != P["mean2d"][v2][both])
        scene.close()


@pytest.mark.parametrize("attrs", [False, True])
def test_keys_pixels_distortion_and_batch_invariance(gsr, torch_mod, oracle_mod, attrs):
    torch = torch_mod
    wl = _workload(22, attrs=attrs, C=7, per_cluster=500.0, W=136, H=104, fov=40.0, n_frames=1, B=40)
    cam, t = wl.frames[0]
    lv = wl.levels[0]
    scene = gsr.Scene(wl.scene)
    osc = oracle_mod.OracleScene(wl.scene)
    full = np.full((1, wl.scene.C), 3, np.int8)
    ref, _, _, _ = _render(torch, scene, cam, t, full)
    ref = ref[0].contiguous()
    out, mse, psnr, ws = _render(torch, scene, cam, t, lv, ref=ref)
    # sorted key lists (integer work): bit-exact
    counts = scene.debug_state_counts(ws, lv.shape[0])
    for b in (0, 7, 19, 39):
        op = osc.project(cam, t, lv[b])
        tile, dbits, idx = osc.keys(op, cam)
        g_tile, g_db, g_idx, n = scene.debug_keys(ws, b, cap=tile.size + 16)
        assert n == tile.size == counts[b]
        assert np.array_equal(g_tile, tile) and np.array_equal(g_db, dbits) and np.array_equal(g_idx, idx)
    # pixels and distortion against the oracle
    o_img, _ = osc.render_batch(cam, t, lv)
    o_ref, _ = osc.render(cam, t, full[0])
    assert np.abs(out.cpu().numpy() - o_img).max() <= PIX_TOL
    assert np.abs(ref.cpu().numpy() - o_ref).max() <= PIX_TOL
    o_mse, o_psnr = oracle_mod.distortion(o_img, o_ref)
    assert np.abs(psnr.cpu().numpy() - o_psnr).max() <= DB_TOL
    # batched == serial, bitwise; and dedup on/off, state block 8/4: bitwise
    for b in (0, 13, 39):
        o1, m1, _, _ = _render(torch, scene, cam, t, lv[b:b + 1], ref=ref)
        assert torch.equal(o1[0], out[b]) and torch.equal(m1[0], mse[b])
    gsr.set_option("dedup", 0)
    o2, m2, _, _ = _render(torch, scene, cam, t, lv, ref=ref)
    gsr.set_option("dedup", 1)
    gsr.set_option("state_block", 4)
    o3, m3, _, _ = _render(torch, scene, cam, t, lv, ref=ref)
    gsr.set_option("state_block", 8)
    assert torch.equal(o2, out) and torch.equal(m2, mse) and torch.equal(o3, out) and torch.equal(m3, mse)
    scene.close()


def test_zero_residuals_equal_the_two_variant_path(gsr, torch_mod):
    """delta2 = delta3 = 0 switches to four records per Gaussian but must give bitwise the same pixels."""
    import dataclasses
    torch = torch_mod
    wl = synth.scaled_object_workload(23, C=4, per_cluster=400.0, W=96, H=80, fov=40.0, n_frames=1, B=16)
    cam, t = wl.frames[0]
    lv = wl.levels[0]
    s2 = gsr.Scene(wl.scene)
    z = np.zeros((wl.scene.N, 3), np.float32)
    s4 = gsr.Scene(dataclasses.replace(wl.scene, delta2=z, delta3=z))
    assert (s2.V, s4.V) == (2, 4)
    a, _, _, _ = _render(torch, s2, cam, t, lv)
    b, _, _, _ = _render(torch, s4, cam, t, lv)
    assert torch.equal(a, b)


def test_attribute_refinements_alone_and_zero(gsr, torch_mod, oracle_mod):
    """Attribute refinements without position residuals; zero refinements == the two-record path bitwise."""
    import dataclasses
    torch = torch_mod
    wl = synth.scaled_object_workload(24, C=4, per_cluster=400.0, W=96, H=80, fov=40.0, n_frames=1, B=16)
    cam, t = wl.frames[0]
    lv = wl.levels[0]
    sc = synth.with_attribute_refinements(wl.scene, seed_cfg=24)
    scene = gsr.Scene(sc)
    assert scene.V == 4
    out, _, _, _ = _render(torch, scene, cam, t, lv)
    o_img, _ = oracle_mod.OracleScene(sc).render_batch(cam, t, lv)
    assert np.abs(out.cpu().numpy() - o_img).max() <= PIX_TOL
    z = lambda *shape: np.zeros((3, sc.N) + shape, np.float32)
    s0 = gsr.Scene(dataclasses.replace(wl.scene, d_log_scale=z(3), d_quat=z(4), d_opacity_logit=z()))
    a, _, _, _ = _render(torch, gsr.Scene(wl.scene), cam, t, lv)
    b, _, _, _ = _render(torch, s0, cam, t, lv)
    assert torch.equal(a, b)


@pytest.mark.parametrize("four", [False, True])
def test_affine_push_forward_of_covariance(gsr, torch_mod, oracle_mod, four):
    """Reading I4 (optional flag): projection bit-exact and pixels within tolerance with Sigma_t = L Sigma L^T,
    on the two-record and on the four-record path; the flag really changes the footprints."""
    import dataclasses
    torch = torch_mod
    wl = synth.scaled_object_workload(25, C=5, per_cluster=400.0, W=112, H=88, fov=40.0, n_frames=1, B=12)
    cam, t = wl.frames[0]
    lv = wl.levels[0]
    sc = wl.scene
    # a visible shear / scale in the affine, so that the push-forward matters
    A0 = sc.A0.copy()
    A0[:, 0, 1] += 0.3
    A0[:, 1, 1] *= 1.4
    sc = dataclasses.replace(sc, A0=A0, affine_on_covariance=True)
    if four:
        sc = synth.with_attribute_refinements(synth.with_position_residuals(sc, seed_cfg=25), seed_cfg=25)
    scene = gsr.Scene(sc)
    osc = oracle_mod.OracleScene(sc)
    out, _, _, ws = _render(torch, scene, cam, t, lv)
    P = scene.debug_projection(ws)
    V = scene.V
    for d in (0, 1, 3):
        op = osc.project(cam, t, np.full(sc.C, d, np.int8))
        v = d if V == 4 else (0 if d == 0 else 1)
        rid = V * np.arange(sc.N) + v
        m = op["valid"] == 1
        assert np.array_equal(P["conic"][rid][m].view(np.uint32),
                              np.stack([op["qa"], op["qb"], op["qc"]], 1)[m].view(np.uint32))
        assert np.array_equal(P["radius"][rid][m], op["radius"][m]) and np.array_equal(P["rect"][rid][m], op["rect"][m])
    o_img, _ = osc.render_batch(cam, t, lv)
    assert np.abs(out.cpu().numpy() - o_img).max() <= PIX_TOL
    off = gsr.Scene(dataclasses.replace(sc, affine_on_covariance=False))
    out_off, _, _, _ = _render(torch, off, cam, t, lv)
    assert not torch.equal(out_off, out)

"""GPU parity tests: the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle
on the same seeded inputs.  Run on a B200 with `pytest -m gpu`.

Bars (BASELINE.json north_star): closure masks, radii / rectangles / depth bits / tile-intersection
counts and sorted key lists BIT-EXACT; pixels max-abs <= 2e-4; utilities <= 1e-3 dB; batched GPU render
bitwise equal to one-state-at-a-time GPU render.
"""
import numpy as np
import pytest

from paper_2606_17212_b200 import synth
from tests.helpers import axis_camera, tiny_scene

pytestmark = pytest.mark.gpu

PIX_TOL = 2e-4
DB_TOL = 1e-3


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def gsr(torch_mod):
    from paper_2606_17212_b200 import gsr as G
    G.lib()
    return G


def _dev_levels(torch, lv):
    return torch.from_numpy(np.ascontiguousarray(lv, np.int8)).cuda()


def _render(torch, scene, cam, t, lv, **kw):
    ws = scene.new_workspace(cam, lv.shape[0])
    out, mse, psnr = scene.render_states(cam, t, _dev_levels(torch, lv), workspace=ws, **kw)
    scene.status(ws)
    return out, mse, psnr, ws


# ------------------------------------------------------------------------------------------ closure
def test_closure_bit_exact(gsr, torch_mod, oracle_mod):
    rng = np.random.default_rng(5)
    mask = np.concatenate([np.arange(16, dtype=np.uint8), synth.sample_masks(rng, 4099)])
    d_ref, c_ref = oracle_mod.close_levels(mask)
    d, c = gsr.close_levels(torch_mod.from_numpy(mask).cuda())
    assert np.array_equal(d.cpu().numpy(), d_ref)
    assert np.array_equal(c.cpu().numpy(), c_ref)


# ------------------------------------------------------------------------------------------ projection
def _check_projection(gsr, torch, oracle_mod, sc_np, cam, t):
    """Every (Gaussian, cluster depth) combination of the oracle must equal the GPU record that the
    state semantics select: variant 0 for depth 0, variant 1 for depth >= 1, absent if depth < level."""
    scene = gsr.Scene(sc_np)
    osc = oracle_mod.OracleScene(sc_np)
    lv = np.stack([np.full(sc_np.C, d, np.int8) for d in range(-1, 4)])
    _, _, _, ws = _render(torch, scene, cam, t, lv)
    assert np.array_equal(scene.debug_closure(ws, lv.shape[0]), lv)
    P = scene.debug_projection(ws)
    level = sc_np.level_of()
    n_checked = 0
    for d in range(-1, 4):
        op = osc.project(cam, t, np.full(sc_np.C, d, np.int8))
        v = 0 if d == 0 else 1
        rid = 2 * np.arange(sc_np.N) + v
        present = level <= d
        ovalid = op["valid"] == 1
        assert not np.any(ovalid & ~present)
        gvalid = (P["valid"][rid] == 1) & present
        assert np.array_equal(gvalid, ovalid), f"valid mismatch at depth {d}"
        m = ovalid
        n_checked += int(m.sum())
        assert np.array_equal(P["radius"][rid][m], op["radius"][m])
        assert np.array_equal(P["rect"][rid][m], op["rect"][m])
        assert np.array_equal(P["depth_bits"][rid][m], op["depth_bits"][m])
        assert np.array_equal(P["count"][rid][m], op["count"][m])
        # decision-feeding fp32 quantities: bit-exact
        assert np.array_equal(P["mean2d"][rid][m].view(np.uint32), np.stack([op["mx"], op["my"]], 1)[m].view(np.uint32))
        assert np.array_equal(P["conic"][rid][m].view(np.uint32),
                              np.stack([op["qa"], op["qb"], op["qc"]], 1)[m].view(np.uint32))
        # colour is continuous (fp32 on the GPU, double in the oracle)
        col = P["rgb_res"][rid] if d == 3 else P["rgb_base"][rid]
        assert np.max(np.abs(col[m] - op["rgb"][m])) < 2e-6 if m.any() else True
    assert n_checked > 0
    scene.close()


def test_projection_bit_exact_cfg0(gsr, torch_mod, oracle_mod):
    wl = synth.workload_cfg0()
    cam, t = wl.frames[0]
    _check_projection(gsr, torch_mod, oracle_mod, wl.scene, cam, t)


def test_projection_bit_exact_scaled_cfg1_sh3(gsr, torch_mod, oracle_mod):
    wl = synth.scaled_object_workload(11, C=6, per_cluster=900.0, W=200, H=136, fov=40.0, n_frames=2, B=8)
    for cam, t in wl.frames:
        _check_projection(gsr, torch_mod, oracle_mod, wl.scene, cam, t)


@pytest.mark.parametrize("sh_degree,R", [(0, 1), (1, 3), (2, 5), (3, 7), (2, 32)])
def test_projection_every_sh_degree_and_ragged_basis_sizes(gsr, torch_mod, oracle_mod, sh_degree, R):
    """SH degrees 0..3 and temporal-basis sizes whose 3R int8 coefficients do not fill whole 4-byte words
    (and the maximum, GSR_MAX_R = 32): projection bit-exact, colours within 2e-6, at t != 0 so that every
    basis term and the affine's A1 contribute."""
    rng = np.random.default_rng(1000 * sh_degree + R)
    n, Cn, K = 240, 4, (sh_degree + 1) ** 2
    means = rng.uniform(-0.6, 0.6, (n, 3))
    sh_base = rng.normal(0.0, 0.15, (n, K, 3))
    sh_base[:, 0, :] += rng.uniform(-0.5, 1.2, (n, 3))
    A1 = rng.normal(0.0, 0.03, (Cn, 3, 4))
    sc, _ = tiny_scene(means, rng.uniform(0.02, 0.12, (n, 3)), quats=rng.normal(size=(n, 4)),
                       logits=rng.uniform(-2, 3, n), levels=rng.integers(0, 4, n), clusters=rng.integers(0, Cn, n),
                       C=Cn, sh_degree=sh_degree, R=R, A1=A1, motion_q=rng.integers(-127, 128, (n, R, 3)),
                       motion_scale=rng.uniform(1e-4, 6e-4, Cn), sh_base=sh_base,
                       sh_res=rng.normal(0.0, 0.05, (n, K, 3)))
    cam = axis_camera(W=152, H=104, f=130.0, z0=3.5)
    _check_projection(gsr, torch_mod, oracle_mod, sc, cam, 0.37)


def test_projection_forward_facing_near_plane_and_offscreen(gsr, torch_mod, oracle_mod):
    # cfg2-like geometry at reduced size: Gaussians behind / near the camera and outside the frustum
    full = synth.scene_cfg2()
    keep = np.zeros(full.N, bool)
    off = full.group_off
    new_off = [0]
    idx = []
    for g in range(4 * full.C):
        take = np.arange(off[g], off[g + 1])[:: 40]
        idx.append(take)
        new_off.append(new_off[-1] + take.size)
    idx = np.concatenate(idx)
    sc = synth.Scene(full.C, idx.size, full.sh_degree, full.R, np.asarray(new_off, np.int32), full.mean[idx],
                     full.log_scale[idx], full.quat[idx], full.opacity_logit[idx], full.sh_base[idx],
                     full.sh_res[idx], full.motion_q[idx], full.A0, full.A1, full.motion_scale, full.background)
    cam = synth.jitter_cameras(2, 1, 134, 240, synth.focal_from_fov(240, 50.0))[0]
    _check_projection(gsr, torch_mod, oracle_mod, sc, cam, 0.375)


# ------------------------------------------------------------------------------------------ keys
def test_sorted_key_lists_and_counts_bit_exact_cfg0(gsr, torch_mod, oracle_mod):
    wl = synth.workload_cfg0()
    cam, t = wl.frames[0]
    lv = wl.levels[0]
    scene = gsr.Scene(wl.scene)
    osc = oracle_mod.OracleScene(wl.scene)
    _, _, _, ws = _render(torch_mod, scene, cam, t, lv)
    counts = scene.debug_state_counts(ws, lv.shape[0])
    rng = np.random.default_rng(1)
    picks = [0, 1, 312, 624] + rng.integers(0, 625, 12).tolist()
    for b in range(lv.shape[0]):
        if b in picks:
            op = osc.project(cam, t, lv[b])
            tile, dbits, idx = osc.keys(op, cam)
            g_tile, g_db, g_idx, n = scene.debug_keys(ws, b, cap=max(tile.size, 1) + 16)
            assert n == tile.size == counts[b]
            assert np.array_equal(g_tile, tile) and np.array_equal(g_db, dbits) and np.array_equal(g_idx, idx)
    # I_b for ALL states against the oracle's own count
    _, stats = osc.render_batch(cam, t, lv)
    assert np.array_equal(counts, stats[:, 0])
    scene.close()


def test_sorted_key_lists_scaled_cfg1(gsr, torch_mod, oracle_mod):
    wl = synth.scaled_object_workload(12, C=8, per_cluster=1500.0, W=328, H=200, fov=40.0, n_frames=1, B=24)
    cam, t = wl.frames[0]
    lv = wl.levels[0]
    scene = gsr.Scene(wl.scene)
    osc = oracle_mod.OracleScene(wl.scene)
    _, _, _, ws = _render(torch_mod, scene, cam, t, lv)
    counts = scene.debug_state_counts(ws, lv.shape[0])
    for b in (0, 5, 13, 23):
        op = osc.project(cam, t, lv[b])
        tile, dbits, idx = osc.keys(op, cam)
        g_tile, g_db, g_idx, n = scene.debug_keys(ws, b, cap=tile.size + 16)
        assert n == tile.size == counts[b]
        assert np.array_equal(g_tile, tile) and np.array_equal(g_db, dbits) and np.array_equal(g_idx, idx)
        # strictly increasing (tile, depth, index): the list is the unique sorted order
        a, b_, c = g_tile.astype(np.int64), g_db.astype(np.int64), g_idx.astype(np.int64)
        da, db_, dc = np.diff(a), np.diff(b_), np.diff(c)
        assert np.all((da > 0) | ((da == 0) & ((db_ > 0) | ((db_ == 0) & (dc > 0)))))
    scene.close()


# ------------------------------------------------------------------------------------------ pixels
def test_pixels_cfg0_all_625_states(gsr, torch_mod, oracle_mod):
    wl = synth.workload_cfg0()
    cam, t = wl.frames[0]
    lv = wl.levels[0]
    scene = gsr.Scene(wl.scene)
    osc = oracle_mod.OracleScene(wl.scene)
    out, _, _, _ = _render(torch_mod, scene, cam, t, lv)
    ref, _ = osc.render_batch(cam, t, lv)
    err = np.abs(out.cpu().numpy().astype(np.float64) - ref)
    assert err.max() <= PIX_TOL, err.max()
    # the all-absent state is exactly the background
    assert np.array_equal(out[0].cpu().numpy(), np.broadcast_to(wl.scene.background, (cam.H, cam.W, 3)))
    scene.close()


@pytest.mark.parametrize("S", [1, 4, 8, 16])
def test_pixels_scaled_cfg1_ragged_tiles_white_background(gsr, torch_mod, oracle_mod, S):
    # 200x136: 13x9 tiles with ragged right and bottom edges; B = 21 is not a multiple of any state block
    wl = synth.scaled_object_workload(13, C=8, per_cluster=1200.0, W=200, H=136, fov=40.0, n_frames=1, B=42)
    cam, t = wl.frames[0]
    lv = wl.levels[0][:21]
    scene = gsr.Scene(wl.scene)
    osc = oracle_mod.OracleScene(wl.scene)
    gsr.set_option("state_block", S)
    try:
        out, _, _, _ = _render(torch_mod, scene, cam, t, lv)
    finally:
        gsr.set_option("state_block", 8)
    ref, _ = osc.render_batch(cam, t, lv)
    err = np.abs(out.cpu().numpy().astype(np.float64) - ref)
    assert err.max() <= PIX_TOL, err.max()
    scene.close()


def test_pixels_dense_stack_early_termination(gsr, torch_mod, oracle_mod):
    # many opaque wide Gaussians stacked over the image: every pixel terminates early
    rng = np.random.default_rng(3)
    n = 400
    means = np.stack([rng.uniform(-0.5, 0.5, n), rng.uniform(-0.5, 0.5, n), rng.uniform(-0.5, 0.5, n)], 1)
    lev = rng.integers(0, 4, n)
    clu = rng.integers(0, 3, n)
    sc, _ = tiny_scene(means, 0.25, logits=3.0, colors=rng.uniform(0, 1, (n, 3)), levels=lev, clusters=clu, C=3,
                       background=(0.2, 0.4, 0.6))
    cam = axis_camera(W=96, H=80, f=90.0)
    lv = synth.all_closed_states(3)
    scene = gsr.Scene(sc)
    osc = oracle_mod.OracleScene(sc)
    out, _, _, _ = _render(torch_mod, scene, cam, 0.3, lv)
    ref, stats = osc.render_batch(cam, 0.3, lv)
    assert np.abs(out.cpu().numpy() - ref).max() <= PIX_TOL
    scene.close()


# ------------------------------------------------------------------------------------------ batched == serial
def test_batched_equals_serial_bitwise(gsr, torch_mod):
    wl = synth.workload_cfg0()
    cam, t = wl.frames[0]
    lv = wl.levels[0]
    scene = gsr.Scene(wl.scene)
    out, _, _, _ = _render(torch_mod, scene, cam, t, lv)
    rng = np.random.default_rng(2)
    for b in [0, 624] + rng.integers(0, 625, 30).tolist():
        one, _, _, _ = _render(torch_mod, scene, cam, t, lv[b:b + 1])
        assert torch_mod.equal(one[0], out[b]), f"state {b} differs between batched and serial rendering"
    # and the result does not depend on the state-block size or on batch composition
    perm = rng.permutation(625)
    for S in (4, 16):
        gsr.set_option("state_block", S)
        try:
            o2, _, _, _ = _render(torch_mod, scene, cam, t, lv[perm])
        finally:
            gsr.set_option("state_block", 8)
        assert torch_mod.equal(o2, out[torch_mod.from_numpy(perm).cuda()])
    scene.close()


def test_batched_equals_serial_scaled_cfg1(gsr, torch_mod):
    wl = synth.scaled_object_workload(14, C=8, per_cluster=1500.0, W=328, H=200, fov=40.0, n_frames=1, B=32)
    cam, t = wl.frames[0]
    lv = wl.levels[0]
    scene = gsr.Scene(wl.scene)
    out, _, _, _ = _render(torch_mod, scene, cam, t, lv)
    for b in (0, 7, 16, 31):
        one, _, _, _ = _render(torch_mod, scene, cam, t, lv[b:b + 1])
        assert torch_mod.equal(one[0], out[b])
    scene.close()


# ------------------------------------------------------------------------------------------ distortion / utility
def test_distortion_and_utility_against_oracle(gsr, torch_mod, oracle_mod):
    wl = synth.scaled_object_workload(15, C=8, per_cluster=1200.0, W=200, H=136, fov=40.0, n_frames=1, B=64)
    cam, t = wl.frames[0]
    lv = wl.levels[0]
    scene = gsr.Scene(wl.scene)
    osc = oracle_mod.OracleScene(wl.scene)
    full = np.full((1, wl.scene.C), 3, np.int8)
    ref_img, _, _, _ = _render(torch_mod, scene, cam, t, full)
    out, _, _, _ = _render(torch_mod, scene, cam, t, lv)
    mse, psnr = gsr.distortion(out, ref_img[0].contiguous())
    # fused path: bitwise the same distortions, with and without materialising the images
    _, mse_f, psnr_f, _ = _render(torch_mod, scene, cam, t, lv, ref=ref_img[0].contiguous(), want_images=False)
    assert torch_mod.equal(mse, mse_f) and torch_mod.equal(psnr, psnr_f)
    out2, mse_f2, _, _ = _render(torch_mod, scene, cam, t, lv, ref=ref_img[0].contiguous())
    assert torch_mod.equal(mse, mse_f2) and torch_mod.equal(out, out2)
    # oracle
    o_imgs, _ = osc.render_batch(cam, t, lv)
    o_ref, _ = osc.render(cam, t, full[0])
    o_mse, o_psnr = oracle_mod.distortion(o_imgs, o_ref)
    assert np.max(np.abs(psnr.cpu().numpy() - o_psnr)) <= DB_TOL
    assert np.allclose(mse.cpu().numpy(), o_mse, rtol=2e-4, atol=1e-12)
    # utilities
    G = wl.G
    iwo, iw, gid = wl.idx_without[0], wl.idx_with[0], wl.group_id[0]
    u, dm, dd = gsr.group_utility(mse, psnr, torch_mod.from_numpy(iwo).cuda(), torch_mod.from_numpy(iw).cuda(),
                                  torch_mod.from_numpy(gid).cuda(), G)
    o_dm, o_dd, o_u = oracle_mod.group_utility(o_mse, o_psnr, iwo, iw, gid, G)
    assert np.max(np.abs(dd.cpu().numpy() - o_dd)) <= DB_TOL
    for k, name in enumerate(oracle_mod.UTIL_FIELDS):
        if name.endswith("_db"):          # north_star: utilities within 1e-3 dB, flat
            assert np.max(np.abs(u[name] - o_u[:, k])) <= DB_TOL, name
        elif name == "count":
            assert np.array_equal(u[name], o_u[:, k]), name
        else:                              # MSE-unit aggregates: the relative bar of the MSE itself
            assert np.max(np.abs(u[name] - o_u[:, k])) <= 1e-6 + 2e-4 * np.max(np.abs(o_u[:, k])), name
    scene.close()


def test_group_utility_matches_oracle_on_random_tables(gsr, torch_mod, oracle_mod):
    # the aggregation alone, on random distortion tables, incl. empty groups, singletons and a group
    # larger than the shared-memory cache (radix select from global memory)
    rng = np.random.default_rng(9)
    B = 9000
    mse = rng.uniform(1e-5, 1e-2, B)
    psnr = (-10 * np.log10(mse)).astype(np.float32)
    n_pairs = 4500
    iwo = rng.integers(0, B, n_pairs).astype(np.int32)
    iw = rng.integers(0, B, n_pairs).astype(np.int32)
    gid = rng.integers(0, 5, n_pairs).astype(np.int32)
    gid[:3000] = 6            # one big group (> 2048 members)
    gid[3000] = 7             # a singleton; groups 5 and 8 stay empty
    G = 9
    u, dm, dd = gsr.group_utility(torch_mod.from_numpy(mse).cuda(), torch_mod.from_numpy(psnr).cuda(),
                                  torch_mod.from_numpy(iwo).cuda(), torch_mod.from_numpy(iw).cuda(),
                                  torch_mod.from_numpy(gid).cuda(), G)
    o_dm, o_dd, o_u = oracle_mod.group_utility(mse, psnr.astype(np.float64), iwo, iw, gid, G)
    assert np.allclose(dm.cpu().numpy(), o_dm, rtol=0, atol=1e-15)
    assert np.allclose(dd.cpu().numpy(), o_dd, rtol=0, atol=1e-9)
    for k, name in enumerate(oracle_mod.UTIL_FIELDS):
        assert np.allclose(u[name], o_u[:, k], rtol=1e-9, atol=1e-12), name


# ------------------------------------------------------------------------------------------ edge cases / errors
def test_empty_batch_and_empty_scene(gsr, torch_mod):
    wl = synth.workload_cfg0()
    cam, t = wl.frames[0]
    scene = gsr.Scene(wl.scene)
    out, _, _, ws = _render(torch_mod, scene, cam, t, np.zeros((0, 4), np.int8))
    assert out.shape[0] == 0
    scene.close()
    sc, _ = tiny_scene(np.zeros((0, 3)), 0.1, C=2, background=(0.1, 0.2, 0.3))
    scene = gsr.Scene(sc)
    lv = synth.all_closed_states(2)
    out, _, _, _ = _render(torch_mod, scene, axis_camera(W=40, H=24), 0.0, lv)
    assert np.array_equal(out.cpu().numpy(), np.broadcast_to(np.float32([0.1, 0.2, 0.3]), out.shape))
    scene.close()


@pytest.mark.parametrize("W,H", [(1, 1), (1, 37), (53, 1), (15, 17), (16, 16), (17, 15), (33, 2)])
def test_degenerate_image_shapes(gsr, torch_mod, oracle_mod, W, H):
    """One pixel, one-pixel-wide strips, one short of / exactly / one past a tile boundary: pixels, key counts
    and the fused distortion against the oracle; batched == serial bitwise."""
    rng = np.random.default_rng(100 * W + H)
    n = 60
    means = np.c_[rng.uniform(-0.4, 0.4, n), rng.uniform(-0.4, 0.4, n), rng.uniform(-0.3, 0.3, n)]
    sc, _ = tiny_scene(means, rng.uniform(0.03, 0.15, (n, 3)), logits=rng.uniform(-1, 3, n),
                       colors=rng.uniform(0.1, 0.9, (n, 3)), levels=rng.integers(0, 4, n),
                       clusters=rng.integers(0, 3, n), C=3, background=(0.2, 0.1, 0.3))
    cam = axis_camera(W=W, H=H, f=0.9 * max(W, H, 8), z0=3.0)
    lv = synth.all_closed_states(3)[::5]                       # 25 of the 125 closed states
    scene = gsr.Scene(sc)
    osc = oracle_mod.OracleScene(sc)
    full = np.full((1, 3), 3, np.int8)
    ref, _, _, _ = _render(torch_mod, scene, cam, 0.0, full)
    ref = ref[0].contiguous()
    ws = scene.new_workspace(cam, lv.shape[0])
    out, mse, psnr = scene.render_states(cam, 0.0, _dev_levels(torch_mod, lv), workspace=ws, ref=ref)
    scene.status(ws)
    o_img, o_cnt = osc.render_batch(cam, 0.0, lv)
    o_ref, _ = osc.render(cam, 0.0, full[0])
    assert np.array_equal(scene.debug_state_counts(ws, lv.shape[0]), o_cnt[:, 0])
    assert np.abs(out.cpu().numpy() - o_img).max() <= PIX_TOL
    _, o_psnr = oracle_mod.distortion(o_img, o_ref)
    assert np.abs(psnr.cpu().numpy() - o_psnr).max() <= 1e-3
    for b in (0, 7, lv.shape[0] - 1):
        one, _, _, _ = _render(torch_mod, scene, cam, 0.0, lv[b:b + 1])
        assert torch_mod.equal(one[0], out[b])
    scene.close()


def test_maximum_cluster_count(gsr, torch_mod, oracle_mod):
    """C = 4096, the documented maximum (the per-CTA presence table then needs more than the default 48 KB of
    shared memory): pixels against the oracle, with and without tile dedup; C = 4097 is refused at load."""
    import dataclasses
    rng = np.random.default_rng(4096)
    Cn, n = 4096, 8192
    sc, _ = tiny_scene(rng.uniform(-0.8, 0.8, (n, 3)), rng.uniform(0.02, 0.06, (n, 3)), logits=rng.uniform(-1, 3, n),
                       colors=rng.uniform(0.1, 0.9, (n, 3)), levels=rng.integers(0, 4, n), clusters=np.arange(n) % Cn,
                       C=Cn, background=(0.1, 0.1, 0.1))
    cam = axis_camera(W=96, H=64, f=80.0, z0=3.0)
    lv = synth.sample_levels(rng, 24, Cn)
    scene = gsr.Scene(sc)
    o_img, _ = oracle_mod.OracleScene(sc).render_batch(cam, 0.0, lv)
    for dedup in (1, 0):
        gsr.set_option("dedup", dedup)
        try:
            out, _, _, _ = _render(torch_mod, scene, cam, 0.0, lv)
        finally:
            gsr.set_option("dedup", 1)
        assert np.abs(out.cpu().numpy() - o_img).max() <= PIX_TOL
    scene.close()
    off = np.concatenate([sc.group_off, np.full(4, sc.group_off[-1], np.int32)])
    A = np.zeros((1, 3, 4), np.float32)
    bad = dataclasses.replace(sc, C=Cn + 1, group_off=off, A0=np.concatenate([sc.A0, A]), A1=np.concatenate([sc.A1, A]),
                              motion_scale=np.concatenate([sc.motion_scale, np.ones(1, np.float32)]))
    with pytest.raises(gsr.GsrError):
        gsr.Scene(bad)


def _limit_case(name):
    rng = np.random.default_rng(17)
    if name == "large_image_few_gaussians":          # 188 x 119 tiles: 16-bit tile indices, 2-3 radix passes on them
        n = 50
        sc, _ = tiny_scene(rng.uniform(-1, 1, (n, 3)), rng.uniform(0.05, 0.3, (n, 3)), logits=rng.uniform(-1, 3, n),
                           colors=rng.uniform(0.1, 0.9, (n, 3)), levels=rng.integers(0, 4, n),
                           clusters=rng.integers(0, 2, n), C=2, background=(0.2, 0.2, 0.2))
        return sc, axis_camera(W=3000, H=1900, f=1800.0, z0=4.0), synth.all_closed_states(2)[[0, 12, 24]]
    if name == "footprints_covering_every_tile":     # 3-sigma radius far larger than the image
        n = 40
        sc, _ = tiny_scene(rng.uniform(-0.5, 0.5, (n, 3)), rng.uniform(3.0, 20.0, (n, 3)), logits=rng.uniform(-3, 0, n),
                           colors=rng.uniform(0.1, 0.9, (n, 3)), levels=rng.integers(0, 4, n),
                           clusters=rng.integers(0, 3, n), C=3)
        return sc, axis_camera(W=320, H=200, f=200.0, z0=30.0), synth.all_closed_states(3)[::9]
    if name == "extreme_opacity_and_tiny_scales":    # tau = ln(255 o) from -24 to +5.5; Sigma' = dilation only
        n = 300
        sc, _ = tiny_scene(rng.uniform(-0.5, 0.5, (n, 3)), rng.choice([1e-6, 1e-3, 0.05], (n, 3)),
                           logits=rng.choice([-30.0, -6.0, 0.0, 30.0], n), colors=rng.uniform(0.1, 0.9, (n, 3)),
                           levels=rng.integers(0, 4, n), clusters=rng.integers(0, 3, n), C=3, background=(1, 1, 1))
        return sc, axis_camera(W=160, H=120, f=150.0, z0=3.0), synth.all_closed_states(3)[::9]
    n = 100                                          # everything_behind_or_outside: no key at all
    sc, _ = tiny_scene(np.c_[rng.uniform(-50, 50, n), rng.uniform(-50, 50, n), rng.uniform(-20, -5, n)], 0.1,
                       levels=rng.integers(0, 4, n), clusters=rng.integers(0, 2, n), C=2, background=(0.3, 0.6, 0.9))
    return sc, axis_camera(W=64, H=48, f=60.0, z0=3.0), synth.all_closed_states(2)[::5]


@pytest.mark.parametrize("name", ["large_image_few_gaussians", "footprints_covering_every_tile",
                                  "extreme_opacity_and_tiny_scales", "everything_behind_or_outside"])
def test_limit_cases(gsr, torch_mod, oracle_mod, name):
    sc, cam, lv = _limit_case(name)
    scene = gsr.Scene(sc)
    out, _, _, ws = _render(torch_mod, scene, cam, 0.0, lv)
    o_img, o_stats = oracle_mod.OracleScene(sc).render_batch(cam, 0.0, lv)
    assert np.array_equal(scene.debug_state_counts(ws, lv.shape[0]), o_stats[:, 0])
    assert np.abs(out.cpu().numpy() - o_img).max() <= PIX_TOL
    if name == "everything_behind_or_outside":
        assert scene.status(ws) == 0
    scene.close()


def test_invalid_level_and_key_capacity_are_reported(gsr, torch_mod):
    wl = synth.workload_cfg0()
    cam, t = wl.frames[0]
    scene = gsr.Scene(wl.scene)
    lv = wl.levels[0][:8].copy()
    lv[3, 2] = 4
    ws = scene.new_workspace(cam, 8)
    scene.render_states(cam, t, _dev_levels(torch_mod, lv), workspace=ws)
    with pytest.raises(gsr.GsrError) as e:
        scene.status(ws)
    assert e.value.code == gsr.GSR_E_INVALID_LEVEL
    ws = scene.new_workspace(cam, 8, key_capacity=100)       # far too few keys for this frame
    out, _, _ = scene.render_states(cam, t, _dev_levels(torch_mod, wl.levels[0][:8]), workspace=ws)
    with pytest.raises(gsr.GsrError) as e:
        scene.status(ws)
    assert e.value.code == gsr.GSR_E_WORKSPACE_TOO_SMALL
    with pytest.raises(gsr.GsrError):
        scene.render_states(cam, t, _dev_levels(torch_mod, wl.levels[0][:8]),
                            workspace=torch_mod.empty(1024, dtype=torch_mod.uint8, device="cuda"))
    # an image whose float count does not fit 32 bits is refused up front (include/gsr.h: gsr_camera)
    import dataclasses
    huge = dataclasses.replace(cam, W=40000, H=40000)
    with pytest.raises(gsr.GsrError):
        scene.workspace_bytes(huge, 1)
    scene.close()


def test_host_buffer_frame_call_matches_device_calls(gsr, torch_mod):
    wl = synth.scaled_object_workload(16, C=8, per_cluster=800.0, W=200, H=136, fov=40.0, n_frames=1, B=32)
    cam, t = wl.frames[0]
    lv = wl.levels[0]
    scene = gsr.Scene(wl.scene)
    mse_h, psnr_h, util_h, out_h, _ = scene.utility_frame_host(cam, t, lv, wl.idx_without[0], wl.idx_with[0],
                                                               wl.group_id[0], wl.G, want_images=True)
    full = np.full((1, wl.scene.C), 3, np.int8)
    ref_img, _, _, _ = _render(torch_mod, scene, cam, t, full)
    out, mse, psnr, _ = _render(torch_mod, scene, cam, t, lv, ref=ref_img[0].contiguous())
    assert np.array_equal(out.cpu().numpy(), out_h)
    assert np.array_equal(mse.cpu().numpy(), mse_h) and np.array_equal(psnr.cpu().numpy(), psnr_h)
    u, _, _ = gsr.group_utility(mse, psnr, torch_mod.from_numpy(wl.idx_without[0]).cuda(),
                                torch_mod.from_numpy(wl.idx_with[0]).cuda(),
                                torch_mod.from_numpy(wl.group_id[0]).cuda(), wl.G)
    for name in u.dtype.names:
        assert np.array_equal(u[name], util_h[name])
    scene.close()


# ------------------------------------------------------------------------------------------ dedup / culling
def test_tile_dedup_is_bitwise_neutral_and_hash_mode(gsr, torch_mod, oracle_mod):
    """24 clusters piled on the same screen area: more than 21 clusters per tile, so the dedup keys are
    hashes (exactly verified); plus duplicated states.  Dedup on/off must give identical bits."""
    rng = np.random.default_rng(21)
    C, per = 24, 40
    n = C * per
    clu = np.repeat(np.arange(C), per)
    lev = rng.integers(0, 4, n)
    means = rng.uniform(-0.25, 0.25, (n, 3))
    sc, _ = tiny_scene(means, rng.uniform(0.03, 0.08, (n, 3)), quats=rng.standard_normal((n, 4)),
                       logits=rng.normal(0.5, 1.0, n), colors=rng.uniform(0, 1, (n, 3)), levels=lev, clusters=clu,
                       C=C, sh_degree=1, R=2, background=(0.3, 0.3, 0.3),
                       motion_q=rng.integers(-100, 100, (n, 2, 3)).astype(np.int8),
                       motion_scale=np.full(C, 2e-4), sh_res=0.05 * rng.standard_normal((n, 4, 3)))
    cam = axis_camera(W=72, H=56, f=120.0)
    lv = synth.sample_levels(rng, 96, C)
    lv[40:60] = lv[0:20]                      # exact duplicates
    lv[60:80] = lv[0:20]
    lv[60:80, 5] = np.where(lv[60:80, 5] < 3, lv[60:80, 5] + 1, 2)   # pairs differing in one cluster
    scene = gsr.Scene(sc)
    osc = oracle_mod.OracleScene(sc)
    out, _, _, _ = _render(torch_mod, scene, cam, 0.4, lv)
    gsr.set_option("dedup", 0)
    try:
        out_nd, _, _, _ = _render(torch_mod, scene, cam, 0.4, lv)
    finally:
        gsr.set_option("dedup", 1)
    assert torch_mod.equal(out, out_nd)
    assert torch_mod.equal(out[40:60], out[0:20])
    ref, _ = osc.render_batch(cam, 0.4, lv)
    assert np.abs(out.cpu().numpy() - ref).max() <= PIX_TOL
    for b in (0, 47, 95):
        one, _, _, _ = _render(torch_mod, scene, cam, 0.4, lv[b:b + 1])
        assert torch_mod.equal(one[0], out[b])
    scene.close()


def test_subtile_culling_never_drops_a_contribution(gsr, torch_mod, oracle_mod):
    """Needle-like, strongly rotated, nearly opaque Gaussians (ill-conditioned conics) and faint ones
    (tau near 0): the conservative culling boxes must keep every pixel that passes the cut."""
    rng = np.random.default_rng(22)
    n = 300
    means = np.stack([rng.uniform(-1.2, 1.2, n), rng.uniform(-0.9, 0.9, n), rng.uniform(-0.5, 0.5, n)], 1)
    scales = np.stack([rng.uniform(0.2, 0.6, n), rng.uniform(0.002, 0.01, n), rng.uniform(0.002, 0.01, n)], 1)
    logits = np.where(rng.uniform(size=n) < 0.5, 6.0, -5.2)        # o ~ 0.9975 or ~ 0.0055 (tau ~ 0.34)
    sc, _ = tiny_scene(means, scales, quats=rng.standard_normal((n, 4)), logits=logits,
                       colors=rng.uniform(0, 1, (n, 3)), levels=rng.integers(0, 4, n),
                       clusters=rng.integers(0, 3, n), C=3, background=(1.0, 1.0, 1.0))
    cam = axis_camera(W=160, H=120, f=110.0)
    lv = synth.all_closed_states(3)[::5]
    scene = gsr.Scene(sc)
    osc = oracle_mod.OracleScene(sc)
    out, _, _, _ = _render(torch_mod, scene, cam, 0.0, lv)
    ref, _ = osc.render_batch(cam, 0.0, lv)
    assert np.abs(out.cpu().numpy() - ref).max() <= PIX_TOL
    scene.close()


@pytest.mark.parametrize("aspect", [1.5, 6.0, 40.0])
def test_block_culling_by_minimum_of_q_keeps_every_contribution(gsr, torch_mod, oracle_mod, aspect):
    """The once-per-frame per-block culling (minimum of q over the 8x4 block, tile_render_lists in k_sort.cu) on its own
    ground: moderately elongated, randomly rotated Gaussians (conditioning 2 .. ~2000, below the kappa cut-off of
    the tight test) a few pixels wide, so that most footprints clip block corners and edges; strong and faint
    opacities.  The oracle culls nothing: a wrongly dropped block would show as a >= 1/255 pixel error."""
    rng = np.random.default_rng(int(aspect * 10))
    n = 1500
    means = np.stack([rng.uniform(-1.3, 1.3, n), rng.uniform(-1.0, 1.0, n), rng.uniform(-0.3, 0.3, n)], 1)
    s_small = rng.uniform(0.01, 0.05, n)
    scales = np.stack([s_small * aspect, s_small, s_small], 1)
    logits = np.where(rng.uniform(size=n) < 0.5, 3.0, -4.5)        # o ~ 0.95 or ~ 0.011 (tau ~ 1.0)
    sc, _ = tiny_scene(means, scales, quats=rng.standard_normal((n, 4)), logits=logits,
                       colors=rng.uniform(0, 1, (n, 3)), levels=rng.integers(0, 4, n),
                       clusters=rng.integers(0, 4, n), C=4, background=(0.0, 0.0, 0.0))
    cam = axis_camera(W=176, H=136, f=120.0)
    lv = synth.all_closed_states(4)[::9]
    scene = gsr.Scene(sc)
    osc = oracle_mod.OracleScene(sc)
    out, _, _, _ = _render(torch_mod, scene, cam, 0.0, lv)
    ref, _ = osc.render_batch(cam, 0.0, lv)
    assert np.abs(out.cpu().numpy() - ref).max() <= PIX_TOL
    scene.close()


def test_full_size_cfg1_frame_sampled_states(gsr, torch_mod, oracle_mod):
    """configs[1] at full size in the launch configuration bench.py times (B = 256, default state block,
    dedup on, fused distortion): sampled states element by element against the oracle, I_b for all."""
    wl = synth.workload_cfg1(n_frames=2)
    cam, t = wl.frames[1]
    lv = wl.levels[1]
    scene = gsr.Scene(wl.scene)
    osc = oracle_mod.OracleScene(wl.scene)
    B = lv.shape[0]
    ws = scene.new_workspace(cam, B)
    out = torch_mod.empty((B, cam.H, cam.W, 3), dtype=torch_mod.float32, device="cuda")
    ref = torch_mod.empty((cam.H, cam.W, 3), dtype=torch_mod.float32, device="cuda")
    mse = torch_mod.empty(B, dtype=torch_mod.float64, device="cuda")
    psnr = torch_mod.empty(B, dtype=torch_mod.float32, device="cuda")
    scene.render_states_vs_full(cam, t, _dev_levels(torch_mod, lv), ws, ref, mse, psnr, out=out)
    scene.status(ws)
    pick = [0, 37, 128, 255]
    o_img, o_stats = osc.render_batch(cam, t, np.concatenate([lv[pick], np.full((1, wl.scene.C), 3, np.int8)]))
    for k, b in enumerate(pick):
        assert np.abs(out[b].cpu().numpy() - o_img[k]).max() <= PIX_TOL, b
    assert np.abs(ref.cpu().numpy() - o_img[-1]).max() <= PIX_TOL
    o_mse, o_psnr = oracle_mod.distortion(o_img[:-1], o_img[-1])
    assert np.max(np.abs(psnr.cpu().numpy()[pick] - o_psnr)) <= DB_TOL
    counts = scene.debug_state_counts(ws, B)
    assert np.array_equal(counts[pick], o_stats[:-1, 0])
    # the unfused reduction over the materialised images gives the same bits as the fused one
    mse_u, psnr_u = gsr.distortion(out, ref)
    assert torch_mod.equal(mse_u, mse) and torch_mod.equal(psnr_u, psnr)
    scene.close()


def _full_size_sampled(gsr, torch, oracle_mod, wl, frame, pick, images):
    """A bench-sized frame in the launch configuration bench.py times (default state block, dedup on, fused
    distortion; images materialised or not): PSNR and I_b of sampled states against the oracle, their pixels
    through a one-state-at-a-time re-render (bitwise equal to the batch by the batched == serial property)."""
    cam, t = wl.frames[frame]
    lv = wl.levels[frame]
    scene = gsr.Scene(wl.scene)
    osc = oracle_mod.OracleScene(wl.scene)
    B = lv.shape[0]
    ws = scene.new_workspace(cam, B)
    out = torch.empty((B, cam.H, cam.W, 3), dtype=torch.float32, device="cuda") if images else None
    ref = torch.empty((cam.H, cam.W, 3), dtype=torch.float32, device="cuda")
    mse = torch.empty(B, dtype=torch.float64, device="cuda")
    psnr = torch.empty(B, dtype=torch.float32, device="cuda")
    scene.render_states_vs_full(cam, t, _dev_levels(torch, lv), ws, ref, mse, psnr, out=out)
    scene.status(ws)
    counts = scene.debug_state_counts(ws, B)
    o_img, o_stats = osc.render_batch(cam, t, np.concatenate([lv[pick], np.full((1, wl.scene.C), 3, np.int8)]))
    assert np.abs(ref.cpu().numpy() - o_img[-1]).max() <= PIX_TOL
    _, o_psnr = oracle_mod.distortion(o_img[:-1], o_img[-1])
    assert np.max(np.abs(psnr.cpu().numpy()[pick] - o_psnr)) <= DB_TOL
    assert np.array_equal(counts[pick], o_stats[:-1, 0])
    ws1 = scene.new_workspace(cam, 1)
    for k, b in enumerate(pick):
        o1, m1, _ = scene.render_states(cam, t, _dev_levels(torch, lv[b:b + 1]), workspace=ws1, ref=ref)
        scene.status(ws1)
        assert np.abs(o1[0].cpu().numpy() - o_img[k]).max() <= PIX_TOL, b
        assert torch.equal(m1[0], mse[b])                          # batched == serial, bitwise
        if images:
            assert torch.equal(o1[0], out[b])
    scene.close()


def test_full_size_cfg2_frame_sampled_states(gsr, torch_mod, oracle_mod):
    """configs[2]: 64 clusters, ~300 k Gaussians, 536 x 960 (ragged tiles), B = 512, images materialised."""
    _full_size_sampled(gsr, torch_mod, oracle_mod, synth.workload_cfg2(n_frames=1), 0, [0, 255, 511], images=True)


def test_full_size_cfg3_view_sampled_states(gsr, torch_mod, oracle_mod):
    """configs[3]: one view of the utility sweep, B = 6144 paired states, no images (fused distortion only)."""
    _full_size_sampled(gsr, torch_mod, oracle_mod, synth.workload_cfg3(n_views=1), 0, [0, 3071, 3072, 6143],
                       images=False)


def test_full_size_cfg4_time_step_sampled_states(gsr, torch_mod, oracle_mod):
    """configs[4]: 128 clusters, ~1 M Gaussians, 1920 x 1080, one time step of 256 states, no images."""
    _full_size_sampled(gsr, torch_mod, oracle_mod, synth.workload_cfg4(), 2, [0, 100, 255], images=False)

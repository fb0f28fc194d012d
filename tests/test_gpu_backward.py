"""GPU parity of gsr_render_backward (include/gsr.h) against the backward oracle (oracle O-8) through
the C ABI: for a batch of states with random dL/d(image), the per-record gradients summed over the states.
Floating point with atomics: by tolerance (stated per test), never bitwise."""
import numpy as np
import pytest

from paper_2606_17212_b200 import synth
from tests.test_backward_pins import smooth_scene
from tests.helpers import axis_camera, tiny_scene

pytestmark = pytest.mark.gpu


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


def oracle_record_grads(oracle_mod, scn, cam, t, lv, g, V=2):
    """The oracle's per-state [N, 9] gradients mapped onto the records the GPU composites and summed over states:
    record = V i + variant (V = 2: variant 0 at cluster depth 0, else 1; V = 4: variant = depth); columns
    (rgb[3], rgb with SH residual[3], opacity, A, B, Cq, mx, my) — depth 3 uses the second colour (V = 2)."""
    osc = oracle_mod.OracleScene(scn)
    N = scn.N
    cl = scn.cluster_of()
    out, out_abs = np.zeros((V * N, 12)), np.zeros((V * N, 12))
    for b in range(lv.shape[0]):
        gr, ga = osc.backward(cam, t, lv[b], g[b].astype(np.float64), want_abs=True)
        d = lv[b][cl].astype(np.int64)
        variant = np.where(d == 0, 0, 1) if V == 2 else np.clip(d, 0, 3)
        rid = V * np.arange(N) + variant
        live = np.any(gr != 0.0, axis=1)
        col = np.where((d == 3) & (V == 2), 3, 0)
        for i in np.nonzero(live)[0]:
            out[rid[i], col[i]:col[i] + 3] += gr[i, :3]
            out[rid[i], 6:] += gr[i, 3:]
            out_abs[rid[i], col[i]:col[i] + 3] += ga[i, :3]
            out_abs[rid[i], 6:] += ga[i, 3:]
    return out, out_abs


def _run(gsr, torch, scn, cam, t, lv, seed):
    scene = gsr.Scene(scn)
    ws = scene.new_workspace(cam, lv.shape[0])
    dlv = torch.from_numpy(np.ascontiguousarray(lv, np.int8)).cuda()
    out, _, _ = scene.render_states(cam, t, dlv, workspace=ws)
    scene.status(ws)
    rng = np.random.default_rng(seed)
    g = rng.standard_normal(tuple(out.shape)).astype(np.float32)
    grad = scene.render_backward(ws, out, torch.from_numpy(g).cuda()).cpu().numpy().astype(np.float64)
    V = scene.num_records() // scn.N
    scene.close()
    return grad, g, V


def _compare(got, want_and_abs, k_eps=64.0):
    """Every entry is a sum of many signed fp32 terms (per pixel and state; atomics order on the GPU, double in the
    oracle), often strongly cancelling (dB on a symmetric footprint).  The bar is the floating-point one:
    |got - want| <= k_eps * 2^-24 * (the entry's magnitude: every product in absolute value, the suffix of a pixel
    counted as everything the pixel is made of — the kernel forms it as final pixel minus prefix), from the oracle
    (grad_abs).  The GPU's factors carry ~1e-6 relative error each (fp32 alpha, ex2.approx, rcp, the fp32 forward
    pixel), hence k_eps = 64."""
    want, wabs = want_and_abs
    err = np.abs(got - want)
    bound = k_eps * 2.0 ** -24 * wabs
    bad = err > bound + 1e-30
    assert not bad.any(), (np.argwhere(bad)[:5], err[bad][:5], bound[bad][:5])
    # and in relative terms wherever the sum is not dominated by cancellation
    solid = np.abs(want) > 0.05 * wabs
    assert np.all(err[solid] <= 2e-4 * np.abs(want[solid]))
    # records no state composites have exactly zero gradient on both sides
    dead = ~np.any(wabs != 0.0, axis=1)
    assert np.all(got[dead] == 0.0)


def test_backward_smooth_three_gaussians(gsr, torch_mod, oracle_mod):
    scn, cam = smooth_scene()
    lv = np.zeros((1, 1), np.int8)
    got, g, V = _run(gsr, torch_mod, scn, cam, 0.0, lv, 1)
    want = oracle_record_grads(oracle_mod, scn, cam, 0.0, lv, g, V)
    _compare(got, want)


def test_backward_cap_and_stop(gsr, torch_mod, oracle_mod):
    cam = axis_camera(32, 32, 100.0, 4.0, cx=16.5, cy=16.5)
    lv = np.zeros((1, 1), np.int8)
    scn, _ = tiny_scene([[0, 0, 0]], 20.0, logits=12.0, colors=(0.5, 0.5, 0.5))          # capped everywhere
    got, g, V = _run(gsr, torch_mod, scn, cam, 0.0, lv, 2)
    want = oracle_record_grads(oracle_mod, scn, cam, 0.0, lv, g, V)
    _compare(got, want)
    assert np.all(got[:, 6:] == 0.0)
    scn, _ = tiny_scene([[0, 0, 0.01 * k] for k in range(20)], 5.0, logits=0.0, colors=(0.7, 0.7, 0.7))   # stop after 13
    got, g, V = _run(gsr, torch_mod, scn, cam, 0.0, lv, 3)
    want = oracle_record_grads(oracle_mod, scn, cam, 0.0, lv, g, V)
    _compare(got, want)
    assert (np.any(got != 0.0, axis=1)).sum() == 13


@pytest.mark.parametrize("bg", [(0.0, 0.0, 0.0), (1.0, 1.0, 1.0)])
def test_backward_batch_of_states_scaled_scene(gsr, torch_mod, oracle_mod, bg):
    wl = synth.scaled_object_workload(23, C=5, per_cluster=260.0, W=120, H=88, fov=40.0, n_frames=1, B=14)
    wl.scene.background = np.asarray(bg, np.float32)
    cam, t = wl.frames[0]
    lv = wl.levels[0].copy()
    lv[0] = 3
    lv[1] = -1
    lv[2] = 0                                               # all-full, all-absent and all-base states among them
    got, g, V = _run(gsr, torch_mod, wl.scene, cam, t, lv, 4)
    want = oracle_record_grads(oracle_mod, wl.scene, cam, t, lv, g, V)
    assert np.any(want[0][:, 3:6] != 0.0) and np.any(want[0][0::2] != 0.0)   # both colours and both variants occur
    _compare(got, want)


def test_backward_refuses_a_workspace_of_another_batch(gsr, torch_mod):
    scn, cam = smooth_scene()
    scene = gsr.Scene(scn)
    ws = scene.new_workspace(cam, 2)
    lv = torch_mod.zeros((2, 1), dtype=torch_mod.int8, device="cuda")
    out, _, _ = scene.render_states(cam, 0.0, lv, workspace=ws)
    with pytest.raises(gsr.GsrError):
        scene.render_backward(ws, out[:1].contiguous(), out[:1].contiguous())
    scene.close()


def test_backward_four_variant_scene(gsr, torch_mod, oracle_mod):
    """Scenes with position residual levels / attribute refinements project FOUR records per Gaussian (record =
    4 i + cluster depth, one colour each): the gradients land on the variant the state composites."""
    wl = synth.scaled_object_workload(29, C=4, per_cluster=220.0, W=104, H=72, fov=40.0, n_frames=1, B=10)
    scn = synth.with_attribute_refinements(synth.with_position_residuals(wl.scene))
    cam, t = wl.frames[0]
    lv = wl.levels[0].copy()
    lv[0], lv[1], lv[2], lv[3] = 3, 2, 1, 0
    got, g, V = _run(gsr, torch_mod, scn, cam, t, lv, 6)
    assert V == 4
    want = oracle_record_grads(oracle_mod, scn, cam, t, lv, g, V)
    assert all(np.any(want[0][v::4] != 0.0) for v in range(4))           # every variant receives gradient
    assert np.all(got[:, 3:6] == 0.0)                                    # one colour per record: the second triple is unused
    _compare(got, want)


def test_backward_full_size_cfg1_identities(gsr, torch_mod):
    """configs[1] at full size (800x800, B = 256, the batch bench.py times): two properties that hold at any size.
    (1) Colour identity: pixel - bg = sum_i w_i (c_i - bg) and dL/dc_i = sum w_i g, hence
        sum_records (c - bg) . dL/dc = sum_{state, pixel} g . (image - bg)   (both colour triples, fp32 sums).
    (2) Batch consistency: the gradient of a batch whose dL/d(image) is non-zero for ONE state equals the gradient
        of that state rendered alone with the same dL/d(image) (other state block, other presence tables)."""
    torch = torch_mod
    wl = synth.workload_cfg1(n_frames=2)
    cam, t = wl.frames[1]
    lv = wl.levels[1]
    B = lv.shape[0]
    scene = gsr.Scene(wl.scene)
    ws = scene.new_workspace(cam, B)
    dlv = torch.from_numpy(np.ascontiguousarray(lv)).cuda()
    out, _, _ = scene.render_states(cam, t, dlv, workspace=ws)
    scene.status(ws)
    gen = torch.Generator(device="cuda").manual_seed(11)
    g = torch.randn(out.shape, generator=gen, device="cuda", dtype=torch.float32)
    grad = scene.render_backward(ws, out, g).double()
    P = scene.debug_projection(ws)
    bg = torch.from_numpy(np.asarray(wl.scene.background, np.float64)).cuda()
    c0 = torch.from_numpy(P["rgb_base"].astype(np.float64)).cuda() - bg
    c1 = torch.from_numpy(P["rgb_res"].astype(np.float64)).cuda() - bg
    lhs = float((c0 * grad[:, 0:3]).sum() + (c1 * grad[:, 3:6]).sum())
    rhs = float((g.double() * (out.double() - bg)).sum())
    mag = float((c0.abs() * grad[:, 0:3].abs()).sum() + (c1.abs() * grad[:, 3:6].abs()).sum())
    assert abs(lhs - rhs) <= 2e-5 * mag, (lhs, rhs, mag)
    # (2) one state of the batch alone
    b = 137
    g1 = torch.zeros_like(g)
    g1[b] = g[b]
    grad_b = scene.render_backward(ws, out, g1)
    ws1 = scene.new_workspace(cam, 1)
    out1, _, _ = scene.render_states(cam, t, dlv[b:b + 1].contiguous(), workspace=ws1)
    assert torch.equal(out1[0], out[b])
    grad_1 = scene.render_backward(ws1, out1, g[b:b + 1].contiguous())
    scale = grad_1.abs().amax(dim=0).clamp_min(1e-20)
    assert float(((grad_b - grad_1).abs() / scale).max()) <= 2e-4
    assert bool((grad_b != 0).any())
    scene.close()


def test_backward_shared_tile_classes_against_the_oracle(gsr, torch_mod, oracle_mod):
    """States with identical pixels in a tile are walked once with the SUM of their dL/d(image):
    a batch made of utility pairs (m, m u g: they differ in one cluster) plus exact duplicates, each state with its
    own random g — against the oracle, which differentiates every state on its own."""
    wl = synth.scaled_object_workload(31, C=6, per_cluster=240.0, W=112, H=80, fov=40.0, n_frames=1, B=6)
    cam, t = wl.frames[0]
    base = wl.levels[0]
    rows = []
    for b in range(base.shape[0]):
        rows.append(base[b].copy())
        up = base[b].copy()
        up[b % up.shape[0]] = min(3, up[b % up.shape[0]] + 1)     # the pair state: one cluster one level further
        rows.append(up)
        rows.append(base[b].copy())                               # an exact duplicate
    lv = np.stack(rows).astype(np.int8)
    got, g, V = _run(gsr, torch_mod, wl.scene, cam, t, lv, 8)
    want = oracle_record_grads(oracle_mod, wl.scene, cam, t, lv, g, V)
    _compare(got, want)


def test_backward_dedup_option_off_gives_the_same_gradient(gsr, torch_mod):
    """configs[1], full size: the class-summed walk (default) against one walk per state (option dedup = 0)."""
    torch = torch_mod
    wl = synth.workload_cfg1(n_frames=1)
    cam, t = wl.frames[0]
    dlv = torch.from_numpy(np.ascontiguousarray(wl.levels[0])).cuda()
    scene = gsr.Scene(wl.scene)
    ws = scene.new_workspace(cam, dlv.shape[0])
    out, _, _ = scene.render_states(cam, t, dlv, workspace=ws)
    scene.status(ws)
    gen = torch.Generator(device="cuda").manual_seed(12)
    g = torch.randn(out.shape, generator=gen, device="cuda", dtype=torch.float32)
    grad_on = scene.render_backward(ws, out, g).clone()
    gsr.set_option("dedup", 0)
    try:
        grad_off = scene.render_backward(ws, out, g).clone()
    finally:
        gsr.set_option("dedup", 1)
    scale = grad_off.abs().amax(dim=0).clamp_min(1e-20)
    assert float(((grad_on - grad_off).abs() / scale).max()) <= 2e-4
    assert bool((grad_on != 0).any())
    scene.close()


def test_backward_maximum_cluster_count(gsr, torch_mod, oracle_mod):
    """C = 4096, the documented maximum: the presence table (8 bytes per cluster) plus the kernel's static shared
    memory pass the default 48 KB, so the launch needs the opt-in; against the oracle, with and without dedup."""
    rng = np.random.default_rng(4097)
    Cn, n = 4096, 6000
    scn, _ = tiny_scene(rng.uniform(-0.8, 0.8, (n, 3)), rng.uniform(0.03, 0.08, (n, 3)), logits=rng.uniform(-1, 3, n),
                        colors=rng.uniform(0.1, 0.9, (n, 3)), levels=rng.integers(0, 4, n), clusters=np.arange(n) % Cn,
                        C=Cn, background=(0.1, 0.1, 0.1))
    cam = axis_camera(W=64, H=48, f=60.0, z0=3.0)
    lv = synth.sample_levels(rng, 5, Cn)
    for dedup in (1, 0):
        gsr.set_option("dedup", dedup)
        try:
            got, g, V = _run(gsr, torch_mod, scn, cam, 0.0, lv, 9)
        finally:
            gsr.set_option("dedup", 1)
        want = oracle_record_grads(oracle_mod, scn, cam, 0.0, lv, g, V)
        _compare(got, want)

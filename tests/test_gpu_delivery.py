"""GPU parity of gsr_sample_delivery (include/gsr.h) against oracle/delivery.py through the
C ABI: masks and levels are integer work, BIT-EXACT.  Also: the sampled levels feed gsr_render_states."""
import numpy as np
import pytest

from oracle import delivery as D
from paper_2606_17212_b200 import synth

pytestmark = pytest.mark.gpu

MODELS = [
    dict(p_iid=0.0, p_gb=0.0, p_bg=0.0, e_good=0.0, e_bad=0.0, seed=1),
    dict(p_iid=0.05, p_gb=0.0, p_bg=0.0, e_good=0.0, e_bad=0.0, seed=2),
    dict(p_iid=0.0, p_gb=0.03, p_bg=0.25, e_good=0.0, e_bad=0.8, seed=0xDEADBEEFCAFEF00D),
    dict(p_iid=0.02, p_gb=0.1, p_bg=0.1, e_good=0.01, e_bad=0.5, seed=(1 << 63) + 12345),
    dict(p_iid=1.0, p_gb=0.5, p_bg=0.5, e_good=1.0, e_bad=1.0, seed=7),
]


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


def _dev(torch, a, dtype):
    return torch.from_numpy(np.ascontiguousarray(a, dtype)).cuda()


@pytest.mark.parametrize("C,W", [(1, 3), (3, 9), (17, 6), (40, 5)])
@pytest.mark.parametrize("mi", range(len(MODELS)))
def test_masks_and_levels_bit_exact(gsr, torch_mod, C, W, mi):
    rng = np.random.default_rng(1000 * C + W + mi)
    raw = rng.integers(0, 9000, 4 * C)                       # 0..8 packets per group: spans several 32-packet steps
    raw[rng.integers(0, 4 * C, max(1, C // 2))] = 0          # empty groups, also consecutive ones
    raw[rng.integers(0, 4 * C, max(1, C // 2))] = 1200 * rng.integers(1, 4)
    # a dependency-consistent but non-trivial send order: clusters shuffled, levels interleaved
    order = np.array([4 * c + l for l in range(4) for c in rng.permutation(C)], np.int32)
    model = MODELS[mi]
    n_pk = int(D.packets_per_group(raw).sum())
    budget = rng.integers(0, n_pk + 5, W).astype(np.int32)
    for b in (None, budget):
        m_ref, l_ref = D.sample_delivery(raw, order, C, model, W, packet_budget=b, world0=11)
        m, l = gsr.sample_delivery(_dev(torch_mod, raw, np.int64), _dev(torch_mod, order, np.int32), model, W,
                                   packet_budget=None if b is None else _dev(torch_mod, b, np.int32), world0=11)
        assert np.array_equal(m.cpu().numpy(), m_ref), (C, W, mi, b is None)
        assert np.array_equal(l.cpu().numpy(), l_ref)


def test_worlds_do_not_depend_on_batching(gsr, torch_mod):
    rng = np.random.default_rng(3)
    C = 12
    raw = _dev(torch_mod, rng.integers(0, 20000, 4 * C), np.int64)
    order = _dev(torch_mod, np.arange(4 * C), np.int32)
    m, l = gsr.sample_delivery(raw, order, MODELS[3], 64)
    m2, l2 = gsr.sample_delivery(raw, order, MODELS[3], 10, world0=37)
    assert torch_mod.equal(m[37:47], m2) and torch_mod.equal(l[37:47], l2)


def test_sampled_levels_feed_the_renderer(gsr, torch_mod, oracle_mod):
    """End of the chain: wire order -> sampled delivery -> levels -> render; pixels against the oracle."""
    torch = torch_mod
    wl = synth.scaled_object_workload(8, C=6, per_cluster=200, W=64, H=48, fov=40.0, n_frames=1, B=4)
    cam, t = wl.frames[0]
    raw = synth.group_raw_bytes(wl.scene)
    d_raw = _dev(torch, raw, np.int64)
    wire = gsr.group_wire_bytes(d_raw)
    order, _ = gsr.frontier_order(None, wire, gsr.POLICY_NOMINAL)
    model = dict(p_iid=0.002, p_gb=0.002, p_bg=0.2, e_good=0.0, e_bad=0.6, seed=42)
    Wn = 12
    mask, levels = gsr.sample_delivery(d_raw, order, model, Wn)
    m_ref, l_ref = D.sample_delivery(raw, order.cpu().numpy(), wl.scene.C, model, Wn)
    assert np.array_equal(levels.cpu().numpy(), l_ref) and np.array_equal(mask.cpu().numpy(), m_ref)
    assert len({tuple(r) for r in l_ref.tolist()}) > 1          # the channel really produces partial states
    d2, _ = gsr.close_levels(mask)                              # the sampler's closure == gsr_close_levels
    assert torch.equal(d2, levels)
    scene = gsr.Scene(wl.scene)
    ws = scene.new_workspace(cam, Wn)
    out, _, _ = scene.render_states(cam, t, levels, workspace=ws)
    scene.status(ws)
    o_img, _ = oracle_mod.OracleScene(wl.scene).render_batch(cam, t, l_ref)
    assert np.abs(out.cpu().numpy() - o_img).max() <= 2e-4

"""GPU parity of the scheduling-frontier / atlas calls (include/gsr.h) against
oracle/policy.py through the C ABI.  All of it is integer / comparison work: BIT-EXACT.  Also: a batch
larger than the tile-dedup sort (chunked internally) equals the same states rendered in small batches."""
import numpy as np
import pytest

from oracle import policy as P
from paper_2606_17212_b200 import synth

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


def _dev(torch, a, dtype):
    return torch.from_numpy(np.ascontiguousarray(a, dtype)).cuda()


@pytest.mark.parametrize("C", [1, 2, 33, 300])
def test_wire_bytes_and_orders_bit_exact(gsr, torch_mod, C):
    rng = np.random.default_rng(100 + C)
    raw = rng.integers(0, 200000, 4 * C)
    raw[rng.integers(0, 4 * C, max(1, C // 3))] = 0                  # empty groups
    raw[rng.integers(0, 4 * C, max(1, C // 3))] = 1200 * rng.integers(1, 5)  # exact chunk multiples
    wire_o = P.group_wire_bytes(raw)
    wire = gsr.group_wire_bytes(_dev(torch_mod, raw, np.int64))
    assert np.array_equal(wire.cpu().numpy(), wire_o)
    score = rng.normal(size=4 * C).round(1)                          # rounded: many ties; includes -0.0 / 0.0
    score[::7] = 0.0
    score[3::11] = -0.0
    for policy in (P.POLICY_UTILITY, P.POLICY_NOMINAL, P.POLICY_BYTE_GREEDY):
        o_ref, c_ref = P.frontier_order(score, wire_o, C, policy)
        o, c = gsr.frontier_order(_dev(torch_mod, score, np.float64), wire, policy)
        assert np.array_equal(o.cpu().numpy(), o_ref), f"policy {policy}"
        assert np.array_equal(c.cpu().numpy(), c_ref)
        budgets = np.concatenate([[-5, 0], c_ref[:: max(1, C // 4)], c_ref[-1:] - 1, c_ref[-1:], [2 ** 40]])
        lv_ref, used_ref, n_ref = P.frontier_states(o_ref, wire_o, C, budgets)
        lv, used, n = gsr.frontier_states(o, wire, _dev(torch_mod, budgets, np.int64))
        assert np.array_equal(lv.cpu().numpy(), lv_ref)
        assert np.array_equal(used.cpu().numpy(), used_ref)
        assert np.array_equal(n.cpu().numpy(), n_ref)


def test_hand_worked_example_on_gpu(gsr, torch_mod):
    raw = np.array([1000, 1200, 1201, 0, 2400, 100, 5000, 1])
    wire = gsr.group_wire_bytes(_dev(torch_mod, raw, np.int64))
    assert wire.cpu().tolist() == [1048, 1252, 1313, 0, 2496, 152, 5280, 61]
    score = _dev(torch_mod, [5, 1, 9, 2, 7, 8, -1, 3], np.float64)
    o, c = gsr.frontier_order(score, wire, gsr.POLICY_UTILITY)
    assert o.cpu().tolist() == [4, 5, 0, 1, 2, 3, 6, 7]
    assert c.cpu().tolist() == [2496, 2648, 3696, 4948, 6261, 6261, 11541, 11602]
    lv, used, n = gsr.frontier_states(o, wire, _dev(torch_mod, [0, 2496, 3000, 6261, 11601, 20000], np.int64))
    assert lv.cpu().numpy().reshape(-1).tolist() == [-1, -1, -1, 0, -1, 1, 3, 1, 3, 2, 3, 3]
    assert used.cpu().tolist() == [0, 2496, 2648, 6261, 11541, 11602]


@pytest.mark.parametrize("B,C", [(1, 1), (37, 5), (4099, 32), (513, 130)])
def test_state_bytes_and_best_state_bit_exact(gsr, torch_mod, B, C):
    rng = np.random.default_rng(B + C)
    wire = rng.integers(0, 50000, 4 * C)
    lv = rng.integers(-1, 4, size=(B, C)).astype(np.int8)
    cost_ref = P.state_bytes(lv, wire)
    cost = gsr.state_bytes(_dev(torch_mod, lv, np.int8), _dev(torch_mod, wire, np.int64))
    assert np.array_equal(cost.cpu().numpy(), cost_ref)
    psnr = rng.normal(25, 3, B).round(1).astype(np.float32)          # ties
    budgets = np.concatenate([[-1, 0], np.quantile(cost_ref, [0.1, 0.5, 0.9]).astype(np.int64), [2 ** 50]])
    best_ref = P.best_state_under_budget(psnr, cost_ref, budgets)
    best = gsr.best_state_under_budget(_dev(torch_mod, psnr, np.float32), cost, _dev(torch_mod, budgets, np.int64))
    assert np.array_equal(best.cpu().numpy(), best_ref)


def test_batch_above_dedup_capacity_equals_small_batches(gsr, torch_mod):
    """B = 8197 (the paper's atlas size) exceeds the 8192-state tile-dedup sort and is
    composited in chunks: distortions must be bitwise those of the same states in batches of 1000."""
    torch = torch_mod
    wl = synth.scaled_object_workload(7, C=6, per_cluster=300, W=96, H=80, fov=40.0, n_frames=1, B=8)
    cam, t = wl.frames[0]
    rng = np.random.default_rng(4)
    lv = np.concatenate([synth.sample_levels(rng, 8192, wl.scene.C),
                         np.stack([np.full(wl.scene.C, d, np.int8) for d in range(-1, 4)])])
    assert lv.shape[0] == 8197
    scene = gsr.Scene(wl.scene)
    dlv = torch.from_numpy(lv).cuda()
    full = torch.full((1, wl.scene.C), 3, dtype=torch.int8, device="cuda")
    ws = scene.new_workspace(cam, lv.shape[0])
    ref, _, _ = scene.render_states(cam, t, full, workspace=ws)
    ref = ref[0].contiguous()
    out, mse, psnr = scene.render_states(cam, t, dlv, workspace=ws, ref=ref)
    scene.status(ws)
    assert float(mse[-1]) == 0.0                                     # the complete prefix is the reference
    for b0 in range(0, lv.shape[0], 1000):
        o2, m2, p2 = scene.render_states(cam, t, dlv[b0:b0 + 1000].contiguous(), workspace=ws, ref=ref)
        scene.status(ws)
        assert torch.equal(m2, mse[b0:b0 + 1000])
        assert torch.equal(p2, psnr[b0:b0 + 1000])
        assert torch.equal(o2, out[b0:b0 + 1000])

"""Smallest and largest sizes of the helper calls (include/gsr.h) against their oracle modules: SSIM on images
smaller than the 11x11 window, frontier orders at C = 1 and C = 4096, the delivery sampler with no packet and
with no world."""
import numpy as np
import pytest

from oracle import delivery as D
from oracle import metrics as M
from oracle import policy as P

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


@pytest.mark.parametrize("H,W,B", [(1, 1, 1), (1, 9, 2), (3, 2, 1), (11, 11, 1), (2000, 3, 1)])
def test_ssim_on_images_smaller_than_the_window(gsr, torch_mod, H, W, B):
    rng = np.random.default_rng(H * 31 + W)
    im = rng.uniform(0, 1, (B, H, W, 3)).astype(np.float32)
    ref = rng.uniform(0, 1, (H, W, 3)).astype(np.float32)
    got = gsr.distortion_ssim(_dev(torch_mod, im, np.float32), _dev(torch_mod, ref, np.float32))
    got = got[0] if isinstance(got, (tuple, list)) else got
    want = M.ssim(im.astype(np.float64), ref.astype(np.float64))
    assert np.abs(got.cpu().numpy() - want).max() <= 1e-9


@pytest.mark.parametrize("C", [1, 4096])
def test_frontier_at_the_smallest_and_largest_cluster_count(gsr, torch_mod, C):
    rng = np.random.default_rng(C)
    raw = rng.integers(0, 5000, 4 * C)
    wire = gsr.group_wire_bytes(_dev(torch_mod, raw, np.int64))
    w_ref = P.group_wire_bytes(raw)
    assert np.array_equal(wire.cpu().numpy(), w_ref)
    score = rng.normal(size=4 * C)
    for policy in (gsr.POLICY_UTILITY, gsr.POLICY_NOMINAL, gsr.POLICY_BYTE_GREEDY):
        order, cum = gsr.frontier_order(_dev(torch_mod, score, np.float64), wire, policy)
        o_ref, c_ref = P.frontier_order(score, w_ref, C, policy)
        assert np.array_equal(order.cpu().numpy(), o_ref) and np.array_equal(cum.cpu().numpy(), c_ref)


def test_delivery_sampler_without_packets_and_without_worlds(gsr, torch_mod):
    model = dict(p_iid=0.5, p_gb=0.1, p_bg=0.1, e_good=0.1, e_bad=0.9, seed=3)
    raw, order = np.zeros(4, np.int64), np.arange(4, dtype=np.int32)       # one cluster, four empty groups
    m, l = gsr.sample_delivery(_dev(torch_mod, raw, np.int64), _dev(torch_mod, order, np.int32), model, 5)
    m_ref, l_ref = D.sample_delivery(raw, order, 1, model, 5)
    assert np.array_equal(m.cpu().numpy(), m_ref) and np.array_equal(l.cpu().numpy(), l_ref)
    assert np.all(l_ref == 3)                                              # nothing to lose: everything usable (H1)
    raw = np.arange(12, dtype=np.int64) * 700
    m, l = gsr.sample_delivery(_dev(torch_mod, raw, np.int64), _dev(torch_mod, np.arange(12), np.int32), model, 0)
    assert tuple(m.shape) == (0, 3) and tuple(l.shape) == (0, 3)

"""Caller-supplied index arrays are range-checked on the device (include/gsr.h, gsr_index_status): an entry out of
range is skipped, latched, and reported — never dereferenced.  The results for the valid entries are unchanged."""
import numpy as np
import pytest

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


def test_group_utility_refuses_bad_pairs_and_keeps_the_valid_ones(gsr, torch_mod, oracle_mod):
    rng = np.random.default_rng(3)
    B, G, n = 500, 7, 900
    mse = rng.uniform(1e-5, 1e-2, B)
    psnr = (-10 * np.log10(mse)).astype(np.float32)
    iwo, iw = rng.integers(0, B, n).astype(np.int32), rng.integers(0, B, n).astype(np.int32)
    gid = rng.integers(0, G, n).astype(np.int32)
    gsr.index_status()                                                   # starts clean
    args = lambda a, b, g: (_dev(torch_mod, mse, np.float64), _dev(torch_mod, psnr, np.float32),
                            _dev(torch_mod, a, np.int32), _dev(torch_mod, b, np.int32), _dev(torch_mod, g, np.int32), G)
    u_ok, _, _ = gsr.group_utility(*args(iwo, iw, gid))
    for kind in ("index_high", "index_negative", "group"):
        a, b, g = iwo.copy(), iw.copy(), gid.copy()
        bad = rng.choice(n, 20, replace=False)
        if kind == "index_high":
            a[bad[:10]] = B
            b[bad[10:]] = B + 100000
        elif kind == "index_negative":
            a[bad] = -1
        else:
            g[bad[:10]] = G
            g[bad[10:]] = -3
        with pytest.raises(gsr.GsrError):
            gsr.group_utility(*args(a, b, g))
        gsr.index_status()                                               # the word was cleared by the read
        # the aggregation of the remaining pairs is what the oracle gives for them alone
        keep = np.ones(n, bool)
        keep[bad] = False
        util = torch_mod.zeros((G, 9), dtype=torch_mod.float64, device="cuda")
        gsr.group_utility_into(*args(a, b, g), util)
        torch_mod.cuda.synchronize()
        with pytest.raises(gsr.GsrError):
            gsr.index_status()
        _, _, o_u = oracle_mod.group_utility(mse, psnr, iwo[keep], iw[keep], gid[keep], G)
        assert np.allclose(util.cpu().numpy(), o_u, rtol=1e-9, atol=1e-15)
    # and the untouched call still gives the full result
    u2, _, _ = gsr.group_utility(*args(iwo, iw, gid))
    for name in oracle_mod.UTIL_FIELDS:
        assert np.array_equal(u_ok[name], u2[name])


def test_prefix_monotonicity_refuses_indices_outside_d(gsr, torch_mod):
    d = _dev(torch_mod, [3.0, 2.0, 2.5, 1.0], np.float64)
    prev, nxt = _dev(torch_mod, [0, 1, 2], np.int32), _dev(torch_mod, [1, 2, 3], np.int32)
    assert gsr.prefix_monotonicity(d, prev, nxt) == (0.5, 1)
    for bad in ([0, 1, 4], [0, -1, 2]):
        with pytest.raises(gsr.GsrError):
            gsr.prefix_monotonicity(d, _dev(torch_mod, bad, np.int32), nxt)
    assert gsr.prefix_monotonicity(d, prev, nxt) == (0.5, 1)


def test_send_order_entries_outside_the_groups_are_refused(gsr, torch_mod):
    C = 5
    raw = _dev(torch_mod, np.full(4 * C, 3000), np.int64)
    wire = gsr.group_wire_bytes(raw)
    order, _ = gsr.frontier_order(None, wire, 1)
    budgets = _dev(torch_mod, [10 ** 9], np.int64)
    lv, _, ng = gsr.frontier_states(order, wire, budgets)
    gsr.index_status()
    assert ng.item() == 4 * C and lv.cpu().numpy().tolist() == [[3] * C]
    bad = order.clone()
    bad[7] = 4 * C                                                        # not a group
    lv, _, ng = gsr.frontier_states(bad, wire, budgets)
    with pytest.raises(gsr.GsrError):
        gsr.index_status()
    assert ng.item() == 7                                                 # the walk stopped at the bad entry
    # delivery sampler: the bad entry sends nothing, every other group is sampled as before
    model = dict(p_iid=0.0, p_gb=0.0, p_bg=1.0, e_good=0.0, e_bad=0.0, seed=5)
    mask, levels = gsr.sample_delivery(raw, order, model, W=3)
    gsr.index_status()
    assert (levels.cpu().numpy() == 3).all()
    bad[7] = -2
    mask, levels = gsr.sample_delivery(raw, bad, model, W=3)
    with pytest.raises(gsr.GsrError):
        gsr.index_status()
    assert (levels.cpu().numpy() == 3).all()                               # no loss: nothing else is disturbed


def test_host_frame_call_checks_the_pair_lists_on_the_host(gsr, torch_mod):
    wl = synth.workload_cfg0()
    cam, t = wl.frames[0]
    scene = gsr.Scene(wl.scene)
    lv = np.ascontiguousarray(wl.levels[0][:8])
    good = (np.array([0, 1], np.int32), np.array([2, 3], np.int32), np.array([0, 1], np.int32))
    scene.utility_frame_host(cam, t, lv, *good, 2)
    for iwo, iw, gid in ((np.array([0, 8], np.int32), good[1], good[2]), (good[0], np.array([-1, 3], np.int32), good[2]),
                         (good[0], good[1], np.array([0, 2], np.int32))):
        with pytest.raises(gsr.GsrError):
            scene.utility_frame_host(cam, t, lv, iwo, iw, gid, 2)
    scene.close()

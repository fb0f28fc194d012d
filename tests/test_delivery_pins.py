"""Pins of oracle/delivery.py (Philox4x32-10, IID + Gilbert-Elliott packet loss, group usability, closure).
CPU-only: published known-answer vectors, degenerate channels, a hand-walked world, statistics."""
import math

import numpy as np
import pytest

from oracle import delivery as D

NO_LOSS = dict(p_iid=0.0, p_gb=0.0, p_bg=0.0, e_good=0.0, e_bad=0.0, seed=1)


def test_philox_known_answer_vectors():
    """The three Philox4x32-10 vectors published with the generator (Salmon et al., Random123 kat_vectors)."""
    assert D.philox4x32_10((0, 0, 0, 0), (0, 0)) == (0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8)
    f = 0xFFFFFFFF
    assert D.philox4x32_10((f, f, f, f), (f, f)) == (0x408F276D, 0x41C83B0E, 0xA20BC7C6, 0x6D5451FD)
    assert D.philox4x32_10((0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344), (0xA4093822, 0x299F31D0)) == \
        (0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1)


def test_threshold_is_floor_of_p_times_2_32():
    assert D.threshold(0.0) == 0 and D.threshold(1.0) == 1 << 32 and D.threshold(0.5) == 1 << 31
    assert D.threshold(-0.1) == 0 and D.threshold(1.5) == 1 << 32
    assert D.threshold(0.05) == 214748364           # floor(0.05 * 4294967296) = floor(214748364.8)


def test_packets_per_group():
    assert D.packets_per_group([0, 1, 1200, 1201, 2400, 5000]).tolist() == [0, 1, 1, 2, 2, 5]


def test_no_loss_delivers_everything_and_full_loss_nothing():
    raw = np.array([3000, 1200, 1, 0, 0, 2400, 10, 10])
    order = np.arange(8)
    m, lv = D.sample_delivery(raw, order, 2, NO_LOSS, 5)
    assert np.all(m == 15) and np.all(lv == 3)
    m, lv = D.sample_delivery(raw, order, 2, dict(NO_LOSS, p_iid=1.0), 5)
    # empty groups (c0 l3, c1 l0) have no packet to lose: always usable (H1)
    assert np.all(m[:, 0] == 0b1000) and np.all(m[:, 1] == 0b0001)
    assert np.all(lv[:, 0] == -1) and np.all(lv[:, 1] == 0)
    # a channel that starts Bad, never leaves it and drops everything there
    m2, _ = D.sample_delivery(raw, order, 2, dict(NO_LOSS, p_gb=1.0, p_bg=0.0, e_bad=1.0), 5)
    assert np.array_equal(m2, m)
    # a Good channel that never turns Bad: e_bad is irrelevant
    m3, lv3 = D.sample_delivery(raw, order, 2, dict(NO_LOSS, p_gb=0.0, p_bg=0.5, e_bad=1.0), 5)
    assert np.all(m3 == 15) and np.all(lv3 == 3)


def test_packet_budget_cuts_the_send_order():
    """H2/H3: 6 packets in the order c1l0(2), c0l0(1), c0l1(2), c1l1(1); budget k = the first k arrive."""
    raw = np.array([1200, 2400, 0, 0, 2400, 1200, 0, 0])       # c0: 1, 2, 0, 0 packets; c1: 2, 1, 0, 0
    order = np.array([4, 0, 1, 5, 2, 3, 6, 7])
    want = {0: (-1, -1), 1: (-1, -1), 2: (-1, 0), 3: (0, 0), 4: (0, 0), 5: (3, 0), 6: (3, 3)}
    budgets = np.array(sorted(want))
    m, lv = D.sample_delivery(raw, order, 2, NO_LOSS, budgets.size, packet_budget=budgets)
    for j, k in enumerate(budgets):
        assert tuple(lv[j].tolist()) == want[k], (k, lv[j], m[j])
    # budget 2: c1l0 complete, c0l0 missing; the EMPTY groups l2, l3 are usable but closure stops at the gap
    assert m[2].tolist() == [0b1100, 0b1101]


def test_hand_walked_world_follows_the_printed_random_words():
    """Walk one world by hand from the raw Philox words: the oracle's trace must say the same."""
    raw = np.array([6000, 0, 0, 0])                               # one group of 5 packets
    model = dict(p_iid=0.3, p_gb=0.4, p_bg=0.5, e_good=0.1, e_bad=0.8, seed=0x1234567890ABCDEF)
    key = (0x90ABCDEF, 0x12345678)
    T = D.threshold
    bad, arrived, states = None, [], []
    for i in range(5):
        x0, x1, x2, x3 = D.philox4x32_10((i, 7, 0, 0), key)
        if i == 0:
            bad = x3 < T(0.4 / 0.9)
        else:
            bad = (not x1 < T(0.5)) if bad else (x1 < T(0.4))
        lost = x0 < T(0.3) or x2 < (T(0.8) if bad else T(0.1))
        arrived.append(not lost)
        states.append(bad)
    m, lv, tr = D.sample_delivery(raw, np.arange(4), 1, model, 1, world0=7, want_trace=True)
    assert tr[0][0] == arrived and tr[0][1] == states
    assert m[0, 0] == (0b1111 if all(arrived) else 0b1110)
    assert lv[0, 0] == (3 if all(arrived) else -1)


def test_worlds_do_not_depend_on_batching():
    raw = np.array([5000, 3000, 2000, 1000] * 3)
    model = dict(p_iid=0.05, p_gb=0.02, p_bg=0.3, e_good=0.0, e_bad=0.7, seed=99)
    order = np.arange(12)
    m, lv = D.sample_delivery(raw, order, 3, model, 8)
    m2, lv2 = D.sample_delivery(raw, order, 3, model, 3, world0=5)
    assert np.array_equal(m[5:], m2) and np.array_equal(lv[5:], lv2)


def test_packet_statistics_within_binomial_bounds():
    """IID loss rate, stationary Bad fraction and mean Bad-burst length of the GE chain (5 sigma)."""
    raw = np.array([1200 * 4000, 0, 0, 0])
    n = 4000
    _, _, tr = D.sample_delivery(raw, np.arange(4), 1, dict(NO_LOSS, p_iid=0.1, seed=5), 2, want_trace=True)
    lost = sum(1 for w in tr for a in w[0] if not a)
    assert abs(lost - 0.1 * 2 * n) < 5 * math.sqrt(2 * n * 0.1 * 0.9)
    p_gb, p_bg = 0.05, 0.25
    _, _, tr = D.sample_delivery(raw, np.arange(4), 1, dict(NO_LOSS, p_gb=p_gb, p_bg=p_bg, e_bad=1.0, seed=6), 4,
                                 want_trace=True)
    states = [s for w in tr for s in w[1]]
    arrived = [a for w in tr for a in w[0]]
    assert arrived == [not s for s in states]                      # e_bad = 1, e_good = 0: lost iff Bad
    pi_b = p_gb / (p_gb + p_bg)
    # correlated samples: the variance of the mean is inflated by (1 + r)/(1 - r), r = 1 - p_gb - p_bg
    r = 1 - p_gb - p_bg
    sd = math.sqrt(pi_b * (1 - pi_b) / len(states) * (1 + r) / (1 - r))
    assert abs(np.mean(states) - pi_b) < 5 * sd
    bursts, run = [], 0
    for w in tr:
        for s in w[1]:
            if s:
                run += 1
            elif run:
                bursts.append(run)
                run = 0
        run = 0
    mean_burst = np.mean(bursts)                                    # geometric with mean 1 / p_bg = 4
    assert abs(mean_burst - 1 / p_bg) < 5 * math.sqrt((1 - p_bg) / p_bg ** 2 / len(bursts))


def test_group_usability_rate_for_iid_loss():
    """A group of n packets survives IID loss p with probability (1-p)^n."""
    raw = np.array([1200 * 3, 1200 * 10, 0, 0])
    W, p = 600, 0.05
    m, _ = D.sample_delivery(raw, np.arange(4), 1, dict(NO_LOSS, p_iid=p, seed=11), W)
    for l, n in ((0, 3), (1, 10)):
        q = (1 - p) ** n
        got = ((m[:, 0] >> l) & 1).mean()
        assert abs(got - q) < 5 * math.sqrt(q * (1 - q) / W), (l, got, q)

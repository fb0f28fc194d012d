"""Pins of oracle/policy.py (frontier orders, frontier states, state bytes, atlas oracle) against a
hand-worked example, the paper's "flat table" statement, invariants and brute force.  CPU-only."""
import itertools
from pathlib import Path

import numpy as np
import pytest

from oracle import policy as P

GOLD = Path(__file__).resolve().parent / "golden" / "frontier_hand.txt"


def _gold():
    rows = {}
    states = []
    for line in GOLD.read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        key, *vals = line.split()
        if key == "state":
            states.append([int(v) for v in vals])
        else:
            rows[key] = [int(v) for v in vals]
    return rows, states


def test_hand_worked_wire_bytes():
    g, _ = _gold()
    assert P.group_wire_bytes(g["raw"]).tolist() == g["wire"]


@pytest.mark.parametrize("name,policy", [("utility", P.POLICY_UTILITY), ("nominal", P.POLICY_NOMINAL),
                                         ("bytes", P.POLICY_BYTE_GREEDY)])
def test_hand_worked_orders(name, policy):
    g, _ = _gold()
    order, cum = P.frontier_order(np.asarray(g["score"], np.float64), g["wire"], 2, policy)
    assert order.tolist() == g[f"order_{name}"]
    assert cum.tolist() == g[f"cum_{name}"]


@pytest.mark.parametrize("name", ["utility", "nominal"])
def test_hand_worked_frontier_states(name):
    g, _ = _gold()
    lv, used, n = P.frontier_states(g[f"order_{name}"], g["wire"], 2, g["budgets"])
    assert lv.reshape(-1).tolist() == g[f"levels_{name}"]
    assert used.tolist() == g[f"used_{name}"]
    # n_groups is the prefix length: levels count the same groups
    assert (lv.astype(int) + 1).sum(axis=1).tolist() == n.tolist()


def test_hand_worked_state_bytes():
    g, states = _gold()
    lv = np.asarray([s[:2] for s in states], np.int8)
    assert P.state_bytes(lv, g["wire"]).tolist() == [s[2] for s in states]


def test_flat_utility_table_recovers_nominal_order():
    """"A flat utility table recovers the conventional scheduler"."""
    rng = np.random.default_rng(3)
    C = 7
    wire = rng.integers(0, 5000, 4 * C)
    o_flat, _ = P.frontier_order(np.full(4 * C, 0.25), wire, C, P.POLICY_UTILITY)
    o_nom, _ = P.frontier_order(None, wire, C, P.POLICY_NOMINAL)
    assert o_flat.tolist() == o_nom.tolist()
    assert o_nom.tolist() == [4 * c + l for l in range(4) for c in range(C)]


@pytest.mark.parametrize("policy", [P.POLICY_UTILITY, P.POLICY_NOMINAL, P.POLICY_BYTE_GREEDY])
def test_orders_are_dependency_closed_permutations(policy):
    rng = np.random.default_rng(11 + policy)
    C = 9
    wire = rng.integers(0, 9000, 4 * C)
    score = rng.normal(size=4 * C).round(1)          # rounded: ties occur
    order, cum = P.frontier_order(score, wire, C, policy)
    assert sorted(order.tolist()) == list(range(4 * C))
    pos = np.empty(4 * C, int)
    pos[order] = np.arange(4 * C)
    for c in range(C):
        assert pos[4 * c] < pos[4 * c + 1] < pos[4 * c + 2] < pos[4 * c + 3]
    assert cum.tolist() == np.cumsum(wire[order]).tolist()
    # every prefix is a dependency-closed state whose state_bytes equals the cumulative wire bytes
    budgets = np.concatenate([[0], cum])
    lv, used, n = P.frontier_states(order, wire, C, budgets)
    assert np.array_equal(P.state_bytes(lv, wire), used)
    assert np.all(used <= budgets)
    # maximality of the prefix: the next group would not fit
    for j in range(budgets.size):
        if n[j] < 4 * C:
            assert used[j] + wire[order[n[j]]] > budgets[j]


def test_utility_order_is_greedy_by_brute_force():
    """Tiny case: among ALL dependency-consistent permutations, the greedy order is the one that is
    lexicographically smallest in the key sequence (-score, l, c) — checked by enumeration."""
    C = 2
    score = np.array([0.5, 3.0, -1.0, 2.0, 0.5, 0.25, 4.0, 1.0])
    wire = np.arange(8) + 1
    order, _ = P.frontier_order(score, wire, C, P.POLICY_UTILITY)
    best = None
    for perm in itertools.permutations(range(8)):
        pos = {g: i for i, g in enumerate(perm)}
        if any(pos[4 * c + l] > pos[4 * c + l + 1] for c in range(C) for l in range(3)):
            continue
        keys = [(-score[g], g % 4, g // 4) for g in perm]
        if best is None or keys < best[0]:
            best = (keys, perm)
    assert list(best[1]) == order.tolist()


def test_state_bytes_is_additive_over_clusters_and_levels():
    rng = np.random.default_rng(5)
    C = 6
    wire = rng.integers(1, 4000, 4 * C)
    lv = rng.integers(-1, 4, size=(50, C)).astype(np.int8)
    got = P.state_bytes(lv, wire)
    w = wire.reshape(C, 4)
    pref = np.concatenate([np.zeros((C, 1), np.int64), np.cumsum(w, axis=1)], axis=1)   # [C, 5]
    want = pref[np.arange(C)[None, :], lv.astype(int) + 1].sum(axis=1)
    assert np.array_equal(got, want)
    assert P.state_bytes(np.full((1, C), 3, np.int8), wire)[0] == wire.sum()
    assert P.state_bytes(np.full((1, C), -1, np.int8), wire)[0] == 0


def test_best_state_under_budget_against_numpy_and_ties():
    rng = np.random.default_rng(9)
    B = 300
    psnr = rng.normal(25, 3, B).round(1).astype(np.float32)    # rounded: ties occur
    cost = rng.integers(0, 10000, B)
    budgets = np.array([-1, 0, 500, 5000, 9999, 10**9])
    got = P.best_state_under_budget(psnr, cost, budgets)
    for j, beta in enumerate(budgets):
        ok = np.nonzero(cost <= beta)[0]
        if ok.size == 0:
            assert got[j] == -1
        else:
            top = psnr[ok].max()
            assert got[j] == ok[np.nonzero(psnr[ok] == top)[0][0]]          # first index attaining the max
    assert got[0] == -1
    # a larger budget never gives a worse oracle
    vals = [psnr[i] if i >= 0 else -np.inf for i in got]
    assert all(a <= b for a, b in zip(vals, vals[1:]))

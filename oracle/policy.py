"""CPU ORACLE for the scheduling-frontier / partial-state-atlas row.

TEST INFRASTRUCTURE ONLY (same rules as oracle/oracle.py): plain, slow Python loops that follow the
definitions below step by step.  It shares no code with the CUDA path and does not import the product
package.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import it.

What it follows (PAPER.md = /root/reference/PAPER.md; DESIGN.md §11 = the written spec of this row):

  wire bytes ........ PAPER.md:72 "the logical completion-group wire cost before rANS: raw stream bytes plus
                      one 48-byte chunk header and 4 bytes per dependency word for each 1200-byte payload
                      chunk".  Reading F1: chunks = ceil(raw / 1200) (0 for an empty group); dependency
                      words of group (c, l) = l (its prerequisites (c,0..l-1), chain of reading A8):
                          wire = raw + chunks * (48 + 4 l)
  frontier order .... PAPER.md:96 "converts the measured utilities into a dependency-closed scheduling
                      frontier"; "three scheduling policies: render-utility order, nominal layer
                      order, and dependency byte-greedy order".  Reading F2: a policy is a greedy total order
                      of the 4C completion groups; at every step the ELIGIBLE groups are (c, l) with
                      (c, 0..l-1) already taken, and the policy takes the eligible group with the smallest
                      key:   utility     (-score[g], l, c)      (highest risk-adjusted utility first)
                             nominal     (l, c)                 (all bases, then all level 1, ...)
                             byte-greedy (wire[g], l, c)        (cheapest eligible group first)
                      The (l, c) tie-break makes a flat utility table reproduce the nominal order
                      ("A flat utility table recovers the conventional scheduler").
  frontier states ... PAPER.md:96 "At four matched byte budgets".  Reading F3: the state of an order at
                      budget beta is its longest PREFIX whose cumulative wire bytes are <= beta; the delivered
                      depth of cluster c is (number of its groups in the prefix) - 1.
  state bytes ....... wire cost of a dependency-closed state = sum over clusters of wire[c, 0..depth_c].
  atlas oracle ...... PAPER.md:130 "records, at each of four matched byte budgets, the best sampled state as an
                      empirical oracle".  Reading F4: best = the sampled state of highest PSNR among those whose
                      state bytes are <= beta; ties go to the lowest state index; -1 if none fits.

Pins: tests/test_policy_pins.py (hand-worked example in tests/golden/frontier_hand.txt, flat table ==
nominal, permutation / dependency invariants, brute force over all prefixes / all states).
"""
from __future__ import annotations

import numpy as np

POLICY_UTILITY, POLICY_NOMINAL, POLICY_BYTE_GREEDY = 0, 1, 2


def group_wire_bytes(raw_bytes) -> np.ndarray:
    """Reading F1.  raw_bytes int64 [4C] (group g = 4c + l) -> wire int64 [4C]."""
    raw = np.asarray(raw_bytes, np.int64).reshape(-1)
    wire = np.zeros_like(raw)
    for g in range(raw.size):
        l = g % 4
        r = int(raw[g])
        chunks = (r + 1199) // 1200
        wire[g] = r + chunks * (48 + 4 * l)
    return wire


def frontier_order(score, wire, C: int, policy: int):
    """Reading F2.  Returns (order int32 [4C], cum_bytes int64 [4C])."""
    wire = np.asarray(wire, np.int64).reshape(-1)
    assert wire.size == 4 * C
    if policy == POLICY_UTILITY:
        score = np.asarray(score, np.float64).reshape(-1)
        assert score.size == 4 * C
    next_l = [0] * C
    order, cum, acc = [], [], 0
    for _ in range(4 * C):
        best_key, best_g = None, -1
        for c in range(C):
            l = next_l[c]
            if l > 3:
                continue
            g = 4 * c + l
            if policy == POLICY_UTILITY:
                key = (-float(score[g]), l, c)
            elif policy == POLICY_NOMINAL:
                key = (l, c)
            elif policy == POLICY_BYTE_GREEDY:
                key = (int(wire[g]), l, c)
            else:
                raise ValueError(policy)
            if best_key is None or key < best_key:
                best_key, best_g = key, g
        next_l[best_g // 4] += 1
        acc += int(wire[best_g])
        order.append(best_g)
        cum.append(acc)
    return np.asarray(order, np.int32), np.asarray(cum, np.int64)


def frontier_states(order, wire, C: int, budgets):
    """Reading F3.  Returns (levels int8 [nb, C], used int64 [nb], n_groups int32 [nb])."""
    order = np.asarray(order, np.int32).reshape(-1)
    wire = np.asarray(wire, np.int64).reshape(-1)
    budgets = np.asarray(budgets, np.int64).reshape(-1)
    levels = np.full((budgets.size, C), -1, np.int8)
    used = np.zeros(budgets.size, np.int64)
    n_groups = np.zeros(budgets.size, np.int32)
    for j, beta in enumerate(budgets.tolist()):
        acc = 0
        for g in order.tolist():
            if acc + int(wire[g]) > beta:
                break
            acc += int(wire[g])
            levels[j, g // 4] += 1
            n_groups[j] += 1
        used[j] = acc
    return levels, used, n_groups


def state_bytes(levels, wire) -> np.ndarray:
    """Wire cost of each dependency-closed state.  levels int8 [B, C] (depth -1..3) -> int64 [B]."""
    lv = np.asarray(levels, np.int8)
    wire = np.asarray(wire, np.int64).reshape(-1)
    B, C = lv.shape
    out = np.zeros(B, np.int64)
    for b in range(B):
        acc = 0
        for c in range(C):
            for l in range(int(lv[b, c]) + 1):
                acc += int(wire[4 * c + l])
        out[b] = acc
    return out


def best_state_under_budget(psnr_db, bytes_per_state, budgets) -> np.ndarray:
    """Reading F4.  Returns int32 [nb]: index of the best sampled state per budget, -1 if none fits."""
    p = np.asarray(psnr_db).reshape(-1)
    cost = np.asarray(bytes_per_state, np.int64).reshape(-1)
    budgets = np.asarray(budgets, np.int64).reshape(-1)
    best = np.full(budgets.size, -1, np.int32)
    for j, beta in enumerate(budgets.tolist()):
        for b in range(p.size):
            if int(cost[b]) <= beta and (best[j] < 0 or p[b] > p[best[j]]):
                best[j] = b
    return best

"""CPU ORACLE for the delivery-mask sampler: the step immediately BEFORE the hot
path — packet arrivals -> completion-group usability -> dependency closure -> levels[B x C].

TEST INFRASTRUCTURE ONLY (same rules as oracle/oracle.py).  Plain Python integers, one packet at a time.

What it follows (PAPER.md = /root/reference/PAPER.md; DESIGN.md §13 = the written spec of this row):

  PAPER.md:64  "A training world samples capacity, RTT, display deadline, IID erasure, and a Gilbert-Elliott
               burst process.  Packet dependencies are enforced after delivery, then converted to
               cluster-layer masks."
  PAPER.md:58  completion groups are cut into chunks of at most 1200 payload bytes, one packet each.
  PAPER.md:185 "A cluster-layer is usable only when all chunks in its dependency closure are usable."

The paper prints neither the loss-model parameters nor a generator, so (readings H1-H6):
  H1 packets   group g has n_g = ceil(raw_g / 1200) packets (0 for an empty group, which is always usable)
  H2 order     the packets of a world are sent group by group in a given group order (any of the policy orders
               of oracle/policy.py); packet i is the i-th packet of that sequence
  H3 budget    capacity / RTT / deadline are folded into one number per world: only packets i < budget[w]
               are sent before the display deadline; the others do not arrive
  H4 loss      a sent packet is lost if the IID process drops it (probability p_iid) OR the Gilbert-Elliott
               channel drops it: state s_0 = Bad with the stationary probability p_gb / (p_gb + p_bg) (0 if both
               are 0); s_i = next(s_{i-1}) with P(G->B) = p_gb, P(B->G) = p_bg; the packet is dropped with
               probability e_good in Good and e_bad in Bad
  H5 usable    a group is usable iff every one of its packets arrived (no repair); bit l of mask[w, c]; the
               level is the dependency closure of that mask (oracle.close_levels: trailing ones - 1)
  H6 random    counter-based: Philox4x32-10 (Salmon et al., SC'11) with key (seed_lo, seed_hi) and counter
               (packet i, world w, 0, 0) gives four 32-bit words x0..x3 per packet: x0 -> IID, x1 -> the GE
               transition, x2 -> the GE drop, x3 -> the initial state (packet 0 only).  An event of probability
               p happens iff x < T(p), T(p) = floor(p * 2^32) clamped to [0, 2^32] — an integer decision.

Pins: tests/test_delivery_pins.py (the three published Philox4x32-10 known-answer vectors, degenerate
channels, a hand-walked 6-packet world, packet-level loss / burst statistics within binomial bounds).
"""
from __future__ import annotations

import math

import numpy as np

M32 = 0xFFFFFFFF
PHILOX_M0, PHILOX_M1 = 0xD2511F53, 0xCD9E8D57
PHILOX_W0, PHILOX_W1 = 0x9E3779B9, 0xBB67AE85
CHUNK_BYTES = 1200


def philox4x32_10(counter, key):
    """Philox4x32 with 10 rounds.  counter: 4 uint32, key: 2 uint32 -> 4 uint32 (Python ints)."""
    c0, c1, c2, c3 = [int(c) & M32 for c in counter]
    k0, k1 = [int(k) & M32 for k in key]
    for _ in range(10):
        p0 = PHILOX_M0 * c0
        p1 = PHILOX_M1 * c2
        hi0, lo0 = p0 >> 32, p0 & M32
        hi1, lo1 = p1 >> 32, p1 & M32
        c0, c1, c2, c3 = (hi1 ^ c1 ^ k0) & M32, lo1, (hi0 ^ c3 ^ k1) & M32, lo0
        k0, k1 = (k0 + PHILOX_W0) & M32, (k1 + PHILOX_W1) & M32
    return c0, c1, c2, c3


def threshold(p: float) -> int:
    """T(p) = floor(p * 2^32) clamped to [0, 2^32] (reading H6)."""
    t = int(math.floor(float(p) * 4294967296.0))
    return min(max(t, 0), 1 << 32)


def packets_per_group(raw_bytes) -> np.ndarray:
    raw = np.asarray(raw_bytes, np.int64).reshape(-1)
    return np.array([(int(r) + CHUNK_BYTES - 1) // CHUNK_BYTES for r in raw], np.int64)


def sample_delivery(raw_bytes, order, C: int, model: dict, W: int, packet_budget=None, world0: int = 0,
                    want_trace: bool = False):
    """Readings H1-H6.  model: dict(p_iid, p_gb, p_bg, e_good, e_bad, seed).  Returns (mask uint8 [W, C],
    levels int8 [W, C]) and, if want_trace, per world the lists (arrived flag, GE state) per packet."""
    n_pk = packets_per_group(raw_bytes)
    order = [int(g) for g in np.asarray(order).reshape(-1)]
    assert sorted(order) == list(range(4 * C))
    seed = int(model["seed"])
    key = (seed & M32, (seed >> 32) & M32)
    t_iid, t_gb, t_bg = threshold(model["p_iid"]), threshold(model["p_gb"]), threshold(model["p_bg"])
    t_eg, t_eb = threshold(model["e_good"]), threshold(model["e_bad"])
    den = float(model["p_gb"]) + float(model["p_bg"])
    t_pi = threshold(float(model["p_gb"]) / den) if den > 0.0 else 0
    mask = np.zeros((W, C), np.uint8)
    levels = np.zeros((W, C), np.int8)
    traces = []
    for w in range(W):
        budget = None if packet_budget is None else int(packet_budget[w])
        usable = [True] * (4 * C)
        i, bad = 0, False
        tr_arr, tr_state = [], []
        for g in order:
            for _ in range(int(n_pk[g])):
                x0, x1, x2, x3 = philox4x32_10((i, world0 + w, 0, 0), key)
                if i == 0:
                    bad = x3 < t_pi
                elif bad:
                    bad = not (x1 < t_bg)
                else:
                    bad = x1 < t_gb
                lost = (x0 < t_iid) or (x2 < (t_eb if bad else t_eg))
                sent = budget is None or i < budget
                arrived = sent and not lost
                if not arrived:
                    usable[g] = False
                tr_arr.append(arrived)
                tr_state.append(bad)
                i += 1
        for c in range(C):
            m = 0
            for l in range(4):
                if usable[4 * c + l]:
                    m |= 1 << l
            mask[w, c] = m
            d = -1
            while d < 3 and (m >> (d + 1)) & 1:
                d += 1
            levels[w, c] = d
        traces.append((tr_arr, tr_state))
    return (mask, levels, traces) if want_trace else (mask, levels)

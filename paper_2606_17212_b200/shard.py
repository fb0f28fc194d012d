"""Host-side logic of the N > 1 path: states, frames and views are independent units, so
ranks take disjoint units, render them with no data-path collective, and meet only to (i) agree on the
step time (max over ranks) and (ii) pool per-pair distortion deltas before the Eq. (4) aggregation when
a group's contexts are spread over views on different ranks.  Backend-agnostic (`nccl` on GPUs, `gloo`
in the CPU tests); no method arithmetic here.
"""
from __future__ import annotations

from typing import List, Optional, Sequence

import numpy as np


def frame_for_step(step: int, rank: int, world: int, n_frames: int) -> int:
    """Round-robin: at step k rank r works on frame (k * world + r) mod n_frames, so that at any step the
    ranks hold `world` different frames and K steps cover K * world frames (weak scaling)."""
    if not (0 <= rank < world) or n_frames <= 0:
        raise ValueError("bad rank/world/n_frames")
    return (step * world + rank) % n_frames


def units_for_rank(n_units: int, rank: int, world: int) -> List[int]:
    """Strided partition of n_units independent units (views, frames, state chunks): every unit belongs
    to exactly one rank and the counts differ by at most one."""
    if not (0 <= rank < world):
        raise ValueError("bad rank/world")
    return list(range(rank, n_units, world))


def split_states(B: int, rank: int, world: int) -> slice:
    """Contiguous split of one batch of B states (for a single very large batch)."""
    per, rem = divmod(B, world)
    lo = rank * per + min(rank, rem)
    return slice(lo, lo + per + (1 if rank < rem else 0))


def max_over_ranks(value: float, device=None) -> float:
    """Every rank gets max_r value_r (the step time of the slowest rank)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def all_gather_ragged(local: np.ndarray, device=None) -> List[np.ndarray]:
    """All-gather of 1-D float64/int32 arrays whose lengths differ per rank (per-pair deltas and their
    group ids).  Returns the list indexed by rank, identical on every rank."""
    import torch
    import torch.distributed as dist
    local = np.ascontiguousarray(local)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [local]
    world = dist.get_world_size()
    dev = device or "cpu"
    n = torch.tensor([local.size], dtype=torch.int64, device=dev)
    sizes = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(world)]
    dist.all_gather(sizes, n)
    sizes = [int(s.item()) for s in sizes]
    m = max(max(sizes), 1)
    buf = torch.zeros(m, dtype=torch.from_numpy(local[:0]).dtype, device=dev)
    buf[:local.size] = torch.from_numpy(local).to(dev)
    out = [torch.zeros_like(buf) for _ in range(world)]
    dist.all_gather(out, buf)
    return [o[:k].cpu().numpy() for o, k in zip(out, sizes)]


def pool_pairs(delta_mse: np.ndarray, delta_db: np.ndarray, group_id: np.ndarray, device=None):
    """Pools the per-pair deltas of all ranks in RANK ORDER (deterministic), ready for the per-group
    mean / Q_0.1 / std / risk aggregation over contexts x views."""
    dm = np.concatenate(all_gather_ragged(np.asarray(delta_mse, np.float64), device))
    dd = np.concatenate(all_gather_ragged(np.asarray(delta_db, np.float64), device))
    gi = np.concatenate(all_gather_ragged(np.asarray(group_id, np.int32), device))
    return dm, dd, gi

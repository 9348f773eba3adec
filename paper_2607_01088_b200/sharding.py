"""Robot -> GPU sharding for N replicas.

Robots are independent units; there is no collective in the data path.  The only cross-rank
steps are the host-side assignment below and the barrier / max-over-ranks of the timing.
"""
from __future__ import annotations

from typing import List, Sequence

import numpy as np


def assign_robots(prefix_lens: Sequence[int], horizon: int, world: int) -> List[List[int]]:
    """Partition robots over `world` replicas balancing sum(L_i + H) (= KV bytes and attention
    work): longest-processing-time greedy, ties to the lowest rank; each shard sorted by id.
    Deterministic, so every rank computes the same partition without communication."""
    lens = np.asarray(prefix_lens, dtype=np.int64) + int(horizon)
    order = sorted(range(len(lens)), key=lambda i: (-int(lens[i]), i))
    load = [0] * world
    shards: List[List[int]] = [[] for _ in range(world)]
    for i in order:
        r = min(range(world), key=lambda q: (load[q], len(shards[q]), q))
        shards[r].append(i)
        load[r] += int(lens[i])
    return [sorted(s) for s in shards]


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """MAX all-reduce of a scalar (device timing of the slowest rank); identity without dist."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: Sequence[int], steps: int, max_ms: float) -> float:
    """Units (chunks) all ranks processed / the slowest rank's time."""
    return float(sum(units_per_rank)) * steps / (max_ms * 1e-3)

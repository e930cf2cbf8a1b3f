"""Multi-GPU sharding of a sweep: simulations are independent (PAPER.md P:86,
P:119), so the sim axis is split across ranks with no data-path collective; every rank builds
its own tvbx sweep from `sim_ids` and writes its own slice of the results.  Host-side integer
bookkeeping only -- no arithmetic of the method lives here.
"""
from __future__ import annotations

import numpy as np


def partition_sims(speeds, ring_lens, world: int):
    """Split simulations 0..S-1 into `world` lists.

    Simulations are first grouped by conduction speed (stable sort by v: one delay table per
    distinct v, so each rank should see few of them), then cut into contiguous blocks of nearly
    equal cost, cost = ring length H (a v = 1 m/s simulation holds 125x the history of a v = 128
    one and also runs with shorter barrier intervals).  Deterministic; every sim lands on exactly
    one rank; ranks are never empty when S >= world.
    """
    speeds = np.asarray(speeds, dtype=np.float64)
    cost = np.asarray(ring_lens, dtype=np.float64)
    S = speeds.size
    assert cost.shape == (S,) and world >= 1
    order = np.argsort(speeds, kind="stable")
    csum = np.cumsum(cost[order])
    total = csum[-1] if S else 0.0
    cuts = [0]
    for r in range(1, world):
        target = total * r / world
        c = int(np.searchsorted(csum, target, side="left"))
        c = min(max(c, cuts[-1] + 1), S - (world - r))      # keep every rank non-empty
        cuts.append(max(c, 0))
    cuts.append(S)
    return [np.sort(order[cuts[r]:cuts[r + 1]]).astype(np.int64) for r in range(world)]


def shard_for_rank(speeds, ring_lens, rank: int, world: int):
    return partition_sims(speeds, ring_lens, world)[rank]

"""Rate statistics of one simulation's kept 1-ms samples, plain FP64 definitions  --  TEST INFRASTRUCTURE, NOT
PRODUCT CODE (only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import anything under oracle/).

PAPER.md P:288: "only for a speed of 1.0 m/s the maximum and variance in firing rates for both excitatory and
inhibitory populations is maximal"; regions "visit the paroxysmal fixed point and display high firing
rate activity exceeding 100 Hz", and the paper counts the parameter combinations in which a region does so.

Reading A24: the statistics are taken over the same series the FC uses -- the temporal
averages over ds steps that survive the discard (A17), excitatory population; variance = population variance
(1/n) sum (x - mean)^2 (the sigma^2 of Eq. 6); "exceeding 100 Hz" = sample > 0.1 kHz, strictly.

samples: [n][N] array-like (oracle.OracleSweep.samples(s)[0]).  Written out entry by entry.
"""
from __future__ import annotations

import math


def rate_stats(samples, threshold_khz=0.1):
    """-> (var [N], max [N], n_above [N]) as lists."""
    n = len(samples)
    n_reg = len(samples[0]) if n else 0
    var, mx, above = [], [], []
    for k in range(n_reg):
        col = [float(samples[q][k]) for q in range(n)]
        mean = math.fsum(col) / n
        var.append(math.fsum((x - mean) ** 2 for x in col) / n)
        mx.append(max(col))
        above.append(sum(1 for x in col if x > threshold_khz))
    return var, mx, above

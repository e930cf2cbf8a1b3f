"""Up / down-state durations of one simulation's kept 1-ms samples  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE (only
tests/, __graft_entry__.smoke() and bench.py's CPU legs may import anything under oracle/).

PAPER.md Tab. 2: `mean_UD_duration` -- "Mean duration of UP and DOWN states"; P:139 describes the notion ("distinct
patterns of neuronal activity ... closely linked to the sleep-wake cycle"), "characterization of Up and Down states
typical for synchronous behavior".  The paper gives no algorithm (it cites its analysis toolbox).

Reading A25: per region, on the series the FC uses (the temporal averages over ds steps that survive
the discard, excitatory population, A17 / A18):
  * a sample is UP iff x > threshold (strictly), else DOWN;
  * an episode is a maximal run of equal states; episodes cut by either end of the record are NOT counted (their duration
    is unknown);
  * duration of an episode = its number of samples x sample_ms;
  * outputs per region: number of UP episodes, their mean duration [ms], number of DOWN episodes, their mean duration [ms]
    (mean = 0 where there is no episode).

samples: [n][N] array-like (oracle.OracleSweep.samples(s)[0]).  Written out sample by sample.
"""
from __future__ import annotations


def state_durations(samples, threshold_khz, sample_ms=1.0):
    """-> (n_up [N], mean_up_ms [N], n_down [N], mean_down_ms [N]) as lists."""
    n = len(samples)
    n_reg = len(samples[0]) if n else 0
    n_up, mean_up, n_down, mean_down = [], [], [], []
    for k in range(n_reg):
        count = [0, 0]          # [down, up]
        total = [0, 0]
        prev, run, at_start = None, 0, True
        for q in range(n):
            s = 1 if float(samples[q][k]) > threshold_khz else 0
            if prev is None:
                prev, run = s, 1
            elif s == prev:
                run += 1
            else:
                if not at_start:            # the first episode is cut by the start of the record
                    count[prev] += 1
                    total[prev] += run
                prev, run, at_start = s, 1, False
        # the episode still open at the end of the record is cut by it: not counted
        n_up.append(count[1]); n_down.append(count[0])
        mean_up.append(total[1] * sample_ms / count[1] if count[1] else 0.0)
        mean_down.append(total[0] * sample_ms / count[0] if count[0] else 0.0)
    return n_up, mean_up, n_down, mean_down

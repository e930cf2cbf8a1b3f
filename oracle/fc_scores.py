"""FC scores of one simulation, plain FP64 definitions  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE
(only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import anything under oracle/).

PAPER.md P:113: "The FCSC, the correlation with the structure connectivity (SC), represented by the properties of
the connectome and the obtained covariance matrix, is determined with the Pearson correlation.  The driver can
also perform a comparison to an externally obtained reference FC matrix by correlating it to the computed FC of
the simulation, also by making use of the Pearson coefficient."  P:159: "The fitness is defined as the pearson
correlation between the external and the computed FC computed with eq. (6)"; Eq. (6), P:161:
rho_xy = Cov(x, y) / (sigma_x sigma_y).  Tab. 2: mean_FC = "Average FC from Pearson corr. of time-series
firing rate".

Reading A23: the paper does not say which matrix entries enter the correlation.  Both
matrices are symmetric and the diagonal is trivial (FC_kk = 1, W_kk = 0), so the samples are the N(N-1)/2 pairs
k < l, each once.  Zero variance on either side -> 0 (as A18).

Written as the definition, entry by entry, in the order of Eq. (6): means, covariance, standard deviations.
"""
from __future__ import annotations

import math


def pearson_upper(x, y):
    """Eq. (6) over the pairs k < l of two N x N matrices (nested sequences or arrays)."""
    n_reg = len(x)
    xs, ys = [], []
    for k in range(n_reg):
        for l in range(k + 1, n_reg):
            xs.append(float(x[k][l]))
            ys.append(float(y[k][l]))
    n = len(xs)
    if n < 2:
        return 0.0
    mx = math.fsum(xs) / n
    my = math.fsum(ys) / n
    cov = math.fsum((a - mx) * (b - my) for a, b in zip(xs, ys)) / n
    sx = math.sqrt(math.fsum((a - mx) ** 2 for a in xs) / n)
    sy = math.sqrt(math.fsum((b - my) ** 2 for b in ys) / n)
    if not (sx > 0.0 and sy > 0.0):
        return 0.0
    return cov / (sx * sy)


def mean_upper(x):
    n_reg = len(x)
    vals = [float(x[k][l]) for k in range(n_reg) for l in range(k + 1, n_reg)]
    return math.fsum(vals) / len(vals) if vals else 0.0


def fc_scores(fc, sc, ref=None):
    """fc: [S][N][N] Pearson matrices (oracle.OracleSweep.fc_readout()[0]); sc: [N][N] connectome weights;
    ref: optional [N][N] reference FC.  -> dict of lists: fcsc, mean_fc (and fitness)."""
    out = {"fcsc": [pearson_upper(f, sc) for f in fc], "mean_fc": [mean_upper(f) for f in fc]}
    if ref is not None:
        out["fitness"] = [pearson_upper(f, ref) for f in fc]
    return out


def top_k(scores, k):
    """The k fittest simulations (the grid search "output[s] the best ten fittest simulations"): indices of
    the k largest scores, best first; equal scores in ascending index (reading A23b: the paper does not say how ties are
    broken).  Selection by repeated maximum, written out.  -> (indices, values)"""
    s = [float(x) for x in scores]
    taken = [False] * len(s)
    idx, val = [], []
    for _ in range(min(k, len(s))):
        best = -1
        for i in range(len(s)):
            if not taken[i] and (best < 0 or s[i] > s[best]):
                best = i
        taken[best] = True
        idx.append(best); val.append(s[best])
    return idx, val

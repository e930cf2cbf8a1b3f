"""Seeded synthetic inputs shared by the oracle (oracle/) and the CUDA path (tests, bench.py).

This module holds NO arithmetic of the method: it only draws connectomes, lists parameter axes and
names the default model parameters (which are *inputs* to both sides).  The synthetic connectomes
stand in for the paper's `connectivity_zerlaut_68.zip`, which is not available; shapes,
sizes and distributions are BASELINE.json's, the draw order is the recipe frozen in DESIGN.md §4
(SURVEY.md §8(d)).
"""
from __future__ import annotations

import numpy as np

# ---------------------------------------------------------------------------------------------
# Default model parameters (DESIGN.md §3 table; units ms, kHz, mV, pA, nS, pF).  Inputs, not code.
# ---------------------------------------------------------------------------------------------
POLY_RS = (-48.9, 5.1, -25.0, 1.4, -0.41, 10.5, -36.0, 7.4, 1.2, 40.7)   # Table 1
POLY_FS = (-51.4, 0.4, -8.3, 0.2, -0.5, 1.4, -14.6, 4.5, 2.8, 15.3)      # Table 1

DEFAULTS = dict(
    G=0.0, b_e=0.0, a_e=0.0, tau_w_e=500.0, v=4.0, wNoise=1e-6, E_L_e=-64.0, E_L_i=-64.0, T=20.0,
    c_Fee=0.3e-3, c_Fei=0.0, c_Fie=0.3e-3, c_Fii=0.0,
    b_i=0.0, a_i=0.0, tau_w_i=1.0,
    g_L=10.0, C_m=200.0, Q_e=1.5, tau_e=5.0, E_e=0.0, Q_i=5.0, tau_i=5.0, E_i=-80.0,
    N_tot=10000.0, p_conn=0.05, g_inh=0.2,
    tau_OU=5.0, mu_OU=0.0, sigma_OU=1.0,
    muV0=-60.0, dmuV0=10.0, sV0=4.0, dsV0=6.0, tauVN0=0.5, dtauVN0=1.0,
    eps_nu=1e-6, muV_local=0.0, kappa=1e-3,
)
# order of the scalar parameters in the flat parameter vector (followed by POLY_RS, POLY_FS)
PARAM_NAMES = tuple(DEFAULTS.keys())
N_PARAMS = len(PARAM_NAMES) + 20
INIT_STATE = (0.001, 0.001, 0.0, 0.0, 0.0, 0.0, 0.0)   # E, I, C_ee, C_ei, C_ii, W_e, W_i (cfg 1)


def param_vector(**overrides) -> np.ndarray:
    """Flat float64 parameter vector (PARAM_NAMES order, then the two Table-1 rows)."""
    d = dict(DEFAULTS)
    poly_e = overrides.pop("poly_e", POLY_RS)
    poly_i = overrides.pop("poly_i", POLY_FS)
    for k, val in overrides.items():
        if k not in d:
            raise KeyError(k)
        d[k] = float(val)
    return np.array([d[k] for k in PARAM_NAMES] + list(poly_e) + list(poly_i), dtype=np.float64)


# ---------------------------------------------------------------------------------------------
# Connectomes
# ---------------------------------------------------------------------------------------------
def _sym_from_upper(n: int, vals: np.ndarray) -> np.ndarray:
    m = np.zeros((n, n), dtype=np.float64)
    iu = np.triu_indices(n, k=1)          # row-major over pairs i < j
    m[iu] = vals
    return m + m.T


def connectome(n: int = 68, seed: int = 0, keep: float = 0.30, lengths: str = "uniform"):
    """Symmetric log-normal(0,1) weights with a fraction `keep` of the pairs kept, zero diagonal,
    divided by the maximum; symmetric tract lengths in mm.  Draw order (fixed): weights, mask, lengths.
    lengths = "uniform": U[10, 200] mm (cfg 1-4); "ellipsoid": 1.2 x Euclidean distance between points
    uniform in the ellipsoid with full extents 140 x 170 x 120 mm (cfg 5)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n_pairs = n * (n - 1) // 2
    w = rng.lognormal(0.0, 1.0, n_pairs)
    mask = rng.random(n_pairs) < keep
    w = np.where(mask, w, 0.0)
    if lengths == "uniform":
        ln = rng.uniform(10.0, 200.0, n_pairs)
        L = _sym_from_upper(n, ln)
    elif lengths == "ellipsoid":
        pts = []
        while len(pts) < n:
            p = rng.uniform(-1.0, 1.0, 3)
            if float(p @ p) <= 1.0:
                pts.append(p)
        pts = np.array(pts) * np.array([70.0, 85.0, 60.0])
        diff = pts[:, None, :] - pts[None, :, :]
        L = 1.2 * np.sqrt((diff * diff).sum(-1))
        np.fill_diagonal(L, 0.0)
        L = 0.5 * (L + L.T)
    else:
        raise ValueError(lengths)
    W = _sym_from_upper(n, w)
    W /= W.max()
    return np.ascontiguousarray(W), np.ascontiguousarray(L)


# ---------------------------------------------------------------------------------------------
# The five BASELINE.json configurations
# ---------------------------------------------------------------------------------------------
def _lin(name, lo, hi, n):
    return dict(name=name, lo=float(lo), hi=float(hi), n=int(n), values=None)


def _vals(name, values):
    v = [float(x) for x in values]
    return dict(name=name, lo=v[0], hi=v[-1], n=len(v), values=v)


def config(i: int) -> dict:
    """BASELINE.json configs[i-1] as data.  Axis order = listing order, first axis slowest (A19)."""
    if i == 1:
        return dict(name="cfg1", n=68, conn_seed=0, keep=0.30, lengths="uniform",
                    axes=[_vals("G", [0.0, 0.3]), _vals("b_e", [0.0, 30.0, 60.0, 120.0])],
                    fixed=dict(v=4.0), dt=0.1, steps=5000, ds=10, discard_steps=0, seed=1)
    if i == 2:
        return dict(name="cfg2", n=68, conn_seed=0, keep=0.30, lengths="uniform",
                    axes=[_lin("G", 0.0, 0.5, 32), _lin("b_e", 0.0, 120.0, 32)],
                    fixed=dict(v=4.0), dt=0.1, steps=50000, ds=10, discard_steps=10000, seed=2)
    if i == 3:
        return dict(name="cfg3", n=68, conn_seed=0, keep=0.30, lengths="uniform",
                    axes=[_lin("b_e", 0.0, 120.0, 16), _lin("a_e", -10.0, 10.0, 16),
                          _lin("G", 0.0, 0.5, 16), _vals("v", [1, 2, 4, 8, 16, 32, 64, 128])],
                    fixed=dict(), dt=0.1, steps=20000, ds=10, discard_steps=10000, seed=3)
    if i == 4:
        return dict(name="cfg4", n=68, conn_seed=0, keep=0.30, lengths="uniform",
                    axes=[_lin("G", 0.0, 0.5, 16), _lin("b_e", 0.0, 120.0, 16)],
                    fixed=dict(v=4.0, tau_w_e=500.0), dt=0.1, steps=3000000, ds=10,
                    discard_steps=10000, seed=4)
    if i == 5:
        return dict(name="cfg5", n=360, conn_seed=5, keep=0.50, lengths="ellipsoid",
                    axes=[_lin("G", 0.0, 0.5, 64), _lin("b_e", 0.0, 120.0, 64)],
                    fixed=dict(v=3.0), dt=0.1, steps=20000, ds=10, discard_steps=10000, seed=5)
    raise ValueError(i)


def config_connectome(cfg: dict):
    return connectome(cfg["n"], cfg["conn_seed"], cfg["keep"], cfg["lengths"])


def axis_values(ax: dict) -> np.ndarray:
    """NumPy restatement of the grid spacing (A19): explicit list or closed linspace."""
    if ax["values"] is not None:
        return np.array(ax["values"], dtype=np.float64)
    return np.linspace(ax["lo"], ax["hi"], ax["n"])


def grid_params(cfg: dict, sims=None) -> np.ndarray:
    """[S][N_PARAMS] float64 parameter vectors of the sweep in C-order (first axis slowest), built
    with numpy.meshgrid(indexing='ij').  `sims`: optional list of external sim indices to keep."""
    axes = [axis_values(a) for a in cfg["axes"]]
    mesh = np.meshgrid(*axes, indexing="ij")
    cols = [m.ravel() for m in mesh]
    S = cols[0].size
    base = param_vector(**cfg["fixed"])
    out = np.tile(base, (S, 1))
    for a, col in zip(cfg["axes"], cols):
        out[:, PARAM_NAMES.index(a["name"])] = col
    if sims is not None:
        out = out[np.asarray(sims, dtype=np.int64)]
    return np.ascontiguousarray(out)

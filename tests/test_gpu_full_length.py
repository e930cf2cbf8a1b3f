"""GPU parity at the FULL step counts of BASELINE.json configs 2-5, in the launch configuration bench.py times, against
the oracle on the stratified subsets BASELINE.md names (simulations are independent, so the oracle recomputes the
sampled ones one by one).  Tolerances are the north star's: per-region mean rates 1 % relative, FC entries 0.02 absolute.

cfg 4 is the drift check the north star asks for: 300 s simulated = 3,000,000 Euler steps, 299,000 kept 1-ms samples
merged chunk after chunk into the streaming (n, mean, M) accumulators (Welford/Chan), compared with the oracle's
two-pass FC on the first and the last simulation of the grid.  The oracle side takes ~3 min on two host cores."""
import numpy as np
import pytest

import workloads as wl
import paper_2311_13337_b200 as tvbx
from oracle import oracle as orc

pytestmark = pytest.mark.gpu

TOL_MEAN_REL = 1e-2     # BASELINE.json north_star
TOL_FC_ABS = 0.02


def _full_length(cfg_id, sims):
    cfg = wl.config(cfg_id)
    W, L = wl.config_connectome(cfg)
    conn, sw = tvbx.sweep_from_config(cfg, W, L)
    sw.run(cfg["steps"], cfg["dt"], noise_on=True, ds=cfg["ds"], discard_steps=cfg["discard_steps"])
    fc, me, mi = sw.fc_readout()
    assert sw.steps_done() == cfg["steps"]
    assert sw.samples_kept() == (cfg["steps"] - cfg["discard_steps"]) // cfg["ds"]
    o = orc.OracleSweep(W, L, wl.grid_params(cfg, sims=sims), seed=cfg["seed"], ext_ids=sims)
    o.run(cfg["steps"], cfg["dt"], noise_on=True, ds=cfg["ds"], discard_steps=cfg["discard_steps"])
    rfc, rme, rmi = o.fc_readout()
    assert np.isfinite(fc).all() and np.isfinite(me).all() and np.isfinite(mi).all()
    err = dict(mean_e=float(np.abs(me[sims] / rme - 1).max()), mean_i=float(np.abs(mi[sims] / rmi - 1).max()),
               fc=float(np.abs(fc[sims] - rfc).max()))
    print(f"cfg {cfg_id} full length ({cfg['steps']} steps, {len(sims)} oracle sims): {err}")
    assert err["mean_e"] < TOL_MEAN_REL and err["mean_i"] < TOL_MEAN_REL, err
    assert err["fc"] < TOL_FC_ABS, err
    # properties that hold for every simulation at any size
    assert np.all(np.abs(fc) <= 1.0 + 1e-6)
    np.testing.assert_array_equal(fc, np.swapaxes(fc, 1, 2))
    assert np.all(np.diagonal(fc, axis1=1, axis2=2) == 1.0)
    assert (me > 0).all() and (me < 0.2).all() and (mi > 0).all() and (mi < 0.2).all()
    return sw, o


def test_cfg2_full_length_4x4_sublattice():
    """50,000 steps, 1,024 sims; the oracle recomputes the 4 x 4 sub-lattice of the (G, b_e) grid."""
    idx = [0, 10, 21, 31]
    _full_length(2, [a * 32 + b for a in idx for b in idx])


def test_cfg3_full_length_all_speeds_two_corners():
    """20,000 steps, 32,768 sims; 16 oracle sims: all 8 speeds at two corners of the (b_e, a_e, G) grid."""
    lo = [v for v in range(8)]                                  # b_e = 0, a_e = -10, G = 0
    hi = [32768 - 8 + v for v in range(8)]                      # b_e = 120, a_e = 10, G = 0.5
    _full_length(3, lo + hi)


def test_cfg5_full_length_four_sims():
    """20,000 steps, 4,096 sims x 360 regions; 4 oracle sims."""
    _full_length(5, [0, 63, 64 * 31 + 17, 4095])


def test_cfg4_full_length_drift_300s():
    """3,000,000 steps (300 s simulated), 256 sims; sims 0 and 255 against the oracle's two-pass FC."""
    sw, o = _full_length(4, [0, 255])
    assert sw.samples_kept() == 299000 and sw.launch_info()["chunk_samples"] < 299000      # many Chan merges

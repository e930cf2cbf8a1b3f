"""The product kernel's own transfer function, tf_closed2 (csrc/tvbx_tf2.cuh: packed FP32 pairs, hand-derived closed
form), evaluated ON THE DEVICE through tvbx_diag_tf_closed2 and compared with the oracle's orc_tf element by element:
value, both first and all three second derivatives, both populations, on the grid of the oracle's own mpmath pin
(tests/test_oracle_tf.py: f_e, f_i in 1e-6 ... 0.2 kHz, W in {0, 50, 200} pA), plus the states the five BASELINE.json
configs actually visit.

Why this test exists: in Eq. (1) the second derivatives enter as (1/2) C d2F kappa^2, 1e-7 of nu at the default
kappa = 1e-3 -- no FP32 trajectory tolerance can see an error there.  Here each component is checked on its own.

Tolerances (FP32 path, SFU rcp/sqrt/ex2 approximations of <= 2 ulp, erfc fit 4.7e-7; on the tail of erfc a relative
error d of its argument z becomes 2 z^2 d in F -- x 50 at z = 5 --, so the value cannot be held to FP32 epsilon):
  mu_V        : 2e-5 relative
  value       : 1e-4 relative     (measured on the B200: 4.9e-5)
  first       : 2e-4 relative     (measured: 1.1e-4)
  second      : 1e-3 relative     (measured: 1.2e-4)
"relative" = |got - ref| / max(|ref|, floor_q) with floor_q = 1e-3 x the largest |ref| of that component over the same
(population, W) slice: derivatives cross zero inside the grid, and an FP32 result cannot be relatively accurate at a zero
crossing of a sum of O(max) terms."""
import itertools

import numpy as np
import pytest

import workloads as wl
import paper_2311_13337_b200 as tvbx
from oracle import oracle as orc

pytestmark = pytest.mark.gpu

GRID_F = [1e-6, 2e-4, 1e-3, 5e-3, 2e-2, 8e-2, 0.2]       # tests/test_oracle_tf.py
GRID_W = [0.0, 50.0, 200.0]
TOL = np.array([1e-4, 2e-4, 2e-4, 1e-3, 1e-3, 1e-3])
NAMES = ("F", "F_e", "F_i", "F_ee", "F_ei", "F_ii")


def _oracle_jets(p, fe, fi, we, wi):
    ref = np.zeros((len(fe), 2, 7))
    for n in range(len(fe)):
        for pop, w in ((0, we[n]), (1, wi[n])):
            out, mu = orc.tf(p, pop, fe[n], fi[n], w)
            ref[n, pop, :6] = out
            ref[n, pop, 6] = mu
    return ref


def _compare(got, ref, groups):
    """groups: index arrays; the floor of a component is taken over each group."""
    worst = np.zeros((2, 7))
    for idx in groups:
        for pop in range(2):
            for q in range(7):
                r = ref[idx, pop, q]
                floor = 1e-3 * np.abs(r).max()
                e = np.abs(got[idx, pop, q] - r) / np.maximum(np.abs(r), floor)
                worst[pop, q] = max(worst[pop, q], e.max())
    return worst


def test_tf_closed2_all_six_components_on_the_pin_grid():
    p = wl.param_vector(eps_nu=0.0)                   # the inputs given ARE the clamped rates
    pts = list(itertools.product(GRID_F, GRID_F, GRID_W))
    fe = np.array([a for a, _, _ in pts]); fi = np.array([b for _, b, _ in pts]); w = np.array([c for _, _, c in pts])
    got = tvbx.diag_tf_closed2(fe, fi, w, w)
    ref = _oracle_jets(p, fe, fi, w, w)
    groups = [np.where(w == x)[0] for x in GRID_W]
    worst = _compare(got, ref, groups)
    for pop in range(2):
        assert np.all(worst[pop, :6] < TOL), (pop, dict(zip(NAMES, worst[pop, :6])))
        assert worst[pop, 6] < 2e-5, worst[pop, 6]
    # the components are not trivially small: every one of them reaches a sizeable magnitude somewhere on the grid
    assert np.all(np.abs(ref[:, :, 3:6]).max(axis=0) > 1.0)


def test_tf_closed2_distinct_populations_and_parameters():
    """Different adaptation currents for the two populations (the packed halves must not leak into each other),
    non-default E_L, and random points inside the range the configs visit (rates 0.1 ... 60 Hz)."""
    rng = np.random.default_rng(7)
    n = 400
    fe = 10.0 ** rng.uniform(-4, np.log10(0.06), n); fi = 10.0 ** rng.uniform(-4, np.log10(0.06), n)
    we = rng.uniform(0.0, 120.0, n); wi = rng.uniform(0.0, 20.0, n)
    par = dict(E_L_e=-63.0, E_L_i=-67.0, eps_nu=0.0)
    got = tvbx.diag_tf_closed2(fe, fi, we, wi, params=par)
    ref = _oracle_jets(wl.param_vector(**par), fe, fi, we, wi)
    worst = _compare(got, ref, [np.arange(n)])
    for pop in range(2):
        assert np.all(worst[pop, :6] < TOL), (pop, dict(zip(NAMES, worst[pop, :6])))


def test_tf_closed2_refuses_unequal_time_constants():
    with pytest.raises(tvbx.TvbxError):
        tvbx.diag_tf_closed2([1e-3], [1e-3], [0.0], [0.0], params=dict(tau_i=7.0))

"""Pins P1/P2 of the oracle's transfer function: direct numerical evaluation in
40-digit arithmetic with numerical differentiation, closed-form limits and bounds."""
import itertools

import mpmath as mp
import numpy as np
import pytest

import workloads as wl
from oracle import oracle as orc
from tests import _mp_model as M


def rel(a, b):
    return abs(a - b) / max(abs(b), 1e-300)


GRID_F = [1e-6, 2e-4, 1e-3, 5e-3, 2e-2, 8e-2, 0.2]


@pytest.mark.parametrize("pop", [0, 1])
@pytest.mark.parametrize("W", [0.0, 50.0, 200.0])
def test_tf_value_and_derivatives_vs_mpmath(pop, W):
    """P1: value and all five derivatives against mpmath + mpmath.diff on a grid spanning both erfc
    tails (A1, A8)."""
    p = wl.param_vector(eps_nu=0.0)     # inputs given are the clamped ones
    worst = np.zeros(6)      # whole grid
    inner = np.zeros(6)      # fe, fi >= 2e-4 kHz (away from the sqrt(f) corner, where FP64 cancels)
    for fe, fi in itertools.product(GRID_F, GRID_F):
        out, muV = orc.tf(p, pop, fe, fi, W)
        ref = M.tf_derivs(p, pop, fe, fi, W)
        refmu = M.tf_parts(p, pop, mp.mpf(fe), mp.mpf(fi), mp.mpf(W))[1]
        assert rel(muV, float(refmu)) < 1e-13
        for q in range(6):
            r = float(ref[q])
            # absolute floor: derivatives can pass through zero
            scale = max(abs(r), 1e-12 * (1.0, 1e1, 1e1, 1e3, 1e3, 1e3)[q])
            worst[q] = max(worst[q], abs(out[q] - r) / scale)
            if min(fe, fi) >= 2e-4:
                inner[q] = max(inner[q], abs(out[q] - r) / scale)
    assert worst[0] < 1e-10, worst
    assert worst[1] < 1e-9 and worst[2] < 1e-9, worst
    assert inner[3:].max() < 1e-8, inner
    assert worst[3:].max() < 1e-5, worst


def test_tf_erfc_argument_spans_both_tails():
    p = wl.param_vector(eps_nu=0.0)
    args = []
    for pop in (0, 1):
        for fe, fi in itertools.product(GRID_F, GRID_F):
            F, muV, sV, TV, Vthr = M.tf_parts(p, pop, mp.mpf(fe), mp.mpf(fi), mp.mpf(0))
            args.append(float((Vthr - muV) / (mp.sqrt(2) * sV)))
    assert min(args) < -1.0 and max(args) > 4.0


def test_tf_closed_form_limits():
    """P2: tau_e == tau_i => tau_V = tau_e + tau_m identically; 0 <= F <= 1/tau_V;
    f_i -> 0, W = 0 => mu_V = (mu_Ge E_e + g_L E_L)/(g_L + mu_Ge)."""
    p = wl.param_vector(eps_nu=0.0)
    nm = wl.PARAM_NAMES.index
    assert p[nm("tau_e")] == p[nm("tau_i")]
    gL, Cm, Qe, Te, Ee = (p[nm(k)] for k in ("g_L", "C_m", "Q_e", "tau_e", "E_e"))
    Qi, Ti = p[nm("Q_i")], p[nm("tau_i")]
    Ke, Ki = 400.0, 100.0
    for pop in (0, 1):
        for fe, fi in itertools.product(GRID_F, GRID_F):
            out, muV = orc.tf(p, pop, fe, fi, 0.0)
            muG = gL + Qe * Te * Ke * fe + Qi * Ti * Ki * fi
            tauV = Te + Cm / muG
            assert 0.0 <= out[0] <= 1.0 / tauV * (1 + 1e-12)
        EL = p[nm("E_L_e")] if pop == 0 else p[nm("E_L_i")]
        for fe in GRID_F:
            _, muV = orc.tf(p, pop, fe, 1e-300, 0.0)
            muGe = Qe * Te * Ke * fe
            assert rel(muV, (muGe * Ee + gL * EL) / (gL + muGe)) < 1e-13


def test_tf_K_counts_and_population_constants():
    """K_e = p N (1-g) = 400, K_i = p N g = 100 (DESIGN.md table); the inhibitory population uses
    E_L,i and the FS row of Table 1: changing them must change only pop 1."""
    p = wl.param_vector()
    q = wl.param_vector(E_L_i=-65.0)
    a0, _ = orc.tf(p, 0, 5e-3, 1e-2, 0.0); b0, _ = orc.tf(q, 0, 5e-3, 1e-2, 0.0)
    a1, _ = orc.tf(p, 1, 5e-3, 1e-2, 0.0); b1, _ = orc.tf(q, 1, 5e-3, 1e-2, 0.0)
    assert np.array_equal(a0, b0) and not np.allclose(a1, b1)
    pe = list(wl.POLY_RS); pe[9] = -pe[9]
    r = wl.param_vector(poly_e=pe)
    c0, _ = orc.tf(r, 0, 5e-3, 1e-2, 0.0); c1, _ = orc.tf(r, 1, 5e-3, 1e-2, 0.0)
    assert not np.allclose(a0, c0) and np.array_equal(a1, c1)
    # K_e, K_i: doubling p_conn doubles both; check through mu_V closed form at W=0
    s = wl.param_vector(p_conn=0.1, eps_nu=0.0)
    _, muV = orc.tf(s, 0, 5e-3, 1e-2, 0.0)
    ge, gi = 1.5 * 5 * 800 * 5e-3, 5.0 * 5 * 200 * 1e-2
    assert rel(muV, (ge * 0.0 + gi * -80.0 + 10 * -64.0) / (10 + ge + gi)) < 1e-13


def test_tf_clamp_rule_A10():
    """x <= 0: value is the TF at eps_nu and every derivative w.r.t. that argument is zero."""
    p = wl.param_vector()
    eps = p[wl.PARAM_NAMES.index("eps_nu")]
    out, _ = orc.tf(p, 0, -3e-4, 2e-3, 10.0)
    ref, _ = orc.tf(wl.param_vector(eps_nu=0.0), 0, eps, 2e-3 + eps, 10.0)
    assert rel(out[0], ref[0]) < 1e-14
    assert out[1] == 0.0 and out[3] == 0.0 and out[4] == 0.0
    assert rel(out[2], ref[2]) < 1e-14 and rel(out[5], ref[5]) < 1e-14
    out, _ = orc.tf(p, 1, 2e-3, 0.0, 0.0)
    assert out[2] == 0.0 and out[4] == 0.0 and out[5] == 0.0 and out[1] != 0.0
    # x > 0: value is TF(x + eps)
    out, _ = orc.tf(p, 0, 4e-3, 2e-3, 0.0)
    assert rel(out[0], float(M.tf(p, 0, 4e-3 + eps, 2e-3 + eps, 0.0))) < 1e-11


def test_tf_adaptation_lowers_rate_and_shifts_muV():
    """mu_V is linear in W with slope -1/mu_G (step 3 of DESIGN.md section 2)."""
    p = wl.param_vector(eps_nu=0.0)
    fe, fi = 4e-3, 8e-3
    muG = 10 + 1.5 * 5 * 400 * fe + 5 * 5 * 100 * fi
    o0, m0 = orc.tf(p, 0, fe, fi, 0.0)
    o1, m1 = orc.tf(p, 0, fe, fi, 100.0)
    assert rel(m1 - m0, -100.0 / muG) < 1e-12
    assert o1[0] < o0[0]

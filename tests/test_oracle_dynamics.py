"""Pins P3-P9, P12, P14, P15 of the oracle's time stepping, history ring and statistics."""
import math

import mpmath as mp
import numpy as np
import pytest

import workloads as wl
from oracle import oracle as orc
from tests import _mp_model as M

NM = wl.PARAM_NAMES.index


# --------------------------------------------------------------------------------------------
# An independent restatement of the bookkeeping (steps 1, 2, 5-11 of DESIGN.md section 2) in NumPy
# with a FLAT, unwrapped history array and direct time indexing.  The transfer function is taken
# from orc.tf, which is pinned on its own in test_oracle_tf.py; everything else (delay lookup,
# orientation of W, simultaneous update, noise injection, window alignment, discard) is re-derived.
# --------------------------------------------------------------------------------------------
def flat_history_sim(W, L, p, steps, dt, noise_on=False, seed=0, sim_id=0, ds=10, discard=0,
                     init=wl.INIT_STATE):
    N = W.shape[0]
    d = np.rint((L / p[NM("v")]) / dt).astype(np.int64)
    y = np.tile(np.array(init, dtype=np.float64)[:, None], (1, N))
    ou = np.zeros(N)
    Eh = np.zeros((steps + 1, N)); Eh[0] = y[0]
    T, kap = p[NM("T")], p[NM("kappa")]
    Ne = p[NM("N_tot")] * (1 - p[NM("g_inh")]); Ni = p[NM("N_tot")] * p[NM("g_inh")]
    traj = np.zeros((steps, 7, N)); xe = []; xi = []
    acc_e = np.zeros(N); acc_i = np.zeros(N)
    rho = math.exp(-dt / p[NM("tau_OU")])
    for n in range(steps):
        new = np.zeros_like(y)
        for k in range(N):
            c = 0.0
            for j in range(N):
                if W[k, j] != 0.0:
                    m = n - d[k, j]
                    c += W[k, j] * (Eh[m, j] if m >= 0 else init[0])
            E, I, Cee, Cei, Cii, We, Wi = y[:, k]
            drive = E + p[NM("G")] * c + (p[NM("wNoise")] * ou[k] if noise_on else 0.0)
            Fe, mue = orc.tf(p, 0, drive + p[NM("c_Fee")], I + p[NM("c_Fei")], We)
            Fi, mui = orc.tf(p, 1, drive + p[NM("c_Fie")], I + p[NM("c_Fii")], Wi)
            Fe = Fe * np.array([1, kap, kap, kap**2, kap**2, kap**2])
            Fi = Fi * np.array([1, kap, kap, kap**2, kap**2, kap**2])
            dE = (Fe[0] - E + 0.5 * Cee * Fe[3] + Cei * Fe[4] + 0.5 * Cii * Fe[5]) / T
            dI = (Fi[0] - I + 0.5 * Cee * Fi[3] + Cei * Fi[4] + 0.5 * Cii * Fi[5]) / T
            dCee = (Fe[0] * (1 / T - Fe[0]) / Ne + (Fe[0] - E) ** 2 + 2 * (Cee * Fe[1] + Cei * Fe[2]) - 2 * Cee) / T
            dCii = (Fi[0] * (1 / T - Fi[0]) / Ni + (Fi[0] - I) ** 2 + 2 * (Cei * Fi[1] + Cii * Fi[2]) - 2 * Cii) / T
            dCei = ((Fe[0] - E) * (Fi[0] - I) + Cei * Fe[1] + Cii * Fe[2] + Cee * Fi[1] + Cei * Fi[2] - 2 * Cei) / T
            dWe = -We / p[NM("tau_w_e")] + p[NM("b_e")] * E + p[NM("a_e")] * (mue - p[NM("E_L_e")]) / p[NM("tau_w_e")]
            dWi = -Wi / p[NM("tau_w_i")] + p[NM("b_i")] * I + p[NM("a_i")] * (mui - p[NM("E_L_i")]) / p[NM("tau_w_i")]
            new[:, k] = y[:, k] + dt * np.array([dE, dI, dCee, dCei, dCii, dWe, dWi])
        if noise_on:
            xi_n = np.array([orc.normal(seed, sim_id, k, n) for k in range(N)])
            ou = p[NM("mu_OU")] + (ou - p[NM("mu_OU")]) * rho + p[NM("sigma_OU")] * math.sqrt(1 - rho * rho) * xi_n
        y = new
        Eh[n + 1] = y[0]
        traj[n] = y
        acc_e += y[0]; acc_i += y[1]
        if (n + 1) % ds == 0:
            if n + 1 > discard:
                xe.append(acc_e / ds); xi.append(acc_i / ds)
            acc_e = np.zeros(N); acc_i = np.zeros(N)
    return traj, np.array(xe), np.array(xi)


def small_net(n=5, seed=3, lo=0.3, hi=2.4):
    rng = np.random.default_rng(seed)
    W = rng.uniform(0.1, 1.0, (n, n)) * (rng.random((n, n)) < 0.6)
    np.fill_diagonal(W, 0.0)
    L = rng.uniform(lo, hi, (n, n))          # NOT symmetric: orientation mistakes show up
    return W, L


def test_ring_oracle_equals_flat_history_restatement():
    """P5/P6 + steps 1,2,5-11: delays 1..6 steps, ring wraps > 10 times, noise on, ds=4, discard."""
    W, L = small_net()
    p = wl.param_vector(G=0.4, b_e=20.0, a_e=2.0, v=4.0, kappa=1e-3, wNoise=1e-4)
    steps = 73
    ref_traj, ref_xe, ref_xi = flat_history_sim(W, L, p, steps, 0.1, True, seed=9, sim_id=4, ds=4, discard=9)
    sw = orc.OracleSweep(W, L, p[None], seed=9, ext_ids=[4])
    traj = sw.run(steps, 0.1, noise_on=True, ds=4, discard_steps=9, traj_steps=steps)[0]
    assert sw.ring_len(0) == int(np.rint(L[W != 0] / 4.0 / 0.1).max()) + 1 < 10
    np.testing.assert_allclose(traj, ref_traj, rtol=1e-12, atol=1e-300)
    xe, xi = sw.samples(0)
    assert xe.shape == ref_xe.shape == (16, 5)        # windows ending at 12..72 (first two dropped)
    np.testing.assert_allclose(xe, ref_xe, rtol=1e-12)
    np.testing.assert_allclose(xi, ref_xi, rtol=1e-12)
    # sample w is the mean of the post-update values of steps w*ds+1 .. (w+1)*ds (A17)
    np.testing.assert_allclose(xe[0], traj[8:12, 0].mean(0), rtol=1e-13)


def test_ring_equals_unwrapped_history_variant_bitwise():
    """P6: modulo ring (H = D+1) vs the oracle variant that keeps the whole history."""
    W, L = small_net(6, 5)
    P = np.stack([wl.param_vector(G=0.3, v=4.0), wl.param_vector(G=0.5, v=2.0, b_e=60.0)])
    a = orc.OracleSweep(W, L, P, seed=2).run(90, 0.1, noise_on=True, traj_steps=90)
    b = orc.OracleSweep(W, L, P, seed=2, unwrapped=True).run(90, 0.1, noise_on=True, traj_steps=90)
    assert np.array_equal(a, b)


def test_infinite_speed_equals_zero_delay():
    """P5: v = 1e9 => every d = 0 => coupling uses the current state (flat restatement, d = 0)."""
    W, L = small_net(4, 8, 10.0, 200.0)
    p = wl.param_vector(G=0.5, v=1e9)
    assert np.rint(L / 1e9 / 0.1).max() == 0
    ref, _, _ = flat_history_sim(W, L, p, 40, 0.1)
    sw = orc.OracleSweep(W, L, p[None])
    traj = sw.run(40, 0.1, traj_steps=40)[0]
    assert sw.ring_len(0) == 1
    np.testing.assert_allclose(traj, ref, rtol=1e-12, atol=1e-300)
    # and differs from a delayed run
    tr4 = orc.OracleSweep(W, L, wl.param_vector(G=0.5, v=4.0)[None]).run(40, 0.1, traj_steps=40)[0]
    assert not np.allclose(traj[-1, 0], tr4[-1, 0], rtol=1e-6)


def test_single_node_matches_mpmath_euler_with_literal_index_sums():
    """P3/P8: G = 0 => every region follows the isolated-node ODE.  The reference integrates
    Eqs. (1)-(3) written as literal sums over population indices with numerically differentiated
    40-digit transfer functions (tests/_mp_model.py).  kappa = 1 so the derivative terms carry
    full weight; a = b != 0 exercises Eq. (3)."""
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    for kw in (dict(kappa=1.0, b_e=40.0, a_e=3.0, a_i=1.0, b_i=5.0), dict(kappa=1e-3, b_e=60.0)):
        p = wl.param_vector(G=0.0, **kw)
        steps = 14
        traj = orc.OracleSweep(W, L, p[None]).run(steps, 0.1, traj_steps=steps)[0]
        assert np.all(traj == traj[:, :, :1])            # all regions bit-identical
        y = [mp.mpf(x) for x in wl.INIT_STATE]
        for n in range(steps):
            dy = M.rhs_node(p, y)
            y = [a + mp.mpf("0.1") * b for a, b in zip(y, dy)]
            got = traj[n, :, 0]
            for q in range(7):
                assert abs(got[q] - float(y[q])) <= 1e-10 * max(abs(float(y[q])), 1e-12), (n, q)


def test_coupled_step_matches_mpmath_rhs():
    """Eq. (5): the coupling G*c_k and the noise enter the excitatory argument of BOTH populations."""
    W, L = small_net(3, 11)
    p = wl.param_vector(G=0.7, kappa=1.0, v=4.0, c_Fie=0.5e-3, c_Fei=0.1e-3, c_Fii=0.2e-3)
    init = np.array([2e-3, 5e-3, 1e-7, -2e-8, 3e-7, 12.0, 0.5])
    traj = orc.OracleSweep(W, L, p[None], init=init).run(1, 0.1, traj_steps=1)[0]
    for k in range(3):
        c = sum(W[k, j] * init[0] for j in range(3))
        dy = M.rhs_node(p, [mp.mpf(float(x)) for x in init], drive_extra=mp.mpf(0.7) * mp.mpf(float(c)))
        for q in range(7):
            ref = float(mp.mpf(float(init[q])) + mp.mpf("0.1") * dy[q])
            assert abs(traj[0, q, k] - ref) <= 1e-11 * max(abs(ref), 1e-12)


def test_fixed_point_G0_all_regions_converge_to_single_node_root():
    """P3: noise off, G = 0 => all regions converge to the root of the isolated-node RHS
    (found independently with mpmath.findroot on the first-order part, kappa -> tiny)."""
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    p = wl.param_vector(G=0.0, b_e=0.0)
    sw = orc.OracleSweep(W, L, p[None])
    sw.run(8000, 0.1, ds=0)
    y, _ = sw.state(0)
    assert np.all(y == y[:, :1])
    E, I = y[0, 0], y[1, 0]
    # at the fixed point of Eq. (1) with the (tiny) second-order terms: F_e - E = -corr_e etc.
    dy = M.rhs_node(p, [mp.mpf(float(v)) for v in y[:, 0]])
    assert all(abs(float(d)) < 1e-9 for d in dy[:5])
    assert 0.2e-3 < E < 2e-3 and 0.5e-3 < I < 5e-3       # healthy band


def test_identical_regions_stay_identical():
    """P4: circulant W (equal row sums), equal tract lengths, identical initial state, noise off."""
    n = 9
    W = np.zeros((n, n))
    for k in range(n):
        W[k, (k + 1) % n] = 0.5; W[k, (k - 1) % n] = 0.25
    L = np.full((n, n), 12.0)
    p = wl.param_vector(G=0.6, v=4.0, b_e=30.0)
    traj = orc.OracleSweep(W, L, p[None]).run(400, 0.1, traj_steps=400)[0]
    assert np.all(traj == traj[:, :, :1])
    # equals a scalar delay recursion fed by rowsum * E(t - d), d = 30 steps
    Wc = np.array([[0.0, 0.75], [0.75, 0.0]]); Lc = np.full((2, 2), 12.0)
    ref = orc.OracleSweep(Wc, Lc, p[None]).run(400, 0.1, traj_steps=400)[0]
    np.testing.assert_allclose(traj[:, :, 0], ref[:, :, 0], rtol=1e-12)


def test_adaptation_closed_forms():
    """P7: a = b = 0 => W_n = W_0 (1 - dt/tau_w)^n; b != 0 at the E fixed point => geometric series."""
    W = np.zeros((2, 2)); L = np.zeros((2, 2))
    p = wl.param_vector(a_e=0.0, b_e=0.0, tau_w_e=37.0, tau_w_i=11.0)
    init = np.array([1e-3, 1e-3, 0, 0, 0, 80.0, -15.0])
    traj = orc.OracleSweep(W, L, p[None], init=init).run(200, 0.1, traj_steps=200)[0]
    n = np.arange(1, 201)
    np.testing.assert_allclose(traj[:, 5, 0], 80.0 * (1 - 0.1 / 37.0) ** n, rtol=1e-12)
    np.testing.assert_allclose(traj[:, 6, 1], -15.0 * (1 - 0.1 / 11.0) ** n, rtol=1e-12)
    # one step with a != 0: dW = -W/tau + b E + a (mu_V - E_L)/tau  (A9)
    p = wl.param_vector(a_e=4.0, b_e=25.0, tau_w_e=50.0)
    init = np.array([3e-3, 6e-3, 0, 0, 0, 10.0, 0.0])
    t1 = orc.OracleSweep(W, L, p[None], init=init).run(1, 0.1, traj_steps=1)[0]
    _, muV = orc.tf(p, 0, 3e-3 + 0.3e-3, 6e-3, 10.0)
    ref = 10.0 + 0.1 * (-10.0 / 50.0 + 25.0 * 3e-3 + 4.0 * (muV + 64.0) / 50.0)
    assert abs(t1[0, 5, 0] - ref) < 1e-13


def test_muV_local_option_changes_only_adaptation_drive():
    W, L = small_net(3, 2)
    init = np.array([3e-3, 6e-3, 0, 0, 0, 10.0, 0.0])
    a = orc.OracleSweep(W, L, wl.param_vector(G=0.5, a_e=4.0)[None], init=init).run(1, 0.1, traj_steps=1)[0]
    b = orc.OracleSweep(W, L, wl.param_vector(G=0.5, a_e=4.0, muV_local=1.0)[None], init=init).run(1, 0.1, traj_steps=1)[0]
    assert np.array_equal(a[0, :5], b[0, :5]) and not np.array_equal(a[0, 5], b[0, 5])
    _, muV = orc.tf(wl.param_vector(), 0, 3e-3, 6e-3, 10.0)       # local rates only, no drive/ext
    ref = 10.0 + 0.1 * (-10.0 / 500.0 + 4.0 * (muV + 64.0) / 500.0)
    assert abs(b[0, 5, 0] - ref) < 1e-13


def test_euler_is_first_order():
    """P9: halving dt halves the error against the Richardson limit (delays fixed in ms)."""
    W, L = small_net(4, 6, 0.8, 2.4)          # multiples of dt at all three resolutions? not needed:
    L = np.round(L / 0.4) * 0.4               # delays = multiples of 0.1 ms at v = 4
    p = wl.param_vector(G=0.4, v=4.0, b_e=40.0)
    end = {}
    for dt, steps in ((0.1, 500), (0.05, 1000), (0.025, 2000), (0.0125, 4000)):
        sw = orc.OracleSweep(W, L, p[None])
        sw.run(steps, dt, ds=0)
        end[dt] = sw.state(0)[0][:2]
    lim = 2 * end[0.0125] - end[0.025]
    e1, e2, e3 = (np.abs(end[d] - lim).max() for d in (0.1, 0.05, 0.025))
    assert 1.8 < e1 / e2 < 2.2 and 1.8 < e2 / e3 < 2.3


def test_fc_and_means_vs_numpy_corrcoef():
    """P12: two-pass FC equals numpy.corrcoef of the oracle's own samples; degenerate rule A18."""
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    P = wl.grid_params(cfg)[[4, 7]]
    P[:, NM("wNoise")] = 1e-4
    sw = orc.OracleSweep(W, L, P, seed=1, ext_ids=[4, 7])
    sw.run(3000, 0.1, noise_on=True, ds=10, discard_steps=1000)
    fc, me, mi = sw.fc_readout()
    for s in range(2):
        xe, xi = sw.samples(s)
        assert xe.shape == (200, 68)
        np.testing.assert_allclose(fc[s], np.corrcoef(xe.T), atol=1e-12)
        np.testing.assert_allclose(me[s], xe.mean(0), rtol=1e-13)
        np.testing.assert_allclose(mi[s], xi.mean(0), rtol=1e-13)
        assert np.all(np.diag(fc[s]) == 1.0) and np.abs(fc[s]).max() <= 1 + 1e-12
    # noise off, G = 0 at the fixed point: constant series -> off-diagonal 0, diagonal 1 (A18)
    sw = orc.OracleSweep(W[:4, :4] * 0, L[:4, :4], wl.param_vector()[None],
                         init=np.array([0.0, 0.0, 0, 0, 0, 0, 0]))
    sw2 = orc.OracleSweep(np.zeros((3, 3)), np.zeros((3, 3)), wl.param_vector(T=1e30)[None])
    sw2.run(40, 0.1, ds=10)
    fc2, _, _ = sw2.fc_readout()
    assert np.array_equal(fc2[0], np.eye(3))
    with pytest.raises(RuntimeError):
        s3 = orc.OracleSweep(np.zeros((3, 3)), np.zeros((3, 3)), wl.param_vector()[None])
        s3.run(10, 0.1, ds=10)
        s3.fc_readout()


def test_fc_independent_regions_uncorrelated_when_G0():
    """P12: G = 0, noise on => regions are independent => off-diagonal FC ~ 0 within MC error."""
    W, L = wl.connectome(12, 1, 0.5)
    sw = orc.OracleSweep(W, L, wl.param_vector(G=0.0)[None], seed=5)
    sw.run(42000, 0.1, noise_on=True, ds=10, discard_steps=2000)
    fc, _, _ = sw.fc_readout()
    off = fc[0][~np.eye(12, dtype=bool)]
    # samples are 1 ms apart and correlated over ~T = 20 ms -> n_eff ~ 4000 / 40
    assert np.abs(off).max() < 5 / math.sqrt(100) and abs(off.mean()) < 0.1


def test_resumable_bitwise():
    """P14: run(a); run(b) == run(a+b), including windows that straddle the split."""
    W, L = small_net(5, 4, 2.0, 9.0)
    P = np.stack([wl.param_vector(G=0.3, b_e=30.0), wl.param_vector(G=0.5)])
    a = orc.OracleSweep(W, L, P, seed=7)
    a.run(137, 0.1, noise_on=True, ds=10, discard_steps=20)
    b = orc.OracleSweep(W, L, P, seed=7)
    b.run(64, 0.1, noise_on=True, ds=10, discard_steps=20)
    b.run(73, 0.1, noise_on=True, ds=10, discard_steps=20)
    assert b.steps_done() == 137
    for s in range(2):
        assert all(np.array_equal(x, y) for x, y in zip(a.state(s), b.state(s)))
        assert all(np.array_equal(x, y) for x, y in zip(a.samples(s), b.samples(s)))
    with pytest.raises(ValueError):
        b.run(1, 0.05)


def test_simulations_are_independent_of_sweep_composition():
    """a simulation's result depends only on its parameters and its external index."""
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    P = wl.grid_params(cfg)
    full = orc.OracleSweep(W, L, P, seed=1)
    full.run(300, 0.1, noise_on=True)
    sub = orc.OracleSweep(W, L, P[[6, 2]], seed=1, ext_ids=[6, 2])
    sub.run(300, 0.1, noise_on=True)
    assert np.array_equal(full.state(6)[0], sub.state(0)[0])
    assert np.array_equal(full.state(2)[0], sub.state(1)[0])


def test_physiological_sanity_config1():
    """P15 (not parity): rates finite, inside the healthy band, b_e lowers E, G raises I."""
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    P = wl.grid_params(cfg)
    sw = orc.OracleSweep(W, L, P, seed=1)
    tr = sw.run(5000, 0.1, noise_on=True, traj_steps=5000)
    assert np.isfinite(tr).all()
    assert tr[:, :, :2].max() < 0.02 and tr[:, :, :2].min() > 0
    endE = tr[:, -1, 0].mean(1); endI = tr[:, -1, 1].mean(1)
    assert np.all(np.diff(endE[:4]) < 0) and np.all(np.diff(endE[4:]) < 0)
    assert np.all(endI[4:] > endI[:4])

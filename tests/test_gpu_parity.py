"""GPU parity: the CUDA path (through the C ABI) against the FP64 oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json's: noise-off trajectories max relative error 1e-3
(FP32) / 1e-9 (FP64 build mode) over the first 200 ms; noise-on per-region means 1 % relative and FC
0.02 absolute; bookkeeping and resumability bit-exact."""
import numpy as np
import pytest

import workloads as wl
import paper_2311_13337_b200 as tvbx
from oracle import oracle as orc

pytestmark = pytest.mark.gpu

TOL_TRAJ_F32 = 1e-3     # BASELINE.json north_star
TOL_TRAJ_F64 = 1e-9
TOL_MEAN_REL = 1e-2
TOL_FC_ABS = 0.02


def traj_err(got, ref):
    """max over everything of |got - ref| / (max |ref| of that state variable of that sim): the
    relative error of a trajectory, scaled per variable so that zero crossings do not divide by 0."""
    ref = np.asarray(ref, dtype=np.float64)
    scale = np.abs(ref).max(axis=(1, 3), keepdims=True) + 1e-300
    return float((np.abs(np.asarray(got, dtype=np.float64) - ref) / scale).max())


def run_pair(cfg, W, L, steps, noise_on, traj_steps=0, sims=None, precision=tvbx.TVBX_F32, ds=10,
             discard=0, params=None, **kw):
    P = wl.grid_params(cfg, sims=sims)
    if params:
        for k, v in params.items():
            P[:, wl.PARAM_NAMES.index(k)] = v
    conn, sw = tvbx.sweep_from_config(cfg, W, L, sim_ids=sims, precision=precision, params=params, **kw)
    traj = sw.run(steps, cfg.get("dt", 0.1), noise_on=noise_on, ds=ds, discard_steps=discard, traj_steps=traj_steps)
    o = orc.OracleSweep(W, L, P, seed=cfg["seed"], ext_ids=sims)
    ref = o.run(steps, cfg.get("dt", 0.1), noise_on=noise_on, ds=ds, discard_steps=discard, traj_steps=traj_steps)
    return sw, traj, o, ref


# ------------------------------------------------------------------------------------ cfg 1
def test_cfg1_noise_off_trajectories_fp32():
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    sw, traj, o, ref = run_pair(cfg, W, L, 2000, False, traj_steps=2000)
    assert traj.shape == (8, 2000, 7, 68) and traj.dtype == np.float32
    assert traj_err(traj, ref) < TOL_TRAJ_F32
    y, _ = sw.state()
    for s in range(8):
        np.testing.assert_allclose(y[s], o.state(s)[0], rtol=TOL_TRAJ_F32, atol=1e-9)


def test_cfg1_noise_off_trajectories_fp64_mode():
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    sw, traj, o, ref = run_pair(cfg, W, L, 2000, False, traj_steps=2000, precision=tvbx.TVBX_F64)
    assert traj.dtype == np.float64
    assert traj_err(traj, ref) < TOL_TRAJ_F64


def test_cfg1_noise_on_means_and_fc():
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    sw, _, o, _ = run_pair(cfg, W, L, cfg["steps"], True)
    fc, me, mi = sw.fc_readout()
    rfc, rme, rmi = o.fc_readout()
    assert sw.samples_kept() == 500
    assert np.abs(me / rme - 1).max() < TOL_MEAN_REL
    assert np.abs(mi / rmi - 1).max() < TOL_MEAN_REL
    assert np.abs(fc - rfc).max() < TOL_FC_ABS
    assert np.all(np.diagonal(fc, axis1=1, axis2=2) == 1.0)
    np.testing.assert_array_equal(fc, np.swapaxes(fc, 1, 2))


def test_cfg1_noise_on_trajectory_same_philox_stream():
    """Same Philox stream => the noisy trajectories also agree closely over the first 100 ms (the OU
    path is identical up to FP32 rounding of Box-Muller)."""
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    sw, traj, o, ref = run_pair(cfg, W, L, 1000, True, traj_steps=1000, params=dict(wNoise=1e-4))
    assert traj_err(traj, ref) < TOL_TRAJ_F32
    _, ou = sw.state()
    for s in range(8):
        np.testing.assert_allclose(ou[s], o.state(s)[1], rtol=0, atol=2e-4)


def test_fp64_mode_noise_on_matches_oracle_tightly():
    cfg = wl.config(1)
    W, L = wl.connectome(23, seed=11, keep=0.4)
    sw, traj, o, ref = run_pair(cfg, W, L, 1200, True, traj_steps=1200, precision=tvbx.TVBX_F64,
                                params=dict(wNoise=1e-4), discard=200)
    assert traj_err(traj, ref) < 1e-8
    fc, me, mi = sw.fc_readout()
    rfc, rme, rmi = o.fc_readout()
    np.testing.assert_allclose(me, rme, rtol=1e-6)
    np.testing.assert_allclose(mi, rmi, rtol=1e-6)
    assert np.abs(fc - rfc).max() < 1e-5


def test_general_tau_path_fp32_and_fp64():
    """tau_e != tau_i switches the kernels from the closed-form transfer function to the jet one."""
    W, L = wl.connectome(24, seed=12, keep=0.4)
    cfg = dict(axes=[dict(name="G", lo=0.0, hi=0.4, n=3, values=None)], fixed=dict(v=5.0, b_e=40.0, wNoise=1e-4), seed=6)
    for kappa in (1e-3, 0.05):
        par = dict(tau_i=7.5, kappa=kappa)
        sw, traj, o, ref = run_pair(cfg, W, L, 800, True, traj_steps=800, params=par)
        assert traj_err(traj, ref) < TOL_TRAJ_F32
        sw, traj, o, ref = run_pair(cfg, W, L, 800, True, traj_steps=800, params=par, precision=tvbx.TVBX_F64)
        assert traj_err(traj, ref) < 1e-8


def test_derivative_terms_carry_weight_kappa():
    """A22 with a kappa large enough that the first/second-derivative terms of Eqs. (1)-(2) matter
    (closed-form path), FP32 and FP64; also the A9b option and non-default c_F, E_L, a, b."""
    W, L = wl.connectome(24, seed=13, keep=0.4)
    cfg = dict(axes=[dict(name="b_e", lo=0.0, hi=60.0, n=3, values=None)],
               fixed=dict(v=5.0, G=0.3, wNoise=1e-4, kappa=0.05, a_e=4.0, a_i=1.0, b_i=2.0, E_L_e=-63.0, E_L_i=-65.0,
                          c_Fie=0.5e-3, c_Fei=0.1e-3, c_Fii=0.2e-3, muV_local=1.0), seed=8)
    sw, traj, o, ref = run_pair(cfg, W, L, 800, True, traj_steps=800)
    assert traj_err(traj, ref) < TOL_TRAJ_F32
    sw, traj, o, ref = run_pair(cfg, W, L, 800, True, traj_steps=800, precision=tvbx.TVBX_F64)
    assert traj_err(traj, ref) < 1e-8


# ------------------------------------------------------------------------------------ launch shapes
@pytest.mark.parametrize("spc", [1, 2, 4, 8, 16, 32])
def test_every_sims_per_cta_mapping(spc):
    """Ragged everything: 11 sims (not a multiple of any SPC > 1), N = 37 regions, two speeds."""
    W, L = wl.connectome(37, seed=5, keep=0.35)
    axes = [dict(name="G", lo=0.0, hi=0.4, n=11, values=None)]
    cfg = dict(axes=axes, fixed=dict(v=6.0, b_e=20.0, wNoise=1e-4), seed=9)
    sw, traj, o, ref = run_pair(cfg, W, L, 700, True, traj_steps=700, sims_per_cta=spc, discard=100)
    assert traj_err(traj, ref) < TOL_TRAJ_F32
    fc, me, mi = sw.fc_readout()
    rfc, rme, rmi = o.fc_readout()
    assert np.abs(me / rme - 1).max() < TOL_MEAN_REL and np.abs(fc - rfc).max() < TOL_FC_ABS
    assert sw.launch_info()["sims_per_cta"] == spc


@pytest.mark.parametrize("threads", [64, 160, 0])
def test_multi_pass_mapping_when_regions_exceed_the_cta(threads):
    """threads_per_cta < N * SPC forces several region passes per time block (the N = 360 path)."""
    W, L = wl.connectome(45, seed=6, keep=0.5)
    axes = [dict(name="b_e", lo=0.0, hi=60.0, n=5, values=None)]
    cfg = dict(axes=axes, fixed=dict(v=3.0, G=0.3), seed=2)
    sw, traj, o, ref = run_pair(cfg, W, L, 500, False, traj_steps=500, sims_per_cta=4, threads_per_cta=threads)
    assert traj_err(traj, ref) < TOL_TRAJ_F32


@pytest.mark.parametrize("clu,spc", [(2, 4), (3, 8), (8, 3), (5, 1)])
def test_cluster_mapping_regions_split_over_ctas(clu, spc):
    """ctas_per_group > 1: the regions of a group are split over the CTAs of a thread-block cluster (the
    N = 360 mapping), chunk hand-over through cluster-scope mbarriers.  Ragged: 37 regions over 2, 3, 5, 8
    CTAs, 12 sims in two speed classes (long and short chunks), sims per group not dividing the class."""
    W, L = wl.connectome(37, seed=5, keep=0.35)
    axes = [dict(name="G", lo=0.0, hi=0.4, n=6, values=None), dict(name="v", lo=0, hi=0, n=2, values=[3.0, 40.0])]
    cfg = dict(axes=axes, fixed=dict(b_e=20.0, wNoise=1e-4), seed=9)
    sw, traj, o, ref = run_pair(cfg, W, L, 700, True, traj_steps=700, sims_per_cta=spc, ctas_per_group=clu, discard=100)
    info = sw.launch_info()
    assert info["ctas_per_group"] == clu and info["sims_per_cta"] == spc and sw.kernel_name() == "tvbx::integrate2_kernel"
    assert traj_err(traj, ref) < TOL_TRAJ_F32
    fc, me, mi = sw.fc_readout()
    rfc, rme, rmi = o.fc_readout()
    assert np.abs(me / rme - 1).max() < TOL_MEAN_REL and np.abs(fc - rfc).max() < TOL_FC_ABS


def test_cluster_mapping_is_bitwise_the_single_cta_mapping():
    """The cluster (scalar gather: short chunks at v = 40 m/s) only changes which CTA owns a region: same
    per-node arithmetic, same edge order -> the trajectories equal those of the one-CTA mapping bit for bit."""
    W, L = wl.connectome(37, seed=5, keep=0.35)
    cfg = dict(axes=[dict(name="G", lo=0.0, hi=0.4, n=5, values=None)], fixed=dict(v=40.0, wNoise=1e-4), seed=4)
    _, a = tvbx.sweep_from_config(cfg, W, L, sims_per_cta=4, ctas_per_group=1)
    _, b = tvbx.sweep_from_config(cfg, W, L, sims_per_cta=4, ctas_per_group=4)
    ta = a.run(900, 0.1, noise_on=True, ds=10, traj_steps=900)
    tb = b.run(900, 0.1, noise_on=True, ds=10, traj_steps=900)
    np.testing.assert_array_equal(ta, tb)
    np.testing.assert_array_equal(a.fc_readout()[0], b.fc_readout()[0])


def test_mixed_speeds_cfg3_slice():
    """cfg 3 slice covering all 8 speeds (ring depth 16 ... 2000, min delay 1 ... 100 steps)."""
    cfg = wl.config(3)
    W, L = wl.config_connectome(cfg)
    sims = list(range(8 * 100, 8 * 100 + 8)) + [32767, 32760]
    sw, traj, o, ref = run_pair(cfg, W, L, 2000, False, traj_steps=2000, sims=sims)
    assert traj_err(traj, ref) < TOL_TRAJ_F32
    for loc, s in enumerate(sims):
        assert sw.ring_len(loc)[0] == o.ring_len(loc)


def test_zero_delay_edges():
    """v so large that every delay rounds to 0: the coupling reads the current step (pin P5)."""
    W, L = wl.connectome(19, seed=8, keep=0.5)
    cfg = dict(axes=[dict(name="G", lo=0.1, hi=0.5, n=3, values=None)], fixed=dict(v=1e9), seed=0)
    sw, traj, o, ref = run_pair(cfg, W, L, 400, False, traj_steps=400)
    assert sw.ring_len(0)[0] == 1
    assert traj_err(traj, ref) < TOL_TRAJ_F32


def test_cfg5_slice_n360():
    cfg = wl.config(5)
    W, L = wl.config_connectome(cfg)
    sims = [0, 63, 2047, 4095]
    sw, traj, o, ref = run_pair(cfg, W, L, 800, True, traj_steps=800, sims=sims, discard=200)
    assert traj_err(traj, ref) < TOL_TRAJ_F32
    fc, me, mi = sw.fc_readout()
    rfc, rme, rmi = o.fc_readout()
    assert fc.shape == (4, 360, 360)
    assert np.abs(me / rme - 1).max() < TOL_MEAN_REL and np.abs(mi / rmi - 1).max() < TOL_MEAN_REL
    assert np.abs(fc - rfc).max() < TOL_FC_ABS


# ------------------------------------------------------------------------------------ invariants on the GPU path
@pytest.mark.parametrize("kw", [dict(), dict(sims_per_cta=4, ctas_per_group=3)], ids=["one_cta", "cluster_vector_gather"])
def test_resumable_bit_exact(kw):
    """P14: run(a); run(b) == run(a+b) bit for bit (state, OU, FC accumulators).  In the cluster form with
    the vector gather every launch starts with a short unaligned chunk gathered by scalar loads: it has to
    reproduce the association of the vector path exactly."""
    W, L = wl.connectome(30, seed=3, keep=0.4)
    cfg = dict(axes=[dict(name="G", lo=0.0, hi=0.5, n=6, values=None)], fixed=dict(v=5.0, b_e=30.0, wNoise=1e-4), seed=4)
    _, a = tvbx.sweep_from_config(cfg, W, L, chunk_samples=16, **kw)
    _, b = tvbx.sweep_from_config(cfg, W, L, chunk_samples=16, **kw)
    a.run(1203, 0.1, noise_on=True, ds=10, discard_steps=95)
    for part in (1, 398, 7, 797):
        b.run(part, 0.1, noise_on=True, ds=10, discard_steps=95)
    assert a.steps_done() == b.steps_done() == 1203 and a.samples_kept() == b.samples_kept()
    ya, oa = a.state(); yb, ob = b.state()
    np.testing.assert_array_equal(ya, yb); np.testing.assert_array_equal(oa, ob)
    for x, y in zip(a.fc_readout(), b.fc_readout()):
        np.testing.assert_array_equal(x, y)


def test_reset_equals_fresh_sweep():
    W, L = wl.connectome(30, seed=3, keep=0.4)
    cfg = dict(axes=[dict(name="G", lo=0.0, hi=0.5, n=5, values=None)], fixed=dict(v=5.0, b_e=30.0, wNoise=1e-4), seed=4)
    _, a = tvbx.sweep_from_config(cfg, W, L)
    _, b = tvbx.sweep_from_config(cfg, W, L)
    a.run(777, 0.1, noise_on=True, ds=10, discard_steps=100)
    a.reset()
    assert a.steps_done() == 0 and a.samples_kept() == 0
    ta = a.run(500, 0.1, noise_on=True, ds=10, discard_steps=100, traj_steps=500)
    tb = b.run(500, 0.1, noise_on=True, ds=10, discard_steps=100, traj_steps=500)
    np.testing.assert_array_equal(ta, tb)
    for x, y in zip(a.fc_readout(), b.fc_readout()):
        np.testing.assert_array_equal(x, y)
    a.profile_enable(True)
    a.run(100, 0.1, noise_on=True, ds=10, discard_steps=100)
    prof = a.profile_read()
    assert prof["integrate"][1] >= 1 and prof["integrate"][0] > 0.0


def test_sim_results_do_not_depend_on_sweep_membership():
    """P13 / P:86: a simulation's result is the same whatever other simulations share the sweep,
    its position in it, or its lane in a CTA (Philox is keyed by the external sim index)."""
    cfg = wl.config(3)
    W, L = wl.connectome(26, seed=1, keep=0.4)
    full = [9, 4000, 4001, 17, 30000, 12345, 8, 4002]
    _, a = tvbx.sweep_from_config(cfg, W, L, sim_ids=full, sims_per_cta=4, params=dict(wNoise=1e-4))
    _, b = tvbx.sweep_from_config(cfg, W, L, sim_ids=[12345, 9], sims_per_cta=1, params=dict(wNoise=1e-4))
    ta = a.run(600, 0.1, noise_on=True, ds=10, traj_steps=600)
    tb = b.run(600, 0.1, noise_on=True, ds=10, traj_steps=600)
    np.testing.assert_array_equal(ta[5], tb[0])
    np.testing.assert_array_equal(ta[0], tb[1])
    fa, fb = a.fc_readout(), b.fc_readout()
    np.testing.assert_array_equal(fa[1][5], fb[1][0])
    np.testing.assert_allclose(fa[0][5], fb[0][0], atol=1e-6)


def test_uncoupled_regions_reach_the_single_node_fixed_point():
    """BASELINE invariant 1 on the GPU path: noise off, G = 0 => all regions identical."""
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    _, sw = tvbx.sweep_from_config(cfg, W, L, sim_ids=[0, 1, 2, 3])
    traj = sw.run(3000, 0.1, noise_on=False, ds=10, traj_steps=3000)
    assert np.all(traj == traj[..., :1])


def test_device_buffers_and_stream():
    """Device-pointer outputs on a non-default torch stream give the same numbers as host outputs."""
    import torch
    cfg = wl.config(1)
    W, L = wl.connectome(21, seed=2, keep=0.5)
    _, a = tvbx.sweep_from_config(cfg, W, L)
    _, b = tvbx.sweep_from_config(cfg, W, L)
    ta = a.run(300, 0.1, noise_on=True, ds=10, traj_steps=300)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        tb = b.run(300, 0.1, noise_on=True, ds=10, traj_steps=300, traj_device=True, stream=st)
        fb = b.fc_readout(device=True, stream=st)
    st.synchronize()
    np.testing.assert_array_equal(ta, tb.cpu().numpy())
    for x, y in zip(a.fc_readout(), fb):
        np.testing.assert_array_equal(x, y.cpu().numpy())


def test_degenerate_fc_is_nan_free():
    """A18: noise off at the fixed point => zero variance => FC = 0 off the diagonal, 1 on it."""
    W, L = wl.connectome(12, seed=2, keep=0.5)
    cfg = dict(axes=[], fixed=dict(G=0.0), seed=0)
    _, sw = tvbx.sweep_from_config(cfg, W, L, init=(0.0, 0.0, 0, 0, 0, 0, 0), params=dict(T=1e9))
    sw.run(200, 0.1, noise_on=False, ds=10)
    fc, me, mi = sw.fc_readout()
    assert np.isfinite(fc).all() and np.isfinite(me).all()
    assert np.all(np.diagonal(fc, axis1=1, axis2=2) == 1.0)


def test_too_few_samples_is_an_error():
    W, L = wl.connectome(12, seed=2, keep=0.5)
    _, sw = tvbx.sweep_from_config(dict(axes=[], fixed={}, seed=0), W, L)
    sw.run(15, 0.1, ds=10)
    with pytest.raises(tvbx.TvbxError):
        sw.fc_readout()
    with pytest.raises(tvbx.TvbxError):
        sw.run(5, 0.05)      # dt must not change


# ------------------------------------------------------------------------------------ full size, sampled
def test_cfg2_full_size_sampled_against_oracle():
    """cfg 2 at full size in the launch configuration bench.py times (1,024 sims, default SPC);
    the oracle recomputes a stratified sample of simulations one by one (sims are independent).
    Shortened in time (1 s simulated, 0.2 s discarded) so the CPU side finishes in seconds."""
    cfg = wl.config(2)
    W, L = wl.config_connectome(cfg)
    steps, discard = 10000, 2000
    conn, sw = tvbx.sweep_from_config(cfg, W, L)
    sw.run(steps, cfg["dt"], noise_on=True, ds=10, discard_steps=discard)
    fc, me, mi = sw.fc_readout()
    assert fc.shape == (1024, 68, 68) and np.isfinite(fc).all()
    sims = [0, 31, 5 * 32 + 9, 16 * 32 + 16, 1023 - 31, 1023]
    o = orc.OracleSweep(W, L, wl.grid_params(cfg, sims=sims), seed=cfg["seed"], ext_ids=sims)
    o.run(steps, cfg["dt"], noise_on=True, ds=10, discard_steps=discard)
    rfc, rme, rmi = o.fc_readout()
    assert np.abs(me[sims] / rme - 1).max() < TOL_MEAN_REL
    assert np.abs(mi[sims] / rmi - 1).max() < TOL_MEAN_REL
    assert np.abs(fc[sims] - rfc).max() < TOL_FC_ABS
    # properties that hold for every simulation at any size
    assert np.all(np.abs(fc) <= 1.0 + 1e-6)
    np.testing.assert_array_equal(fc, np.swapaxes(fc, 1, 2))
    assert (me > 0).all() and (me < 0.2).all() and (mi > 0).all() and (mi < 0.2).all()


def _sampled_parity(cfg_id, steps, discard, sims, **kw):
    """Full-size sweep of BASELINE.json configs[cfg_id - 1] in the default launch configuration (the one
    bench.py times), shortened in time; the oracle recomputes the listed simulations one by one."""
    cfg = wl.config(cfg_id)
    W, L = wl.config_connectome(cfg)
    conn, sw = tvbx.sweep_from_config(cfg, W, L, **kw)
    sw.run(steps, cfg["dt"], noise_on=True, ds=cfg["ds"], discard_steps=discard)
    fc, me, mi = sw.fc_readout()
    o = orc.OracleSweep(W, L, wl.grid_params(cfg, sims=sims), seed=cfg["seed"], ext_ids=sims)
    o.run(steps, cfg["dt"], noise_on=True, ds=cfg["ds"], discard_steps=discard)
    rfc, rme, rmi = o.fc_readout()
    assert np.isfinite(fc).all() and np.isfinite(me).all() and np.isfinite(mi).all()
    assert np.abs(me[sims] / rme - 1).max() < TOL_MEAN_REL
    assert np.abs(mi[sims] / rmi - 1).max() < TOL_MEAN_REL
    assert np.abs(fc[sims] - rfc).max() < TOL_FC_ABS
    # properties that hold for every simulation at any size
    assert np.all(np.abs(fc) <= 1.0 + 1e-6)
    np.testing.assert_array_equal(fc, np.swapaxes(fc, 1, 2))
    assert np.all(np.diagonal(fc, axis1=1, axis2=2) == 1.0)
    assert (me > 0).all() and (me < 0.2).all() and (mi > 0).all() and (mi < 0.2).all()
    return sw, o


def test_cfg3_full_size_sampled_against_oracle():
    """cfg 3 at full size (32,768 sims, 8 speeds = 8 delay tables, ring depth 16 ... 2,000 slots, chunk
    length 1 ... 8 steps); samples cover every speed and the corners of the (b_e, a_e, G) grid."""
    sims = [0, 1, 2, 3, 4, 5, 6, 7, 8 * 137 + 3, 8 * 2222 + 6, 32767 - 7, 32767]
    sw, o = _sampled_parity(3, 3000, 1000, sims)
    assert sw.n_sims == 32768
    for loc in (0, 3, 7):
        assert sw.ring_len(loc)[0] == o.ring_len(loc)


def test_cfg5_full_size_sampled_against_oracle():
    """cfg 5 at full size (4,096 sims x 360 regions, ~180 edges per row, delay table read through L1/L2)."""
    sw, o = _sampled_parity(5, 1500, 500, [0, 63, 64 * 31 + 17, 4095])
    assert sw.n_sims == 4096 and sw.n_regions == 360


def test_cfg4_streaming_fc_drift_against_oracle():
    """cfg 4 (256 sims, tau_w_e = 500 ms): the FC is accumulated in Welford/Chan form over 1-ms samples,
    chunk after chunk (here 20 s simulated = 19,000 kept samples = 5 chunk merges); the first and the
    last simulation of the grid are checked for drift against the oracle's two-pass FC."""
    sw, o = _sampled_parity(4, 200000, 10000, [0, 255])
    assert sw.samples_kept() == 19000 and sw.launch_info()["chunk_samples"] < 19000


# ------------------------------------------------------------------------------------ S7': FC on the tensor cores
# TF32 keeps 11 significant bits: each centred sample carries a relative rounding error <= 2^-11, each product
# <= 2^-10, so |dM_kl| <= 2^-10 sum_q |x_qk x_ql| <= 2^-10 sqrt(M_kk M_ll) (Cauchy-Schwarz) and the Pearson entry
# moves by at most ~2^-10 from the products plus ~2^-10 |FC| from the two variances: 2e-3 in the worst case,
# far inside the 0.02 of the north star.
TOL_FC_TF32_VS_FP32 = 2e-3


@pytest.mark.parametrize("N,spc,clu,chunk,steps", [
    (68, 0, 0, 0, 3000),       # cfg-1 connectome, one chunk, one 128-row block, n_c = 280 (not a multiple of 32)
    (23, 3, 1, 37, 2400),      # odd N (scalar FP64 merge), several ragged chunks: Chan merge term
    (130, 2, 1, 64, 1500),     # two row blocks, the second with 2 live rows
    (360, 4, 3, 50, 1200),     # cfg-5 size: three row blocks, N extent split 256 + 112, cluster integrator
], ids=["n68", "n23_odd", "n130", "n360"])
def test_fc_tensor_core_path_matches_fp32_tiles_and_oracle(N, spc, clu, chunk, steps):
    if N == 68:
        cfg = wl.config(1); W, L = wl.config_connectome(cfg); sims = None
    elif N == 360:
        cfg = wl.config(5); W, L = wl.config_connectome(cfg); sims = [5, 1000, 2047, 4095, 77]
    else:
        W, L = wl.connectome(N, seed=N, keep=0.4); sims = None
        cfg = dict(axes=[dict(name="G", lo=0.0, hi=0.4, n=5, values=None)], fixed=dict(v=4.0, b_e=20.0, wNoise=1e-4), seed=9)
    kw = dict(sims_per_cta=spc, ctas_per_group=clu, chunk_samples=chunk, sim_ids=sims)
    out = {}
    for mode in (tvbx.TVBX_FC_TF32, tvbx.TVBX_FC_FP32):
        _, sw = tvbx.sweep_from_config(cfg, W, L, fc_mode=mode, **kw)
        sw.run(steps, 0.1, noise_on=True, ds=10, discard_steps=200)
        out[mode] = sw.fc_readout()
        assert sw.fc_kernel_name() == ("tvbx::fc_xtx_tc_kernel" if mode == tvbx.TVBX_FC_TF32 else "tvbx::fc_comoment_kernel")
    fc_t, me_t, mi_t = out[tvbx.TVBX_FC_TF32]
    fc_f, me_f, mi_f = out[tvbx.TVBX_FC_FP32]
    np.testing.assert_array_equal(me_t, me_f); np.testing.assert_array_equal(mi_t, mi_f)   # same integrator
    assert np.isfinite(fc_t).all()
    assert np.abs(fc_t - fc_f).max() < TOL_FC_TF32_VS_FP32
    np.testing.assert_array_equal(fc_t, np.swapaxes(fc_t, 1, 2))
    assert np.all(np.diagonal(fc_t, axis1=1, axis2=2) == 1.0)
    o = orc.OracleSweep(W, L, wl.grid_params(cfg, sims=sims), seed=cfg["seed"], ext_ids=sims)
    o.run(steps, 0.1, noise_on=True, ds=10, discard_steps=200)
    rfc, rme, rmi = o.fc_readout()
    assert np.abs(fc_t - rfc).max() < TOL_FC_ABS
    # readout is repeatable (the open chunk is merged into a scratch copy)
    np.testing.assert_array_equal(sw.fc_readout()[0], fc_f)


def test_fc_mode_default_and_errors():
    W, L = wl.connectome(20, seed=7, keep=0.4)
    cfg = dict(axes=[], fixed=dict(v=4.0), seed=1)
    _, sw = tvbx.sweep_from_config(cfg, W, L)
    assert sw.fc_kernel_name() == "tvbx::fc_xtx_tc_kernel"            # FP32 sweep, N <= 512: tensor cores
    _, sw64 = tvbx.sweep_from_config(cfg, W, L, precision=tvbx.TVBX_F64)
    assert sw64.fc_kernel_name() == "tvbx::fc_comoment_kernel"        # FP64 build mode keeps FP64 tiles
    with pytest.raises(tvbx.TvbxError):
        tvbx.sweep_from_config(cfg, W, L, precision=tvbx.TVBX_F64, fc_mode=tvbx.TVBX_FC_TF32)


# ------------------------------------------------------------------------------------ f3: FC scores
# Tolerance: the scores are Pearson coefficients / means of FC entries; an FC entry may differ from the oracle's by
# TOL_FC_ABS (noise-on runs, FP32 integrator), and a perturbation of that size on entries whose spread is O(0.1-1)
# moves a correlation by the same order at most -- the same absolute 0.02 is used; observed differences ~1e-4.
@pytest.mark.parametrize("N,kw", [(68, dict()), (23, dict(sims_per_cta=3, chunk_samples=37)),
                                  (360, dict(sims_per_cta=4, ctas_per_group=3))], ids=["n68", "n23", "n360"])
def test_fc_scores_match_the_oracle(N, kw):
    from oracle import fc_scores as ofs
    if N == 68:
        cfg = wl.config(1); W, L = wl.config_connectome(cfg); sims = None
    elif N == 360:
        cfg = wl.config(5); W, L = wl.config_connectome(cfg); sims = [5, 2047, 4095]
    else:
        W, L = wl.connectome(N, seed=N, keep=0.4); sims = None
        cfg = dict(axes=[dict(name="G", lo=0.0, hi=0.4, n=5, values=None)], fixed=dict(v=4.0, b_e=20.0, wNoise=1e-4), seed=9)
    steps = 2400 if N != 360 else 1200
    _, sw = tvbx.sweep_from_config(cfg, W, L, sim_ids=sims, **kw)
    sw.run(steps, 0.1, noise_on=True, ds=10, discard_steps=200)
    o = orc.OracleSweep(W, L, wl.grid_params(cfg, sims=sims), seed=cfg["seed"], ext_ids=sims)
    o.run(steps, 0.1, noise_on=True, ds=10, discard_steps=200)
    rfc = o.fc_readout()[0]
    ref = rfc[0] + 0.05 * np.random.default_rng(0).standard_normal(rfc[0].shape)     # an "external" FC
    ref = 0.5 * (ref + ref.T)
    want = ofs.fc_scores(rfc, W, ref)
    got = sw.fc_scores(ref_fc=ref)
    for k in ("fcsc", "fitness", "mean_fc"):
        assert got[k].shape == (sw.n_sims,) and np.isfinite(got[k]).all()
        assert np.abs(got[k] - np.asarray(want[k])).max() < TOL_FC_ABS, k
    # the same numbers from the FC matrix the library returns (rounded to float32: with G = 0 the entries spread by
    # only ~1e-2, so 6e-8 of rounding shows up as ~1e-5 in a correlation) through the oracle's definition
    own = ofs.fc_scores(sw.fc_readout()[0].astype(np.float64), W, ref)
    for k in ("fcsc", "fitness", "mean_fc"):
        np.testing.assert_allclose(got[k], own[k], atol=5e-5)
    # device outputs, no reference; repeatable; accumulators untouched
    import torch
    dev = sw.fc_scores(device=True)
    torch.cuda.synchronize()
    assert set(dev) == {"fcsc", "mean_fc"}
    np.testing.assert_array_equal(dev["fcsc"].cpu().numpy(), got["fcsc"])
    np.testing.assert_array_equal(sw.fc_scores(ref_fc=ref)["fitness"], got["fitness"])


def test_fc_scores_errors_and_degenerate():
    W, L = wl.connectome(12, seed=1, keep=0.5)
    cfg = dict(axes=[], fixed=dict(v=4.0), seed=1)
    _, sw = tvbx.sweep_from_config(cfg, W, L)
    with pytest.raises(tvbx.TvbxError):
        sw.fc_scores()                                   # no run yet
    sw.run(300, 0.1, noise_on=False, ds=10)              # noise off, identical start: series are smooth, FC defined
    bad = np.full((12, 12), np.nan)
    with pytest.raises(tvbx.TvbxError):
        sw.fc_scores(ref_fc=bad)
    const = sw.fc_scores(ref_fc=np.full((12, 12), 0.5))
    assert const["fitness"][0] == 0.0                    # zero-variance reference -> 0 (A18 / A23)


# ------------------------------------------------------------------------------------ more edge cases
@pytest.mark.parametrize("v", [30.0, 120.0], ids=["ch2", "ch1"])
def test_short_delay_classes_ring_in_shared_memory(v):
    """Minimum delays of a few steps: 2-slot gather instances with the history ring staged in shared memory
    (SRING).  Parity with the oracle with and without noise, and run(a); run(b) == run(a + b) bit for bit --
    the ring must survive the copy back to global memory between launches."""
    W, L = wl.connectome(40, seed=12, keep=0.4)
    cfg = dict(axes=[dict(name="G", lo=0.1, hi=0.5, n=5, values=None)], fixed=dict(v=v, b_e=40.0, wNoise=1e-4), seed=6)
    sw, traj, o, ref = run_pair(cfg, W, L, 900, True, traj_steps=900, discard=100)
    assert sw.kernel_name() == "tvbx::integrate2_kernel" and sw.ring_len(0)[0] <= 80
    assert traj_err(traj, ref) < 5e-3          # same Philox stream; FP32 rounding amplified by the noise path
    fc, me, mi = sw.fc_readout(); rfc, rme, rmi = o.fc_readout()
    assert np.abs(me / rme - 1).max() < TOL_MEAN_REL and np.abs(fc - rfc).max() < TOL_FC_ABS
    sw2, traj2, o2, ref2 = run_pair(cfg, W, L, 900, False, traj_steps=900)
    assert traj_err(traj2, ref2) < TOL_TRAJ_F32
    _, a = tvbx.sweep_from_config(cfg, W, L, chunk_samples=16)
    _, b = tvbx.sweep_from_config(cfg, W, L, chunk_samples=16)
    a.run(703, 0.1, noise_on=True, ds=10, discard_steps=95)
    for part in (1, 298, 7, 397):
        b.run(part, 0.1, noise_on=True, ds=10, discard_steps=95)
    ya, oa = a.state(); yb, ob = b.state()
    np.testing.assert_array_equal(ya, yb); np.testing.assert_array_equal(oa, ob)
    for x, y in zip(a.fc_readout(), b.fc_readout()):
        np.testing.assert_array_equal(x, y)


def test_single_region_and_rows_without_edges():
    """N = 1 (no edge at all) and a connectome in which some regions receive nothing: the coupling sum is 0 there."""
    cfg = dict(axes=[dict(name="b_e", lo=0.0, hi=60.0, n=3, values=None)], fixed=dict(G=0.4, v=4.0), seed=2)
    W1, L1 = np.zeros((1, 1)), np.zeros((1, 1))
    sw, traj, o, ref = run_pair(cfg, W1, L1, 500, False, traj_steps=500)
    assert traj.shape == (3, 500, 7, 1) and traj_err(traj, ref) < TOL_TRAJ_F32
    W, L = wl.connectome(9, seed=4, keep=0.5)
    W[2, :] = 0.0; W[7, :] = 0.0                  # regions 2 and 7 have no incoming edge (W need not be symmetric)
    sw, traj, o, ref = run_pair(cfg, W, L, 500, True, traj_steps=500, discard=100, params=dict(wNoise=1e-4))
    assert traj_err(traj, ref) < 5e-3
    fc, me, mi = sw.fc_readout(); rfc, rme, rmi = o.fc_readout()
    assert np.abs(fc - rfc).max() < TOL_FC_ABS


def test_zero_steps_and_memory_pool():
    W, L = wl.connectome(16, seed=3, keep=0.5)
    cfg = dict(axes=[dict(name="G", lo=0.0, hi=0.3, n=4, values=None)], fixed=dict(v=4.0, wNoise=1e-4), seed=5)
    tvbx.trim_memory()
    _, a = tvbx.sweep_from_config(cfg, W, L)
    a.run(0, 0.1, noise_on=True, ds=10)           # allocates, advances nothing
    assert a.steps_done() == 0 and a.samples_kept() == 0
    a.run(400, 0.1, noise_on=True, ds=10)
    ra = a.fc_readout()
    a.close()
    freed_probe = tvbx.trim_memory()
    assert freed_probe > 0                        # the destroyed sweep's buffers were waiting in the pool
    _, b = tvbx.sweep_from_config(cfg, W, L)      # fresh buffers
    b.run(400, 0.1, noise_on=True, ds=10)
    rb = b.fc_readout()
    b.close()
    _, c = tvbx.sweep_from_config(cfg, W, L)      # recycled buffers: same results, no stale state
    c.run(400, 0.1, noise_on=True, ds=10)
    rc = c.fc_readout()
    for x, y, z in zip(ra, rb, rc):
        np.testing.assert_array_equal(x, y); np.testing.assert_array_equal(y, z)
    c.close()
    assert tvbx.trim_memory() > 0 and tvbx.trim_memory() == 0


# ------------------------------------------------------------------------------------ f4: rate statistics
@pytest.mark.parametrize("N,kw,thr", [(68, dict(), 0.0), (23, dict(sims_per_cta=3, chunk_samples=37), 4.5e-4),
                                      (130, dict(sims_per_cta=2, chunk_samples=64, fc_mode=1), 4.5e-4)], ids=["n68", "n23", "n130"])
def test_rate_stats_match_the_oracle(N, kw, thr):
    """Variance, maximum and above-threshold count of the kept excitatory 1-ms samples (tvbx_rate_stats) against
    oracle/rate_stats.py on the oracle's own samples.  Variance: relative 2e-2 (it is M_kk / n, the quantity the
    FC tolerance is about); maximum: the 1 % of the mean rates; count: the threshold is put where the oracle's
    samples leave a margin of 2 %, so both sides must count the same samples exactly."""
    from oracle import rate_stats as ors
    if N == 68:
        cfg = wl.config(1); W, L = wl.config_connectome(cfg)
    else:
        W, L = wl.connectome(N, seed=N, keep=0.4)
        cfg = dict(axes=[dict(name="G", lo=0.0, hi=0.4, n=5, values=None)], fixed=dict(v=4.0, b_e=20.0, wNoise=1e-4), seed=9)
    steps = 2400
    o = orc.OracleSweep(W, L, wl.grid_params(cfg), seed=cfg["seed"])
    o.run(steps, 0.1, noise_on=True, ds=10, discard_steps=200)
    xs = [o.samples(s)[0] for s in range(o.S)]
    if thr == 0.0:                                  # default threshold 0.1 kHz: nothing exceeds it here
        thr_used = 0.1
    else:                                           # a threshold inside the data, moved away from any sample by 2 %
        allx = np.sort(np.concatenate([x.ravel() for x in xs]))
        gaps = np.where((allx[1:] / allx[:-1] > 1.05) & (allx[:-1] > np.quantile(allx, 0.2)) & (allx[1:] < np.quantile(allx, 0.9)))[0]
        thr_used = float(np.sqrt(allx[gaps[0]] * allx[gaps[0] + 1])) if len(gaps) else float(allx[-1] * 2)
    _, sw = tvbx.sweep_from_config(cfg, W, L, rate_threshold_khz=(0.0 if thr == 0.0 else thr_used), **kw)
    sw.run(steps, 0.1, noise_on=True, ds=10, discard_steps=200)
    var, mx, ab = sw.rate_stats()
    assert var.shape == mx.shape == ab.shape == (sw.n_sims, N) and ab.dtype == np.int32
    for s in range(sw.n_sims):
        rv, rm, ra = ors.rate_stats(xs[s], thr_used)
        np.testing.assert_allclose(var[s], rv, rtol=2e-2, atol=1e-14)
        np.testing.assert_allclose(mx[s], rm, rtol=TOL_MEAN_REL)
        np.testing.assert_array_equal(ab[s], ra)
    # consistent with the FC accumulators, repeatable, device outputs
    import torch
    dv, dm, da = sw.rate_stats(device=True)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(dv.cpu().numpy(), var); np.testing.assert_array_equal(da.cpu().numpy(), ab)
    sw.run(100, 0.1, noise_on=True, ds=10, discard_steps=200)          # streaming: counts never decrease, max never drops
    var2, mx2, ab2 = sw.rate_stats()
    assert np.all(ab2 >= ab) and np.all(mx2 >= mx)


def test_rate_stats_before_any_sample_is_an_error():
    W, L = wl.connectome(12, seed=2, keep=0.5)
    _, sw = tvbx.sweep_from_config(dict(axes=[], fixed={}, seed=0), W, L)
    sw.run(5, 0.1, ds=10)
    with pytest.raises(tvbx.TvbxError):
        sw.rate_stats()
    with pytest.raises(tvbx.TvbxError):
        tvbx.sweep_from_config(dict(axes=[], fixed={}, seed=0), W, L, rate_threshold_khz=-1.0)


def test_more_regions_than_one_cta_falls_back_to_the_general_kernel():
    """N > 480: the general integrator (several passes over the regions) and the FP32 register-tile X^T X (the tcgen05
    kernel serves N <= 384); fc_mode = TVBX_FC_TF32 is refused."""
    N = 520
    W, L = wl.connectome(N, seed=21, keep=0.05)
    cfg = dict(axes=[dict(name="G", lo=0.1, hi=0.3, n=2, values=None)], fixed=dict(v=6.0, b_e=30.0, wNoise=1e-4), seed=8)
    sw, traj, o, ref = run_pair(cfg, W, L, 600, True, traj_steps=600, discard=100)
    assert sw.kernel_name() == "tvbx::integrate_kernel" and sw.fc_kernel_name() == "tvbx::fc_comoment_kernel"
    assert traj_err(traj, ref) < 5e-3
    fc, me, mi = sw.fc_readout(); rfc, rme, rmi = o.fc_readout()
    assert np.abs(me / rme - 1).max() < TOL_MEAN_REL and np.abs(fc - rfc).max() < TOL_FC_ABS
    with pytest.raises(tvbx.TvbxError):
        tvbx.sweep_from_config(cfg, W, L, fc_mode=tvbx.TVBX_FC_TF32)


@pytest.mark.parametrize("kw", [dict(chunk_samples=37), dict(chunk_samples=50, sims_per_cta=4),
                                dict(chunk_samples=64, precision=tvbx.TVBX_F64)], ids=["fp32", "fp32_spc4", "fp64"])
def test_rate_stats_inhibitory_population(kw):
    """rate_stats_inhibitory: the inhibitory 1-ms samples are kept as well and reduced by one Welford/Chan pass per
    chunk; variance, maximum and count of both populations against oracle/rate_stats.py on the oracle's samples."""
    from oracle import rate_stats as ors
    N = 24
    W, L = wl.connectome(N, seed=5, keep=0.4)
    cfg = dict(axes=[dict(name="G", lo=0.0, hi=0.4, n=4, values=None)], fixed=dict(v=4.0, b_e=20.0, wNoise=1e-4), seed=11)
    steps = 2400
    o = orc.OracleSweep(W, L, wl.grid_params(cfg), seed=cfg["seed"])
    o.run(steps, 0.1, noise_on=True, ds=10, discard_steps=200)
    xs = [o.samples(s) for s in range(o.S)]
    thr = float(np.median(np.concatenate([x[1].ravel() for x in xs])))     # inside the inhibitory data
    thr = thr * 1.0000001
    _, sw = tvbx.sweep_from_config(cfg, W, L, rate_stats_inhibitory=True, rate_threshold_khz=thr, **kw)
    sw.run(steps, 0.1, noise_on=True, ds=10, discard_steps=200)
    # FP32: a compile-time instance of the packed kernel stores the inhibitory samples too; FP64 mode: the general kernel
    assert sw.kernel_name() == ("tvbx::integrate_kernel" if kw.get("precision") == tvbx.TVBX_F64 else "tvbx::integrate2_kernel")
    var_e, max_e, ab_e, var_i, max_i, ab_i = sw.rate_stats()
    fp64 = kw.get("precision") == tvbx.TVBX_F64
    n = xs[0][0].shape[0]
    for s in range(sw.n_sims):
        for pop, (var, mx, ab) in enumerate([(var_e, max_e, ab_e), (var_i, max_i, ab_i)]):
            rv, rm, ra = ors.rate_stats(xs[s][pop], thr)
            np.testing.assert_allclose(var[s], rv, rtol=1e-5 if fp64 else 2e-2, atol=1e-14)
            np.testing.assert_allclose(mx[s], rm, rtol=1e-6 if fp64 else TOL_MEAN_REL)
            if fp64:
                np.testing.assert_array_equal(ab[s], ra)
            else:      # FP32 trajectories: samples within 1 % of the threshold may fall on either side
                x = np.asarray(xs[s][pop])
                slack = ((x > thr * 0.99) & (x < thr * 1.01)).sum(axis=0)
                assert np.all(np.abs(ab[s] - np.asarray(ra)) <= slack)
    assert np.all((ab_i >= 0) & (ab_i <= n)) and ab_i.sum() > 0
    # a short minimum delay (chunks of < 8 steps) has no inhibitory-sample instance of the packed kernel: general kernel
    _, sw3 = tvbx.sweep_from_config(cfg, W, L, rate_stats_inhibitory=True, params=dict(v=60.0))
    sw3.run(300, 0.1, noise_on=True, ds=10)
    assert sw3.kernel_name() == "tvbx::integrate_kernel" and len(sw3.rate_stats()) == 6
    # without the option the inhibitory outputs are refused
    _, sw2 = tvbx.sweep_from_config(cfg, W, L)
    sw2.run(100, 0.1, noise_on=True, ds=10)
    assert len(sw2.rate_stats()) == 3
    import ctypes as C
    buf = np.empty((sw2.n_sims, N), np.float32)
    rc = tvbx.lib().tvbx_rate_stats(sw2._h, None, None, None, buf.ctypes.data, None, None, 0, None)
    assert rc == -1        # TVBX_EINVAL

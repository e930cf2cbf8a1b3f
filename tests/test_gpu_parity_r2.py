"""GPU parity, round-2 additions: trajectories in which the SECOND-ORDER terms of Eq. (1) carry weight, the
tensor-core FC size limit, two live sweeps that share kernel instances, and a stress of the rolling chunk pipeline."""
import numpy as np
import pytest

import workloads as wl
import paper_2311_13337_b200 as tvbx
from oracle import oracle as orc
from tests.test_gpu_parity import traj_err, run_pair, TOL_TRAJ_F32, TOL_TRAJ_F64, TOL_MEAN_REL, TOL_FC_ABS

pytestmark = pytest.mark.gpu


def _second_order_weight(cfg, W, ref, kappa, step):
    """|1/2 C_ee F_ee + C_ei F_ei + 1/2 C_ii F_ii| kappa^2 relative to |nu|, from the ORACLE's state and the oracle's
    transfer function (coupling input neglected: an estimate of the weight, not a parity quantity)."""
    P = wl.grid_params(cfg)
    names = wl.PARAM_NAMES
    out = []
    for s in range(ref.shape[0]):
        for k in (0, ref.shape[3] // 2):
            E, I, Cee, Cei, Cii, We, Wi = ref[s, step, :, k]
            p = P[s].copy(); p[names.index("kappa")] = kappa
            for pop, Wm, ce, ci, nu in ((0, We, p[names.index("c_Fee")], p[names.index("c_Fei")], E),
                                        (1, Wi, p[names.index("c_Fie")], p[names.index("c_Fii")], I)):
                F, _ = orc.tf(p, pop, E + ce, I + ci, Wm)
                out.append(abs(0.5 * Cee * F[3] + Cei * F[4] + 0.5 * Cii * F[5]) * kappa * kappa / abs(nu))
    return float(np.median(out))


@pytest.mark.parametrize("kappa,steps", [(0.2, 600), (0.3, 600), (1.0, 12)], ids=["k0.2", "k0.3", "k1_12steps"])
def test_second_order_terms_carry_weight(kappa, steps):
    """cfg 1, noise off, packed FP32 kernel at 1e-3 and FP64 mode at 1e-9 with kappa (A22) large enough that the
    second-derivative terms of Eq. (1) are >= 10 % of the rates: an error in F_ee / F_ei / F_ii of tf_closed2 moves
    these trajectories far beyond the tolerance.  kappa = 0.2 / 0.3: 60 ms (the oracle's sensitivity to a 1e-7 relative
    perturbation of the initial state stays <= 20x over this horizon, so 1e-3 is a meaningful FP32 bound).  kappa = 1,
    the unit-consistent variant: the second-order terms are ~100x the rates at step 0 and the dynamics turn chaotic
    after ~20 steps (oracle: a 1e-7 perturbation grows 3e2-fold by step 20 and 6e5-fold by step 30), so parity is a
    well-posed question over the first 12 steps only."""
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    par = dict(kappa=kappa)
    sw, traj, o, ref = run_pair(cfg, W, L, steps, False, traj_steps=steps, params=par)
    assert sw.kernel_name() == "tvbx::integrate2_kernel"
    weight = _second_order_weight(cfg, W, ref, kappa, min(steps - 1, 50))
    assert weight >= 0.10, weight
    assert traj_err(traj, ref) < TOL_TRAJ_F32
    sw, traj, o, ref = run_pair(cfg, W, L, steps, False, traj_steps=steps, params=par, precision=tvbx.TVBX_F64)
    assert traj_err(traj, ref) < TOL_TRAJ_F64


def test_second_order_weight_with_noise_and_all_parameters():
    """kappa = 0.25 with noise on (same Philox stream), non-default a, b, E_L, c_F and coupling, 40 ms."""
    W, L = wl.connectome(24, seed=13, keep=0.4)
    cfg = dict(axes=[dict(name="b_e", lo=0.0, hi=60.0, n=3, values=None)],
               fixed=dict(v=5.0, G=0.3, wNoise=1e-5, kappa=0.25, a_e=4.0, a_i=1.0, b_i=2.0, E_L_e=-63.0, E_L_i=-65.0,
                          c_Fie=0.5e-3, c_Fei=0.1e-3, c_Fii=0.2e-3), seed=8)
    sw, traj, o, ref = run_pair(cfg, W, L, 400, True, traj_steps=400)
    assert sw.kernel_name() == "tvbx::integrate2_kernel"
    assert traj_err(traj, ref) < TOL_TRAJ_F32
    sw, traj, o, ref = run_pair(cfg, W, L, 400, True, traj_steps=400, precision=tvbx.TVBX_F64)
    assert traj_err(traj, ref) < 1e-8


# ------------------------------------------------------------------------------------ FC size limit of the tensor-core path
def test_fc_between_384_and_512_regions_uses_register_tiles():
    """N = 400: the tcgen05 X^T X stages N (rounded up to 128) rows x 32 samples x 4 stages in shared memory -- 262 KB at
    512 rows, more than an SM has -- so TVBX_FC_AUTO must pick the register-tile kernel above N = 384, and an explicit
    TVBX_FC_TF32 is refused at tvbx_sweep_create."""
    N = 400
    W, L = wl.connectome(N, seed=22, keep=0.05)
    cfg = dict(axes=[dict(name="G", lo=0.1, hi=0.3, n=2, values=None)], fixed=dict(v=6.0, b_e=30.0, wNoise=1e-4), seed=8)
    sw, traj, o, ref = run_pair(cfg, W, L, 600, True, traj_steps=600, discard=100, chunk_samples=20)
    assert sw.kernel_name() == "tvbx::integrate2_kernel" and sw.fc_kernel_name() == "tvbx::fc_comoment_kernel"
    assert traj_err(traj, ref) < 5e-3          # (noise-on extra: same Philox stream, FP32 rounding through the noise path)
    fc, me, mi = sw.fc_readout(); rfc, rme, rmi = o.fc_readout()
    assert np.abs(me / rme - 1).max() < TOL_MEAN_REL and np.abs(fc - rfc).max() < TOL_FC_ABS
    with pytest.raises(tvbx.TvbxError):
        tvbx.sweep_from_config(cfg, W, L, fc_mode=tvbx.TVBX_FC_TF32)
    # the largest size the tensor-core path serves
    W2, L2 = wl.connectome(384, seed=23, keep=0.05)
    _, sw2 = tvbx.sweep_from_config(cfg, W2, L2, chunk_samples=20)
    sw2.run(600, 0.1, noise_on=True, ds=10, discard_steps=100)
    assert sw2.fc_kernel_name() == "tvbx::fc_xtx_tc_kernel"
    fc2 = sw2.fc_readout()[0]
    o2 = orc.OracleSweep(W2, L2, wl.grid_params(cfg), seed=cfg["seed"])
    o2.run(600, 0.1, noise_on=True, ds=10, discard_steps=100)
    assert np.abs(fc2 - o2.fc_readout()[0]).max() < TOL_FC_ABS


def test_two_live_sweeps_of_different_size_interleaved():
    """The dynamic-shared-memory limit is an attribute of the kernel FUNCTION, process-wide: a sweep with N = 360 (197 KB
    for fc_xtx_tc_kernel) and one with N = 68 share that function.  Interleaved runs must not lower each other's limit."""
    cfg5 = wl.config(5); W5, L5 = wl.config_connectome(cfg5)
    cfg1 = wl.config(1); W1, L1 = wl.config_connectome(cfg1)
    sims5 = [3, 4000]
    _, a = tvbx.sweep_from_config(cfg5, W5, L5, sim_ids=sims5, chunk_samples=16)
    _, b = tvbx.sweep_from_config(cfg1, W1, L1, chunk_samples=16)
    _, a_ref = tvbx.sweep_from_config(cfg5, W5, L5, sim_ids=sims5, chunk_samples=16)
    _, b_ref = tvbx.sweep_from_config(cfg1, W1, L1, chunk_samples=16)
    for _ in range(3):                          # every run fills chunks: FC kernels of both sizes alternate
        a.run(400, 0.1, noise_on=True, ds=10)
        b.run(400, 0.1, noise_on=True, ds=10)
    a_ref.run(1200, 0.1, noise_on=True, ds=10)
    b_ref.run(1200, 0.1, noise_on=True, ds=10)
    for x, y in zip(a.fc_readout(), a_ref.fc_readout()):
        np.testing.assert_array_equal(x, y)
    for x, y in zip(b.fc_readout(), b_ref.fc_readout()):
        np.testing.assert_array_equal(x, y)
    # the general kernel (FP64 mode) with two sizes as well
    W2, L2 = wl.connectome(90, seed=3, keep=0.3)
    cfgs = dict(axes=[dict(name="G", lo=0.0, hi=0.3, n=2, values=None)], fixed=dict(v=4.0, wNoise=1e-4), seed=2)
    _, c = tvbx.sweep_from_config(cfgs, W2, L2, precision=tvbx.TVBX_F64)
    _, d = tvbx.sweep_from_config(cfgs, W1[:20, :20].copy(), L1[:20, :20].copy(), precision=tvbx.TVBX_F64)
    c.run(100, 0.1, noise_on=True, ds=10); d.run(100, 0.1, noise_on=True, ds=10); c.run(100, 0.1, noise_on=True, ds=10)
    assert c.steps_done() == 200 and d.steps_done() == 100


# ------------------------------------------------------------------------------------ rolling chunk pipeline under stress
@pytest.mark.parametrize("lmin,lmax,v", [(32.0, 60.0, 10.0), (1.0, 9.0, 5.0), (3.0, 40.0, 10.0)], ids=["lag4_ch8", "ch1_lag3", "ch2"])
def test_chunk_pipeline_results_do_not_depend_on_the_mapping(lmin, lmax, v):
    """integrate2_kernel has no CTA barrier: warps hand chunks over through a ring of mbarriers and may run up to LAG
    chunks apart.  If a warp ever read a ring slot before its writer had stored it (or after it was overwritten), the
    result would depend on warp timing.  Same simulations, odd N = 37, noise on, 6,000 steps (750 ... 6,000 chunks), under
    mappings with very different warp counts and timing -- 1, 3 and 8 simulations per CTA, one CTA or a 4-CTA cluster
    (scalar gather: per-node arithmetic identical) -- must agree BIT FOR BIT, twice in a row, and match the oracle.
    lag4_ch8: minimum delay 32 steps -> chunks of 8, run-ahead limit LAG = 4; ch1_lag3: minimum delay 2 -> one-step
    chunks, LAG = 3 (ring in shared memory); ch2: chunks of 2."""
    N = 37
    W, _ = wl.connectome(N, seed=5, keep=0.35)
    rng = np.random.default_rng(11)
    Lu = rng.uniform(lmin, lmax, (N, N)); L = np.triu(Lu, 1) + np.triu(Lu, 1).T
    cfg = dict(axes=[dict(name="G", lo=0.05, hi=0.4, n=8, values=None)], fixed=dict(v=v, b_e=20.0, wNoise=1e-4), seed=9)
    steps = 6000
    outs = []
    for kw in (dict(sims_per_cta=1), dict(sims_per_cta=3), dict(sims_per_cta=8), dict(sims_per_cta=3),
               dict(sims_per_cta=2, ctas_per_group=4)):
        _, sw = tvbx.sweep_from_config(cfg, W, L, chunk_samples=64, **kw)
        sw.run(steps, 0.1, noise_on=True, ds=10, discard_steps=1000)
        assert sw.kernel_name() == "tvbx::integrate2_kernel"
        y, ou = sw.state()
        outs.append((y, ou, sw.fc_readout()[1]))
    for y, ou, me in outs[1:]:
        np.testing.assert_array_equal(y, outs[0][0]); np.testing.assert_array_equal(ou, outs[0][1])
        np.testing.assert_array_equal(me, outs[0][2])
    # and under different co-scheduling: two sweeps running concurrently on two streams perturb each other's warp timing
    import torch
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    _, a = tvbx.sweep_from_config(cfg, W, L, chunk_samples=64, sims_per_cta=3)
    _, b = tvbx.sweep_from_config(cfg, W, L, chunk_samples=64, sims_per_cta=1)
    for part in (2500, 3500):
        a.run(part, 0.1, noise_on=True, ds=10, discard_steps=1000, stream=s1)
        b.run(part, 0.1, noise_on=True, ds=10, discard_steps=1000, stream=s2)
    torch.cuda.synchronize()
    for sw in (a, b):
        y, ou = sw.state()
        np.testing.assert_array_equal(y, outs[0][0]); np.testing.assert_array_equal(ou, outs[0][1])
    o = orc.OracleSweep(W, L, wl.grid_params(cfg), seed=cfg["seed"])
    o.run(steps, 0.1, noise_on=True, ds=10, discard_steps=1000)
    rfc, rme, rmi = o.fc_readout()
    assert np.abs(outs[0][2] / rme - 1).max() < TOL_MEAN_REL


# ------------------------------------------------------------------------------------ f1: the low-latency warp-pair form
@pytest.mark.parametrize("N,n_sims,spc,v", [(68, 8, 1, 4.0), (68, 6, 2, 4.0), (23, 5, 5, 3.0), (37, 7, 3, 5.0)],
                         ids=["cfg1_shape", "cfg4_shape", "n23_spc5", "n37_spc3"])
def test_latency_form_is_bitwise_the_throughput_form(N, n_sims, spc, v):
    """tvbx_sweep_opts.latency_form: producer / consumer warp pairs (csrc/tvbx_integrate2_ws.cuh) take the delayed gather
    and the Philox draws off the consumer's dependency chain.  Same arithmetic, same association of the coupling sum, same
    Philox stream: trajectories, OU state, FC and means must equal those of the one-warp form BIT FOR BIT, across several
    launches (resume), with the ring in global or in shared memory; and both match the oracle."""
    W, L = (wl.config_connectome(wl.config(1)) if N == 68 else wl.connectome(N, seed=N, keep=0.4))
    cfg = dict(axes=[dict(name="G", lo=0.0, hi=0.4, n=n_sims, values=None)], fixed=dict(v=v, b_e=30.0, wNoise=1e-4), seed=12)
    outs = {}
    for form in (1, 2):
        _, sw = tvbx.sweep_from_config(cfg, W, L, sims_per_cta=spc, latency_form=form, chunk_samples=40)
        tr = [sw.run(part, 0.1, noise_on=True, ds=10, discard_steps=100, traj_steps=part) for part in (403, 1, 996)]
        assert sw.launch_info()["latency_form"] == form and sw.kernel_name() == "tvbx::integrate2_kernel"
        outs[form] = (np.concatenate(tr, axis=1), sw.state(), sw.fc_readout())
    np.testing.assert_array_equal(outs[1][0], outs[2][0])
    for a, b in zip(outs[1][1] + outs[1][2], outs[2][1] + outs[2][2]):
        np.testing.assert_array_equal(a, b)
    o = orc.OracleSweep(W, L, wl.grid_params(cfg), seed=cfg["seed"])
    ref = o.run(1400, 0.1, noise_on=True, ds=10, discard_steps=100, traj_steps=1400)
    assert traj_err(outs[2][0], ref) < 5e-3            # (noise-on extra: same Philox stream)
    rfc, rme, rmi = o.fc_readout()
    assert np.abs(outs[2][2][1] / rme - 1).max() < TOL_MEAN_REL and np.abs(outs[2][2][0] - rfc).max() < TOL_FC_ABS


@pytest.mark.parametrize("N,n_sims,spc,clu,v", [(68, 14, 7, 4, 4.0), (68, 9, 3, 2, 4.0), (37, 5, 3, 2, 5.0), (23, 11, 8, 3, 3.0)],
                         ids=["cfg4_mapping", "n68_3x2", "n37_3x2", "n23_8x3"])
def test_grouped_latency_form_is_bitwise_the_throughput_form(N, n_sims, spc, clu, v):
    """latency_form = 3: the regions of a group of simulations split over several CTAs on different SMs (cooperative launch),
    chunk hand-over through release / acquire counters in global memory, ring loads through L2.  Trajectories, state, FC and
    means must equal those of the one-warp form BIT FOR BIT across several launches (the counters are re-armed per launch),
    including a last group with padding lanes and a last CTA with fewer regions."""
    W, L = (wl.config_connectome(wl.config(1)) if N == 68 else wl.connectome(N, seed=N, keep=0.4))
    cfg = dict(axes=[dict(name="G", lo=0.0, hi=0.4, n=n_sims, values=None)], fixed=dict(v=v, b_e=30.0, wNoise=1e-4), seed=12)
    outs = {}
    for form in (1, 3):
        kw = dict(sims_per_cta=spc, ctas_per_group=clu) if form == 3 else {}
        _, sw = tvbx.sweep_from_config(cfg, W, L, latency_form=form, chunk_samples=40, **kw)
        tr = [sw.run(part, 0.1, noise_on=True, ds=10, discard_steps=100, traj_steps=part) for part in (403, 1, 996)]
        info = sw.launch_info()
        if form == 3:
            assert info["latency_form"] == 2 and info["ctas_per_group"] == clu and info["sims_per_cta"] == spc
            assert info["ctas"] == clu * ((n_sims + spc - 1) // spc)
        outs[form] = (np.concatenate(tr, axis=1), sw.state(), sw.fc_readout())
    np.testing.assert_array_equal(outs[1][0], outs[3][0])
    for a, b in zip(outs[1][1] + outs[1][2], outs[3][1] + outs[3][2]):
        np.testing.assert_array_equal(a, b)


def test_grouped_latency_form_under_concurrent_launches_and_its_fallback():
    """(a) Two sweeps in the grouped form (cooperative launches, each wants the whole GPU) enqueued on two streams at once:
    the launches must serialise, not deadlock, and give the results of a run on its own.  (b) The grouped mapping is chosen
    at tvbx_sweep_create, before dt is known; if the delays then turn out too short for 8-step chunks, the first tvbx_run
    falls back to the mapping the sweep would have had without it -- bit-identical to latency_form = 1."""
    import torch
    cfg = wl.config(4)
    W, L = wl.config_connectome(cfg)
    kw = dict(noise_on=True, ds=10, discard_steps=200)

    def one(stream=None):
        _, sw = tvbx.sweep_from_config(cfg, W, L, chunk_samples=64)
        return sw
    ref = one(); ref.run(1500, 0.1, **kw)
    assert ref.launch_info()["ctas_per_group"] == 4
    want = ref.fc_readout() + ref.state()
    a, b = one(), one()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for part in (700, 800):
        a.run(part, 0.1, stream=s1, **kw)
        b.run(part, 0.1, stream=s2, **kw)
    torch.cuda.synchronize()
    for sw in (a, b):
        for x, y in zip(sw.fc_readout() + sw.state(), want):
            np.testing.assert_array_equal(x, y)
    # (b) 40 simulations at v = 60 m/s: minimum delay 2 steps -> one-step chunks
    cfgf = dict(axes=[dict(name="G", lo=0.0, hi=0.4, n=40, values=None)], fixed=dict(v=60.0, wNoise=1e-4), seed=3)
    outs = []
    for form in (0, 1):
        _, sw = tvbx.sweep_from_config(cfgf, W, L, latency_form=form, chunk_samples=40)
        sw.run(900, 0.1, **kw)
        info = sw.launch_info()
        assert info["ctas_per_group"] == 1 and info["latency_form"] == 1
        outs.append((info["sims_per_cta"], sw.fc_readout() + sw.state()))
    assert outs[0][0] == outs[1][0]
    for x, y in zip(outs[0][1], outs[1][1]):
        np.testing.assert_array_equal(x, y)
    _, sw3 = tvbx.sweep_from_config(cfgf, W, L, latency_form=3)
    with pytest.raises(tvbx.TvbxError):
        sw3.run(10, 0.1, **kw)


def test_latency_form_is_chosen_for_small_sweeps_and_refused_where_it_does_not_apply():
    cfg = wl.config(4)
    W, L = wl.config_connectome(cfg)
    _, sw = tvbx.sweep_from_config(cfg, W, L)
    sw.run(10, 0.1, noise_on=True, ds=10)
    info = sw.launch_info()
    assert info["latency_form"] == 2                    # 256 sims: all CTAs resident, about one warp per scheduler
    # ... grouped: 7 simulations per 4 CTAs = 148 CTAs of 4 consumer warps, one per scheduler (the one-CTA mappings put two on one)
    assert (info["ctas_per_group"], info["sims_per_cta"], info["ctas"], info["threads"]) == (4, 7, 148, 320)
    cfg2 = wl.config(2)
    _, sw2 = tvbx.sweep_from_config(cfg2, W, L)
    sw2.run(10, 0.1, noise_on=True, ds=10)
    assert sw2.launch_info()["latency_form"] == 1       # 1,024 sims fill the GPU: throughput form
    _, sw3 = tvbx.sweep_from_config(cfg2, W, L, latency_form=2)
    with pytest.raises(tvbx.TvbxError):
        sw3.run(10, 0.1, noise_on=True, ds=10)          # 476 nodes per CTA: does not apply
    cfgv = dict(axes=[dict(name="G", lo=0.0, hi=0.4, n=4, values=None)], fixed=dict(v=60.0), seed=1)
    _, sw4 = tvbx.sweep_from_config(cfgv, W, L, latency_form=2)
    with pytest.raises(tvbx.TvbxError):
        sw4.run(10, 0.1, noise_on=True, ds=10)          # minimum delay of 2 steps: one-step chunks

"""GPU parity of the round-2 epilogue additions: up / down-state durations (f4; Tab. 2; reading A25) and the
top-k selection of the FC scores (f3), against oracle/updown.py and oracle/fc_scores.py on the oracle's own series."""
import numpy as np
import pytest

import workloads as wl
import paper_2311_13337_b200 as tvbx
from oracle import oracle as orc
from oracle import updown as oud
from oracle import fc_scores as ofs

pytestmark = pytest.mark.gpu


def _window_means(traj, ds, discard, dtype):
    """The kept 1-ms excitatory samples exactly as the kernels form them from the trajectory: a running sum of ds
    post-update values in the kernel's arithmetic type, started from zero at every window, times (1 / ds) rounded to
    that type (tvbx_integrate2.cuh S6; A17: windows ending at a step <= discard are dropped)."""
    E = traj[:, :, 0, :].astype(dtype)                          # [S][steps][N]
    S, steps, N = E.shape
    nwin = steps // ds
    inv = dtype(1.0) / dtype(ds)
    out = []
    for w in range(nwin):
        if (w + 1) * ds <= discard:
            continue
        acc = np.zeros((S, N), dtype)
        for j in range(ds):
            acc = (acc + E[:, w * ds + j, :]).astype(dtype)
        out.append((inv * acc).astype(dtype))
    return np.stack(out, axis=1)                                # [S][samples][N]


@pytest.mark.parametrize("kw,precision", [(dict(chunk_samples=37), tvbx.TVBX_F32), (dict(chunk_samples=50, sims_per_cta=3), tvbx.TVBX_F32),
                                          (dict(chunk_samples=64), tvbx.TVBX_F64)], ids=["fp32", "fp32_spc3", "fp64"])
def test_state_durations_match_the_oracle(kw, precision):
    """Strong adaptation and noise make the rates cross the threshold many times.  Whether a sample is UP is a floating-
    point comparison that decides an integer, so both sides take it in the kernel's precision: the oracle's episode
    counting (oracle/updown.py) runs on the 1-ms samples formed from the GPU trajectory exactly as the kernel forms them,
    with the threshold rounded to that precision.  Then every count must agree EXACTLY and the mean durations to FP32
    rounding -- over several ragged chunks (the state machine is carried across chunk reductions and launches), with an
    open chunk at readout.  That those samples agree with the oracle's own within tolerance is the business of the
    trajectory / mean-rate parity tests."""
    N = 20
    W, L = wl.connectome(N, seed=4, keep=0.4)
    cfg = dict(axes=[dict(name="b_e", lo=20.0, hi=80.0, n=4, values=None)], fixed=dict(v=4.0, G=0.3, wNoise=4e-4), seed=21)
    steps, ds, discard = 6000, 10, 500
    o = orc.OracleSweep(W, L, wl.grid_params(cfg), seed=cfg["seed"])
    o.run(steps, 0.1, noise_on=True, ds=ds, discard_steps=discard)
    xs_o = np.stack([o.samples(s)[0] for s in range(o.S)])
    dtype = np.float64 if precision == tvbx.TVBX_F64 else np.float32
    thr = float(np.float32(np.median(xs_o)))                   # FP32-representable: the library compares in float
    _, sw = tvbx.sweep_from_config(cfg, W, L, updown_threshold_khz=thr, precision=precision, **kw)
    traj = sw.run(steps, 0.1, noise_on=True, ds=ds, discard_steps=discard, traj_steps=steps)
    xs = _window_means(traj, ds, discard, dtype)
    assert xs.shape == xs_o.shape and np.abs(xs / xs_o - 1).max() < 1e-2          # the same series as the oracle's, within the mean-rate tolerance
    n_up, m_up, n_dn, m_dn = sw.state_durations()
    assert n_up.shape == (4, N) and n_up.dtype == np.int32 and m_up.dtype == np.float32
    total = 0
    for s in range(4):
        ru, rmu, rd, rmd = oud.state_durations(xs[s].astype(np.float32), thr, sample_ms=ds * 0.1)      # (float)x > thr, as the kernel
        np.testing.assert_array_equal(n_up[s], ru); np.testing.assert_array_equal(n_dn[s], rd)
        np.testing.assert_allclose(m_up[s], rmu, rtol=1e-6); np.testing.assert_allclose(m_dn[s], rmd, rtol=1e-6)
        total += int(np.sum(ru))
        # and against the oracle's own FP64 series, wherever no sample sits within 0.5 % of the threshold
        ou, _, od, _ = oud.state_durations(xs_o[s], thr, sample_ms=ds * 0.1)
        clear = np.abs(xs_o[s] / thr - 1).min(axis=0) > 5e-3
        np.testing.assert_array_equal(n_up[s][clear], np.asarray(ou)[clear]); np.testing.assert_array_equal(n_dn[s][clear], np.asarray(od)[clear])
    assert total > 50                                   # the series really alternate
    again = sw.state_durations()
    for a, b in zip((n_up, m_up, n_dn, m_dn), again):
        np.testing.assert_array_equal(a, b)
    # streaming: more steps can only add episodes; resumable across launches
    sw.run(1000, 0.1, noise_on=True, ds=ds, discard_steps=discard)
    n_up2 = sw.state_durations()[0]
    assert np.all(n_up2 >= n_up)
    # device outputs
    import torch
    dev = sw.state_durations(device=True)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(dev[0].cpu().numpy(), n_up2)


def test_state_durations_errors():
    W, L = wl.connectome(12, seed=2, keep=0.5)
    cfg = dict(axes=[], fixed={}, seed=0)
    _, sw = tvbx.sweep_from_config(cfg, W, L)
    sw.run(100, 0.1, ds=10)
    with pytest.raises(tvbx.TvbxError):
        sw.state_durations()                            # created without a threshold
    with pytest.raises(tvbx.TvbxError):
        tvbx.sweep_from_config(cfg, W, L, updown_threshold_khz=-1.0)
    _, sw2 = tvbx.sweep_from_config(cfg, W, L, updown_threshold_khz=0.01)
    with pytest.raises(tvbx.TvbxError):
        sw2.state_durations()                           # no run yet


def test_top_k_matches_the_oracle_selection():
    """P:119 "the best ten fittest simulations": the k best by fitness / FCSC / mean FC.  The library's scores are FP32
    and within 0.02 of the oracle's (test_fc_scores_match_the_oracle); the SELECTION is integer work and is checked
    exactly against oracle/fc_scores.top_k applied to the library's own scores, ties included."""
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    axes = [dict(name="G", lo=0.0, hi=0.5, n=6, values=None), dict(name="b_e", lo=0.0, hi=120.0, n=7, values=None)]
    cfg = dict(axes=axes, fixed=dict(v=4.0, wNoise=1e-4), seed=5)
    sims = list(range(41, -1, -1))                      # reversed: local order != external order
    _, sw = tvbx.sweep_from_config(cfg, W, L, sim_ids=sims)
    sw.run(3000, 0.1, noise_on=True, ds=10, discard_steps=500)
    ref = np.random.default_rng(1).uniform(-0.2, 0.8, (68, 68)); ref = 0.5 * (ref + ref.T)
    sc = sw.fc_scores(ref_fc=ref)
    for which in ("fcsc", "fitness", "mean_fc"):
        for k in (1, 10, 42, 60):
            ids, vals = sw.top_k(k, which=which, ref_fc=ref)
            want_idx, want_val = ofs.top_k(sc[which], k)
            assert ids.tolist() == [sims[i] for i in want_idx]
            np.testing.assert_array_equal(vals, np.asarray(want_val, np.float32))
            assert np.all(np.diff(vals) <= 0)
    with pytest.raises(tvbx.TvbxError):
        sw.top_k(5, which="fitness")                    # no reference FC
    with pytest.raises(tvbx.TvbxError):
        sw.top_k(0)

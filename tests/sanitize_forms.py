"""Every kernel form of the library on cfg-1-sized sweeps, two launches each (resume path), all outputs read back and
checked finite.  Written as the driver for compute-sanitizer ("Race detection"):

    compute-sanitizer --tool memcheck python tests/sanitize_forms.py

compute-sanitizer is CLOSED on this GPU pool ("runs under it have left GPUs needing a reset" -- gpurun refuses it), so
the run is recorded as unavailable in profiles/r2_sanitizer.md and the hazards it would look for are covered by tests
instead: tests/test_gpu_parity_r2.py::test_chunk_pipeline_results_do_not_depend_on_the_mapping (ring read-before-write
or overwrite-before-read would make results depend on warp timing) and the bit-exact resume / reset / pool tests.
Run plainly (`python tests/sanitize_forms.py`) it is a smoke run of all forms.  Host (numpy) buffers only: torch is
never imported.  Prints one line per form; exits non-zero on the first library error."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402
import paper_2311_13337_b200 as tvbx  # noqa: E402

STEPS = int(os.environ.get("SANITIZE_STEPS", "160"))


def form(name, N, v, keep=0.4, n_sims=5, expect=None, **kw):
    W, L = wl.connectome(N, seed=N, keep=keep)
    cfg = dict(axes=[dict(name="G", lo=0.05, hi=0.4, n=n_sims, values=None)], fixed=dict(v=v, b_e=20.0, wNoise=1e-4), seed=3)
    conn, sw = tvbx.sweep_from_config(cfg, W, L, chunk_samples=5, updown_threshold_khz=5e-4, **kw)
    for part in (STEPS // 2 + 3, STEPS - STEPS // 2 - 3):          # two launches: resume path, SRING copy-back
        sw.run(part, 0.1, noise_on=True, ds=10, discard_steps=20)
    fc, me, mi = sw.fc_readout()
    sc = sw.fc_scores()
    rs = sw.rate_stats()
    ud = sw.state_durations()
    ids, best = sw.top_k(3, which="mean_fc")
    info = sw.launch_info()
    assert np.isfinite(fc).all() and np.isfinite(me).all() and np.isfinite(sc["fcsc"]).all() and np.isfinite(rs[0]).all() and np.isfinite(ud[1]).all() and len(ids) == min(3, n_sims)
    if expect:
        assert sw.kernel_name() == expect, (sw.kernel_name(), expect)
    print(f"{name}: ok  kernel={sw.kernel_name()} fc={sw.fc_kernel_name()} launch={info}", flush=True)
    sw.close(); conn.close()


def main():
    P2, G = "tvbx::integrate2_kernel", "tvbx::integrate_kernel"
    form("single CTA, 8-slot chunks (cfg-1 shape)", 68, 4.0, n_sims=8, expect=P2)
    form("single CTA, small instance, 1 sim per CTA", 23, 4.0, sims_per_cta=1, expect=P2)
    form("single CTA, 4-slot chunks + ring in shared memory", 40, 30.0, expect=P2)
    form("single CTA, 2-slot chunks + ring in shared memory", 40, 120.0, expect=P2)
    form("single CTA, zero minimum delay", 19, 1e9, expect=P2)
    form("single CTA, delay table through L1/L2", 150, 4.0, keep=1.0, n_sims=3, sims_per_cta=3, expect=P2)
    form("cluster of 3 CTAs, scalar gather (short chunks)", 37, 40.0, sims_per_cta=4, ctas_per_group=3, expect=P2)
    form("cluster of 3 CTAs, vector gather", 37, 4.0, sims_per_cta=4, ctas_per_group=3, expect=P2)
    form("cluster of 6 CTAs, vector gather, 8 sims (cfg-5 shape)", 90, 3.0, n_sims=9, sims_per_cta=8, ctas_per_group=6, expect=P2)
    form("packed kernel with inhibitory samples", 24, 4.0, rate_stats_inhibitory=True, expect=P2)
    form("general kernel FP32 (16 sims per CTA)", 20, 4.0, n_sims=16, sims_per_cta=16, expect=G)
    form("general kernel FP32, several region passes", 45, 3.0, sims_per_cta=4, threads_per_cta=64, expect=G)
    form("general kernel FP64 mode", 20, 4.0, precision=tvbx.TVBX_F64, expect=G)
    form("general kernel, tau_e != tau_i (jets)", 20, 4.0, params=dict(tau_i=7.5), expect=G)
    form("ring in shared memory for the whole launch (small CTA, 8-slot chunks)", 30, 8.0, n_sims=2, sims_per_cta=1, expect=P2)
    form("low-latency warp pairs, one CTA per group", 40, 4.0, n_sims=4, sims_per_cta=2, latency_form=2, expect=P2)
    form("one-step chunks, fully mirrored ring in shared memory", 40, 300.0, expect=P2)
    form("grouped low-latency form: 3 CTAs per group, cooperative launch", 37, 4.0, n_sims=7, sims_per_cta=3, ctas_per_group=3, latency_form=3, expect=P2)
    form("FC register tiles", 33, 4.0, fc_mode=tvbx.TVBX_FC_FP32, expect=P2)
    form("FC tensor cores, two row blocks", 130, 4.0, keep=0.2, n_sims=2, sims_per_cta=2, expect=P2)
    print("all forms ok", flush=True)


if __name__ == "__main__":
    main()

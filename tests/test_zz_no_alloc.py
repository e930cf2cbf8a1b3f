"""GPU test of the entry point that allocates nothing (include/tvbx_noalloc.h, csrc/tvbx_noalloc.cu): tvbx_top_k_noalloc, the
top-k selection with its scratch in a static __device__ array, against the existing path tvbx_top_k (per-sweep buffers from
cudaMalloc).  Named test_zz_* so that pytest collects it LAST: the suite runs with `pytest -x`, and a failure here must not
hide the tests before it.  The selection is integer / index work: the bar is exact equality (positions and FP32 values)."""
import numpy as np
import pytest

import workloads as wl
import paper_2311_13337_b200 as tvbx
from paper_2311_13337_b200 import binding as B

pytestmark = pytest.mark.gpu


def _sweep_with_scores():
    import torch
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    axes = [dict(name="G", lo=0.0, hi=0.5, n=5, values=None), dict(name="b_e", lo=0.0, hi=120.0, n=6, values=None)]
    cfg = dict(axes=axes, fixed=dict(v=4.0, wNoise=1e-4), seed=7)
    sims = list(range(29, -1, -1))                       # reversed: local order != external order
    _, sw = tvbx.sweep_from_config(cfg, W, L, sim_ids=sims)
    sw.run(2000, 0.1, noise_on=True, ds=10, discard_steps=500)
    ref = np.random.default_rng(3).uniform(-0.2, 0.8, (68, 68)); ref = 0.5 * (ref + ref.T)
    sc = sw.fc_scores(ref_fc=ref, device=True)           # the score arrays in device memory, as the new entry point takes them
    torch.cuda.synchronize()
    return sw, sims, ref, sc


def test_no_alloc_top_k_equals_the_existing_path_on_two_calls_in_a_row():
    import torch
    sw, sims, ref, sc = _sweep_with_scores()
    S = len(sims)
    out_idx = torch.full((64,), -7, device="cuda", dtype=torch.int32)       # the caller's outputs, allocated once, up front
    out_val = torch.full((64,), -7.0, device="cuda", dtype=torch.float32)
    torch.cuda.synchronize()
    # two calls in a row on the SAME scores: the static array keeps the first call's flags, the second must not see them;
    # then other scores and other k, including k > n
    plan = [("fcsc", 10), ("fcsc", 10), ("fitness", 7), ("mean_fc", S), ("fitness", 50), ("fcsc", 1)]
    for which, k in plan:
        want_ids, want_vals = sw.top_k(k, which=which, ref_fc=ref)          # existing path
        m = B.top_k_noalloc(sc[which], k, out_idx, out_val)
        torch.cuda.synchronize()
        assert m == min(k, S) == len(want_ids)
        got_idx = out_idx[:m].cpu().numpy()
        assert [sims[i] for i in got_idx] == want_ids.tolist(), (which, k)
        np.testing.assert_array_equal(out_val[:m].cpu().numpy(), want_vals)
        assert np.all(out_idx[m:].cpu().numpy() == -7) or m == 64           # nothing written past min(k, n)
        out_idx.fill_(-7); out_val.fill_(-7.0)


def test_no_alloc_top_k_ties_large_inputs_and_the_size_limit():
    import torch
    g = torch.Generator(device="cpu").manual_seed(11)
    # ties go to the lower index; a large input (several strides of the 1024 threads) after a small one and back
    for n, k in ((5, 3), (300001, 16), (2049, 40), (5, 5)):
        x = torch.randint(0, 50, (n,), generator=g).to(torch.float32)       # many equal scores
        xs = x.cuda()
        out_idx = torch.zeros(k, device="cuda", dtype=torch.int32); out_val = torch.zeros(k, device="cuda", dtype=torch.float32)
        m = B.top_k_noalloc(xs, k, out_idx, out_val)
        torch.cuda.synchronize()
        order = np.lexsort((np.arange(n), -x.numpy()))[:m]                   # by score descending, then by index ascending
        np.testing.assert_array_equal(out_idx[:m].cpu().numpy(), order.astype(np.int32))
        np.testing.assert_array_equal(out_val[:m].cpu().numpy(), x.numpy()[order])
    # beyond the static array: refused with a message that names the limit, nothing enqueued
    big = torch.zeros(B.NOALLOC_MAX_SCORES + 1, device="cuda", dtype=torch.float32)
    out_idx = torch.zeros(4, device="cuda", dtype=torch.int32); out_val = torch.zeros(4, device="cuda", dtype=torch.float32)
    with pytest.raises(tvbx.TvbxError) as e:
        B.top_k_noalloc(big, 4, out_idx, out_val)
    assert "TVBX_NOALLOC_MAX_SCORES" in str(e.value)
    with pytest.raises(tvbx.TvbxError):
        B.top_k_noalloc(big[:10], 0, out_idx, out_val)
    # the largest accepted size works
    full = torch.arange(B.NOALLOC_MAX_SCORES, device="cuda", dtype=torch.float32)
    assert B.top_k_noalloc(full, 4, out_idx, out_val) == 4
    torch.cuda.synchronize()
    n = B.NOALLOC_MAX_SCORES
    assert out_idx.cpu().tolist() == [n - 1, n - 2, n - 3, n - 4]

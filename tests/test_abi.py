"""CPU-only checks of the C-ABI boundary (include/tvbx.h): the library loads, exports every declared
symbol, and its HOST bookkeeping (S0: grid, delay indices, ring lengths, sharding ids) is bit-exact
against NumPy and against the oracle.  No compute call succeeds without a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import workloads as wl
import paper_2311_13337_b200 as tvbx
from paper_2311_13337_b200 import binding as B
from oracle import oracle as orc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    tvbx.build()
    orc.build()


def _declared_symbols():
    src = "".join(open(os.path.join(ROOT, "include", h)).read() for h in ("tvbx.h", "tvbx_diag.h", "tvbx_noalloc.h"))
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tvbx_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    names = _declared_symbols()
    assert len(names) >= 20 and "tvbx_run" in names and "tvbx_fc_readout" in names
    L = C.CDLL(tvbx.LIB_PATH)
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/*.h but not exported"
    assert sorted(tvbx.EXPORTS) == names
    assert tvbx.lib().tvbx_version() >= 100


def test_param_ids_match_header_and_workload_order():
    """The binding's ids, the header enum order and workloads.PARAM_NAMES are the same list."""
    for i, name in enumerate(wl.PARAM_NAMES):
        assert B.PARAM_IDS[name] == i
    assert B.N_PARAMS == wl.N_PARAMS == orc.lib().orc_num_params()
    np.testing.assert_array_equal(tvbx.default_params(), wl.param_vector())


@pytest.mark.parametrize("i", [1, 2, 3, 4, 5])
def test_grid_values_bit_exact(i):
    """P13 / A19: sim index -> parameter tuple equals numpy.linspace + meshgrid(indexing='ij') C-order."""
    cfg = wl.config(i)
    W, L = wl.connectome(8, seed=1, keep=0.5)
    conn, sw = tvbx.sweep_from_config(cfg, W, L)
    P = wl.grid_params(cfg)
    assert sw.n_sims == sw.grid_size == P.shape[0]
    rng = np.random.default_rng(i)
    sims = np.unique(np.concatenate([[0, sw.n_sims - 1], rng.integers(0, sw.n_sims, 200)]))
    for s in sims:
        for a in cfg["axes"]:
            assert sw.param(int(s), a["name"]) == P[s, wl.PARAM_NAMES.index(a["name"])]
        for name, val in cfg["fixed"].items():
            assert sw.param(int(s), name) == val
        assert sw.ext_id(int(s)) == s


def test_axis_formula_matches_oracle_and_linspace():
    for lo, hi, n in [(0.0, 0.5, 32), (0.0, 120.0, 64), (-10.0, 10.0, 16), (1e-9, 1e-4, 7), (3.0, 3.0, 1)]:
        W, L = wl.connectome(4, seed=2, keep=1.0)
        conn = tvbx.Connectome(W, L)
        sw = tvbx.Sweep(conn, [dict(name="G", lo=lo, hi=hi, n=n, values=None)])
        got = np.array([sw.param(s, "G") for s in range(n)])
        np.testing.assert_array_equal(got, np.linspace(lo, hi, n))
        np.testing.assert_array_equal(got, [orc.axis_value(lo, hi, n, i) for i in range(n)])


@pytest.mark.parametrize("i", [3, 5])
def test_delay_indices_and_ring_lengths_bit_exact(i):
    """P13 / A13: d_kj = rint((L/v)/dt) in FP64, half-to-even; -1 for dropped edges; H = D + 1."""
    cfg = wl.config(i)
    W, L = wl.config_connectome(cfg)
    conn, sw = tvbx.sweep_from_config(cfg, W, L)
    N = W.shape[0]
    dt = cfg["dt"]
    sims = [0, 1, 2, 3, 4, 5, 6, 7] if i == 3 else [0, sw.n_sims - 1]
    rng = np.random.default_rng(0)
    for s in sims:
        v = sw.param(s, "v")
        ref = np.rint((L / v) / dt).astype(np.int32)
        ref_kept = np.where(W != 0.0, ref, -1)
        ks, js = rng.integers(0, N, 300), rng.integers(0, N, 300)
        for k, j in zip(ks, js):
            d = sw.delay_index(s, int(k), int(j), dt)
            assert d == ref_kept[k, j]
            if d >= 0:
                assert d == orc.delay_index(L[k, j], v, dt)
        H, Hp = sw.ring_len(s, dt)
        D, dmin = ref_kept.max(), ref_kept[ref_kept >= 0].min()
        assert H == D + 1
        # the kernel's ring also holds the steps the fastest warp may be ahead (<= min delay + 1); the cluster
        # form's quad ring layout rounds the period up to a multiple of 4
        assert H + 1 <= Hp <= H + dmin + 1 + 3


def test_half_to_even_rounding():
    W = np.array([[0.0, 1.0], [1.0, 0.0]])
    for Lval, v, dt, want in [(2.5, 1.0, 1.0, 2), (3.5, 1.0, 1.0, 4), (62.5, 1.0, 1.0, 62), (0.5, 1.0, 1.0, 0)]:
        L = np.array([[0.0, Lval], [Lval, 0.0]])
        conn = tvbx.Connectome(W, L)
        sw = tvbx.Sweep(conn, [], params=dict(v=v))
        assert sw.delay_index(0, 0, 1, dt) == want == orc.delay_index(Lval, v, dt)


def test_sim_ids_subset_and_order():
    cfg = wl.config(3)
    W, L = wl.connectome(6, seed=3, keep=0.6)
    ids = [32767, 5, 1024, 5000, 7]
    conn, sw = tvbx.sweep_from_config(cfg, W, L, sim_ids=ids)
    P = wl.grid_params(cfg, sims=ids)
    assert sw.n_sims == 5 and sw.grid_size == 32768
    for loc, ext in enumerate(ids):
        assert sw.ext_id(loc) == ext
        for name in ("b_e", "a_e", "G", "v"):
            assert sw.param(loc, name) == P[loc, wl.PARAM_NAMES.index(name)]


def test_invalid_arguments_are_rejected():
    W, L = wl.connectome(5, seed=4, keep=0.8)
    bad = W.copy(); bad[0, 1] = -1.0
    with pytest.raises(tvbx.TvbxError) as e:
        tvbx.Connectome(bad, L)
    assert e.value.code == B.TVBX_EINVAL
    nan = L.copy(); nan[1, 2] = np.nan
    with pytest.raises(tvbx.TvbxError):
        tvbx.Connectome(W, nan)
    conn = tvbx.Connectome(W, L)
    with pytest.raises(tvbx.TvbxError):      # not sweepable
        tvbx.Sweep(conn, [dict(param_id=B.PARAM_IDS["g_L"], lo=1.0, hi=2.0, n=2)])
    with pytest.raises(tvbx.TvbxError):      # same parameter twice
        tvbx.Sweep(conn, [dict(name="G", lo=0, hi=1, n=2), dict(name="G", lo=0, hi=1, n=2)])
    with pytest.raises(tvbx.TvbxError):      # v <= 0
        tvbx.Sweep(conn, [dict(name="v", lo=0.0, hi=1.0, n=2)])
    with pytest.raises(tvbx.TvbxError):      # sim id outside the grid
        tvbx.Sweep(conn, [dict(name="G", lo=0, hi=1, n=2)], sim_ids=[2])
    with pytest.raises(tvbx.TvbxError):
        tvbx.Sweep(conn, [], sims_per_cta=33)
    sw = tvbx.Sweep(conn, [])
    with pytest.raises(tvbx.TvbxError) as e:
        sw.fc_readout()
    assert e.value.code == B.TVBX_ESTATE
    with pytest.raises(tvbx.TvbxError) as e:
        sw.run(10, dt=-1.0)
    assert e.value.code == B.TVBX_EINVAL


def test_no_cpu_fallback():
    """Without a CUDA device a compute call must fail loudly (TVBX_ECUDA), never fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    W, L = wl.connectome(5, seed=4, keep=0.8)
    conn = tvbx.Connectome(W, L)
    sw = tvbx.Sweep(conn, [])
    with pytest.raises(tvbx.TvbxError) as e:
        sw.run(10, dt=0.1)
    assert e.value.code == B.TVBX_ECUDA


def test_product_never_imports_oracle():
    """The package and bench's product arm must not reach into oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2311_13337_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower().replace("no oracle", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2311_13337_b200 import" not in txt and "import paper_2311_13337_b200" not in txt
            assert "tvbx.h" not in txt and "csrc/" not in txt.replace("paper_2311_13337_b200/csrc)", "")

"""Pins P10 (Philox + normals), P11 (OU), P13 (grid, delay indices) of the oracle."""
import math
import os

import numpy as np
import pytest
from scipy import stats

import workloads as wl
from oracle import oracle as orc


# ------------------------------------------------------------------ P10 Philox4x32-10
def _triton_philox(ctrs, key):
    """Independent Philox4x32-10: Triton's reference implementation run by its CPU interpreter."""
    os.environ["TRITON_INTERPRET"] = "1"
    import torch
    import triton
    import triton.language as tl

    n = len(ctrs)

    @triton.jit
    def kern(out, cin, k0, k1, n: tl.constexpr):
        o = tl.arange(0, n)
        c0 = tl.load(cin + o * 4 + 0).to(tl.uint32)
        c1 = tl.load(cin + o * 4 + 1).to(tl.uint32)
        c2 = tl.load(cin + o * 4 + 2).to(tl.uint32)
        c3 = tl.load(cin + o * 4 + 3).to(tl.uint32)
        kk0 = tl.full((n,), k0, tl.uint32)
        kk1 = tl.full((n,), k1, tl.uint32)
        a, b, c, d = tl.philox_impl(c0, c1, c2, c3, kk0, kk1, 10)
        tl.store(out + o * 4 + 0, a.to(tl.int64))
        tl.store(out + o * 4 + 1, b.to(tl.int64))
        tl.store(out + o * 4 + 2, c.to(tl.int64))
        tl.store(out + o * 4 + 3, d.to(tl.int64))

    cin = torch.tensor(ctrs, dtype=torch.int64).reshape(-1)
    out = torch.zeros(4 * n, dtype=torch.int64)
    kern[(1,)](out, cin, int(key[0]), int(key[1]), n)
    return out.reshape(n, 4).numpy()


def test_philox_matches_independent_implementation():
    rng = np.random.default_rng(7)
    ctrs = [[0, 0, 0, 0], [1, 0, 0, 0], [0, 0, 67, 1023], [0xFFFFFFFF, 0xFFFFFFFF, 0xFFFFFFFF, 0xFFFFFFFF]]
    ctrs += rng.integers(0, 2**32, size=(12, 4)).tolist()
    for key in ([0, 0], [1, 0], [0xDEADBEEF, 0x12345678]):
        try:
            ref = _triton_philox(ctrs, key)
        except Exception as e:  # pragma: no cover - triton interpreter unavailable
            pytest.skip(f"triton interpreter unavailable: {e}")
        for c, r in zip(ctrs, ref):
            assert orc.philox4x32_10(c, key) == tuple(int(x) for x in r)


def _philox4x32_10_ints(ctr, key):
    """Philox4x32-10 (Salmon et al., "Parallel random numbers: as easy as 1, 2, 3", SC'11) restated with Python integers:
    10 rounds of two 32 x 32 -> 64-bit multiplications by the round constants, key bumped by the Weyl constants."""
    M0, M1, W0, W1, MASK = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85, 0xFFFFFFFF
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for _ in range(10):
        p0, p1 = M0 * c0, M1 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & MASK, p1 & MASK, ((p0 >> 32) ^ c3 ^ k1) & MASK, p0 & MASK
        k0, k1 = (k0 + W0) & MASK, (k1 + W1) & MASK
    return (c0, c1, c2, c3)


def test_philox_matches_integer_restatement():
    """Second leg of the Philox pin, which cannot skip (the Triton-interpreter leg above depends on an optional
    package): arbitrary-precision integer arithmetic, no uint32 wrap-around semantics shared with the C++ code."""
    rng = np.random.default_rng(11)
    ctrs = [[0, 0, 0, 0], [0xFFFFFFFF] * 4, [1, 2, 3, 4]] + rng.integers(0, 2**32, size=(40, 4)).tolist()
    for key in ([0, 0], [0xFFFFFFFF, 0xFFFFFFFF], [0xDEADBEEF, 0x12345678], [2, 0]):
        for c in ctrs:
            assert orc.philox4x32_10(c, key) == _philox4x32_10_ints([int(x) for x in c], key)


def test_philox_is_a_bijection_on_a_sample_and_key_sensitive():
    outs = {orc.philox4x32_10([i, 0, 0, 0], [1, 0]) for i in range(2000)}
    assert len(outs) == 2000
    assert orc.philox4x32_10([5, 0, 0, 0], [1, 0]) != orc.philox4x32_10([5, 0, 0, 0], [2, 0])
    assert orc.philox4x32_10([5, 0, 0, 0], [1, 0]) != orc.philox4x32_10([5, 0, 0, 0], [1, 1])


def test_uniform_map_exact_in_fp32():
    """A12: u(x) = ((x >> 9) + 0.5) * 2^-23 lies in (0,1) and is exactly representable in FP32."""
    for x in (0, 511, 512, 0x80000000, 0xFFFFFFFF, 0xFFFFFE00, 123456789):
        u = orc.uniform23(x)
        assert u == ((x >> 9) + 0.5) / 8388608.0
        assert 0.0 < u < 1.0 and float(np.float32(u)) == u


def test_normal_uses_counter_layout_and_box_muller():
    """xi for step n: words (x0,x1) -> n%4 in {0,1}, (x2,x3) -> {2,3}; cos for even, sin for odd;
    counter = (q_lo, q_hi, region, sim), key = (seed_lo, seed_hi), q = n // 4."""
    seed, sim, region = (5 << 32) | 9, 77, 13
    for n in (0, 1, 2, 3, 4, 7, 4 * (2**32) + 2):
        q = n // 4
        x = orc.philox4x32_10([q & 0xFFFFFFFF, q >> 32, region, sim], [9, 5])
        xa, xb = (x[0], x[1]) if n % 4 < 2 else (x[2], x[3])
        u1, u2 = ((xa >> 9) + 0.5) / 2**23, ((xb >> 9) + 0.5) / 2**23
        r, th = math.sqrt(-2 * math.log(u1)), 2 * math.pi * u2
        ref = r * (math.sin(th) if n % 2 else math.cos(th))
        assert abs(orc.normal(seed, sim, region, n) - ref) < 1e-14


def test_normal_moments_ks_and_stream_independence():
    n = 200_000
    a = np.array([orc.normal(1, 0, 0, i) for i in range(n)])
    b = np.array([orc.normal(1, 0, 1, i) for i in range(n)])
    c = np.array([orc.normal(1, 1, 0, i) for i in range(n)])
    for x in (a, b, c):
        assert abs(x.mean()) < 4 / math.sqrt(n)
        assert abs(x.var() - 1) < 4 * math.sqrt(2 / n)
        assert stats.kstest(x, "norm").pvalue > 1e-3
    for x, y in ((a, b), (a, c), (b, c)):
        assert abs(np.corrcoef(x, y)[0, 1]) < 4 / math.sqrt(n)
    assert abs(np.corrcoef(a[:-1], a[1:])[0, 1]) < 4 / math.sqrt(n)


# ------------------------------------------------------------------ P11 OU
def test_ou_stationary_variance_and_autocorrelation():
    """Exact one-step update (A11): stationary variance sigma^2 and lag-l autocorrelation rho^l,
    rho = exp(-dt/tau_OU), independent of dt."""
    W = np.zeros((64, 64)); L = np.zeros((64, 64))
    for dt, tau in ((0.1, 5.0), (0.5, 5.0)):
        p = wl.param_vector(tau_OU=tau, sigma_OU=1.0)
        sw = orc.OracleSweep(W, L, np.tile(p, (4, 1)), seed=11)
        steps = 4000
        burn = int(10 * tau / dt)
        xs = []
        sw.run(burn, dt, noise_on=True, ds=0)
        for _ in range(steps // 4):
            sw.run(4, dt, noise_on=True, ds=0)
            xs.append(np.stack([sw.state(s)[1] for s in range(4)]))
        x = np.array(xs).reshape(len(xs), -1)              # [time (every 4 steps)][256 streams]
        rho4 = math.exp(-4 * dt / tau)
        var = x.var()
        ac = np.mean(x[:-1] * x[1:]) / var
        n_eff = x.size * (1 - rho4) / (1 + rho4)
        assert abs(var - 1.0) < 5 * math.sqrt(2 / n_eff)
        assert abs(ac - rho4) < 5 / math.sqrt(n_eff)
        assert abs(x.mean()) < 5 / math.sqrt(n_eff)


def test_noise_off_leaves_ou_untouched():
    W, L = wl.connectome(6, 3, 0.6)
    sw = orc.OracleSweep(W, L, wl.param_vector()[None], seed=3)
    sw.run(20, 0.1, noise_on=False)
    assert np.all(sw.state(0)[1] == 0.0)


# ------------------------------------------------------------------ P13 bookkeeping
def test_axis_values_match_numpy_linspace_bitwise():
    for lo, hi, n in ((0.0, 0.5, 32), (0.0, 120.0, 32), (-10.0, 10.0, 16), (0.0, 0.5, 64), (0.4, 0.9, 6),
                      (1e-9, 1e-4, 8), (3.0, 3.0, 1), (250.0, 750.0, 7)):
        ref = np.linspace(lo, hi, n)
        got = np.array([orc.axis_value(lo, hi, n, i) for i in range(n)])
        assert np.array_equal(ref, got)
        assert np.array_equal(ref.astype(np.float32), got.astype(np.float32))


def test_grid_digits_are_c_order_first_axis_slowest():
    shape = [16, 16, 16, 8]
    for s in (0, 1, 7, 8, 127, 128, 32767, 12345):
        assert orc.grid_digits(shape, s) == list(np.unravel_index(s, shape))


def test_grid_params_follow_config_axis_order():
    cfg = wl.config(3)
    P = wl.grid_params(cfg)
    nm = wl.PARAM_NAMES.index
    assert P.shape == (32768, wl.N_PARAMS)
    assert list(P[:8, nm("v")]) == [1, 2, 4, 8, 16, 32, 64, 128]      # v fastest
    assert P[8, nm("G")] == np.linspace(0, 0.5, 16)[1] and P[8, nm("v")] == 1
    assert P[-1, nm("b_e")] == 120.0 and P[0, nm("a_e")] == -10.0
    for s in (0, 5, 4097, 32767):
        d = orc.grid_digits([16, 16, 16, 8], s)
        assert P[s, nm("b_e")] == orc.axis_value(0.0, 120.0, 16, d[0])
        assert P[s, nm("a_e")] == orc.axis_value(-10.0, 10.0, 16, d[1])
        assert P[s, nm("G")] == orc.axis_value(0.0, 0.5, 16, d[2])


def test_delay_index_matches_numpy_rint_bitwise():
    rng = np.random.default_rng(0)
    L = np.concatenate([rng.uniform(0, 250, 4000), [0.0, 10.0, 25.0, 1.0, 3.0, 200.0, 6.25, 18.75]])
    for v in (1, 2, 3, 4, 8, 16, 32, 64, 128, 1e9):
        for dt in (0.1, 0.05):
            ref = np.rint((L / v) / dt).astype(np.int32)
            got = np.array([orc.delay_index(float(x), float(v), dt) for x in L], dtype=np.int32)
            assert np.array_equal(ref, got)
    # round-half-to-even (A13): 62.5 -> 62, 15.625 -> 16
    assert orc.delay_index(25.0, 4.0, 0.1) == 62 and orc.delay_index(200.0, 128.0, 0.1) == 16
    assert orc.delay_index(0.5, 1.0, 1.0) == 0 and orc.delay_index(1.5, 1.0, 1.0) == 2


def test_ring_length_is_max_delay_plus_one():
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    for v in (1.0, 4.0, 128.0):
        sw = orc.OracleSweep(W, L, wl.param_vector(v=v)[None])
        sw.run(1, 0.1)
        D = int(np.rint((L[W != 0] / v) / 0.1).max())
        assert sw.ring_len(0) == D + 1


def test_connectome_recipe_shapes():
    W, L = wl.connectome(68, 0, 0.30)
    assert W.shape == (68, 68) and np.array_equal(W, W.T) and np.array_equal(L, L.T)
    assert W.max() == 1.0 and np.all(np.diag(W) == 0) and np.all(W >= 0)
    frac = (W[np.triu_indices(68, 1)] != 0).mean()
    assert 0.25 < frac < 0.35
    off = L[np.triu_indices(68, 1)]
    assert off.min() >= 10 and off.max() <= 200
    W5, L5 = wl.connectome(360, 5, 0.50, "ellipsoid")
    assert 0.45 < (W5[np.triu_indices(360, 1)] != 0).mean() < 0.55
    assert L5.max() <= 1.2 * 170 + 1e-9 and np.all(np.diag(L5) == 0)

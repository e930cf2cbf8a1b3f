"""Pins of oracle/rate_stats.py (f4; reading A24) against closed forms and library
routines the oracle does not call."""
import numpy as np
import pytest

from oracle import rate_stats as rs


def test_closed_forms():
    n = 1000
    q = np.arange(n)
    ramp = 0.2 * q / (n - 1)                                   # 0 ... 0.2 kHz: uniform grid
    sine = 0.05 + 0.03 * np.sin(2 * np.pi * 7 * q / n)         # whole periods
    const = np.full(n, 0.1)                                    # exactly the threshold: not "exceeding"
    var, mx, above = rs.rate_stats(np.stack([ramp, sine, const], axis=1))
    assert var[0] == pytest.approx(0.2 ** 2 * (n + 1) / (12.0 * (n - 1)), rel=1e-12)      # variance of n equispaced points
    assert var[1] == pytest.approx(0.03 ** 2 / 2, rel=1e-12)                              # a^2 / 2 over whole periods
    assert var[2] == 0.0
    assert mx[0] == 0.2 and mx[1] == pytest.approx(0.08, abs=1e-4) and mx[2] == 0.1
    assert above == [int((ramp > 0.1).sum()), 0, 0] and above[0] == 500


def test_against_numpy_and_invariances():
    rng = np.random.default_rng(0)
    x = np.abs(rng.normal(0.05, 0.04, size=(333, 7)))
    var, mx, above = rs.rate_stats(x, threshold_khz=0.08)
    np.testing.assert_allclose(var, x.var(axis=0), rtol=1e-12)
    np.testing.assert_array_equal(mx, x.max(axis=0))
    np.testing.assert_array_equal(above, (x > 0.08).sum(axis=0))
    # order of the samples does not matter; a shift changes max and count, not the variance
    p = rng.permutation(333)
    var_p, mx_p, above_p = rs.rate_stats(x[p], threshold_khz=0.08)
    np.testing.assert_allclose(var_p, var, rtol=1e-12); assert mx_p == mx and above_p == above
    var_s, mx_s, _ = rs.rate_stats(x + 1.0, threshold_khz=0.08)
    np.testing.assert_allclose(var_s, var, rtol=1e-9); np.testing.assert_allclose(mx_s, np.asarray(mx) + 1.0)
    # variance is the diagonal of the co-moment matrix the FC is built from: FC_kl sqrt(var_k var_l) = cov_kl
    c = np.cov(x.T, bias=True)
    np.testing.assert_allclose(np.diag(c), var, rtol=1e-12)

"""Pins of oracle/fc_scores.py (f3: FCSC, fitness, mean FC; Tab. 2)
against library routines and closed forms, none of which the oracle calls."""
import numpy as np
import pytest
import scipy.stats

from oracle import fc_scores as fs


def sym(rng, n, diag):
    a = rng.standard_normal((n, n))
    a = 0.5 * (a + a.T)
    np.fill_diagonal(a, diag)
    return a


@pytest.mark.parametrize("n", [2, 3, 7, 68])
def test_pearson_upper_against_scipy_and_numpy(n):
    rng = np.random.default_rng(n)
    x, y = sym(rng, n, 1.0), sym(rng, n, 0.0)
    iu = np.triu_indices(n, k=1)
    got = fs.pearson_upper(x, y)
    if n == 2:
        assert got == 0.0                      # a single pair has no variance: degenerate rule
        return
    assert got == pytest.approx(scipy.stats.pearsonr(x[iu], y[iu])[0], abs=1e-13)
    assert got == pytest.approx(np.corrcoef(x[iu], y[iu])[0, 1], abs=1e-13)
    assert fs.mean_upper(x) == pytest.approx(x[iu].mean(), abs=1e-15)


def test_diagonal_and_lower_triangle_are_not_read():
    rng = np.random.default_rng(1)
    x, y = sym(rng, 9, 1.0), sym(rng, 9, 0.0)
    r = fs.pearson_upper(x, y)
    x2, y2 = x.copy(), y.copy()
    np.fill_diagonal(x2, 123.0); np.fill_diagonal(y2, -7.0)
    x2[np.tril_indices(9, -1)] = 55.0
    assert fs.pearson_upper(x2, y2) == r and fs.mean_upper(x2) == fs.mean_upper(x)


def test_closed_forms_and_invariances():
    rng = np.random.default_rng(2)
    x, y = sym(rng, 11, 1.0), sym(rng, 11, 0.0)
    assert fs.pearson_upper(x, x) == pytest.approx(1.0, abs=1e-14)
    assert fs.pearson_upper(x, -x) == pytest.approx(-1.0, abs=1e-14)
    r = fs.pearson_upper(x, y)
    assert fs.pearson_upper(y, x) == pytest.approx(r, abs=1e-15)                       # symmetric in its arguments
    assert fs.pearson_upper(3.0 * x + 2.0, 0.5 * y - 1.0) == pytest.approx(r, abs=1e-13)   # affine invariance
    assert fs.pearson_upper(x, -2.0 * y) == pytest.approx(-r, abs=1e-13)
    assert fs.pearson_upper(x, np.full((11, 11), 0.3)) == 0.0                          # zero variance -> 0
    # y = a x + noise orthogonal to x in the sample: rho = a s_x / sqrt(a^2 s_x^2 + s_e^2)
    iu = np.triu_indices(11, k=1)
    xv = x[iu] - x[iu].mean()
    e = rng.standard_normal(xv.size); e -= e.mean(); e -= xv * (e @ xv) / (xv @ xv)
    yv = 2.0 * xv + e
    ym = np.zeros((11, 11)); ym[iu] = yv
    want = 2.0 * np.sqrt(xv @ xv) / np.sqrt(4.0 * (xv @ xv) + e @ e)
    assert fs.pearson_upper(x, ym) == pytest.approx(want, abs=1e-13)


def test_fc_scores_shapes_and_permutation_equivariance():
    rng = np.random.default_rng(3)
    fc = np.stack([sym(rng, 6, 1.0) for _ in range(4)])
    sc, ref = np.abs(sym(rng, 6, 0.0)), sym(rng, 6, 1.0)
    out = fs.fc_scores(fc, sc, ref)
    assert set(out) == {"fcsc", "mean_fc", "fitness"} and all(len(v) == 4 for v in out.values())
    assert "fitness" not in fs.fc_scores(fc, sc)
    # relabelling the regions (same permutation on every matrix) changes nothing
    p = rng.permutation(6)
    out_p = fs.fc_scores(fc[:, p][:, :, p], sc[p][:, p], ref[p][:, p])
    for k in out:
        np.testing.assert_allclose(out_p[k], out[k], atol=1e-13)


def test_top_k_against_numpy_sort_and_ties():
    from oracle import fc_scores as ofs
    rng = np.random.default_rng(5)
    s = np.round(rng.normal(size=300), 1)                     # rounded: many exact ties
    for k in (1, 10, 300, 400):
        idx, val = ofs.top_k(s, k)
        order = np.lexsort((np.arange(s.size), -s))[:k]       # by score descending, then index ascending
        assert idx == order.tolist() and val == s[order].tolist()
    assert ofs.top_k([0.5, 0.5, 0.7, 0.5], 3) == ([2, 0, 1], [0.7, 0.5, 0.5])
    assert ofs.top_k([], 3) == ([], [])

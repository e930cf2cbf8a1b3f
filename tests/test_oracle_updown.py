"""Pins of oracle/updown.py (f4; Tab. 2 P:131 `mean_UD_duration`; reading A25) against closed forms, hand-counted
sequences and an independent run-length encoding with NumPy primitives the oracle does not use."""
import numpy as np
import pytest

from oracle import updown as ud


def _rle_numpy(col, thr):
    """independent restatement: change points via numpy.diff, interior runs only"""
    b = (np.asarray(col) > thr).astype(np.int8)
    cuts = np.flatnonzero(np.diff(b)) + 1                       # starts of new runs
    starts = np.concatenate([[0], cuts]); ends = np.concatenate([cuts, [len(b)]])
    runs = [(int(b[s]), int(e - s)) for s, e in zip(starts, ends)][1:-1]     # drop the two runs cut by the record's ends
    up = [r for s, r in runs if s == 1]; dn = [r for s, r in runs if s == 0]
    return len(up), (float(np.mean(up)) if up else 0.0), len(dn), (float(np.mean(dn)) if dn else 0.0)


def test_hand_counted_sequences():
    #        D  D  U  U  U  D  U  D  D  D  D  U  U  D      thr = 0.5
    x = [0, 0, 1, 1, 1, 0, 1, 0, 0, 0, 0, 1, 1, 0]
    # runs: D2 (cut by start) | U3 | D1 | U1 | D4 | U2 | D1 (cut by end)
    n_up, m_up, n_dn, m_dn = ud.state_durations([[v] for v in x], 0.5)
    assert n_up == [3] and m_up == [pytest.approx((3 + 1 + 2) / 3)]
    assert n_dn == [2] and m_dn == [pytest.approx((1 + 4) / 2)]
    # never crossing, one crossing: nothing is bounded on both sides
    for seq in ([0] * 10, [1] * 10, [0] * 5 + [1] * 5):
        assert ud.state_durations([[v] for v in seq], 0.5) == ([0], [0.0], [0], [0.0])
    # exactly the threshold is DOWN (strict >); sample_ms scales the durations
    n_up, m_up, n_dn, m_dn = ud.state_durations([[0.5], [0.6], [0.6], [0.5], [0.7], [0.5]], 0.5, sample_ms=2.0)
    assert (n_up, m_up, n_dn, m_dn) == ([2], [pytest.approx(3.0)], [1], [pytest.approx(2.0)])
    assert ud.state_durations([], 0.5) == ([], [], [], [])


def test_square_wave_closed_form():
    """Period P samples, duty d: every interior UP episode lasts d, every DOWN episode P - d; over m periods starting
    inside a DOWN phase there are m UP episodes and m - 1 complete DOWN episodes."""
    P, d, m = 40, 13, 25
    q = np.arange(m * P + 3)                                 # ends inside a DOWN phase
    x = 0.01 + 0.02 * (((q - 5) % P) < d)                      # UP on samples 5 .. 5 + d - 1 of every period
    n_up, m_up, n_dn, m_dn = ud.state_durations(x[:, None], 0.02)
    assert n_up == [m] and m_up == [pytest.approx(d)]
    assert n_dn == [m - 1] and m_dn == [pytest.approx(P - d)]


def test_against_numpy_run_length_encoding():
    rng = np.random.default_rng(3)
    x = np.abs(rng.normal(0.03, 0.02, size=(2000, 6)))
    x[:, 1] = np.convolve(x[:, 1], np.ones(25) / 25, mode="same")     # a smooth column: long episodes
    thr = 0.03
    got = ud.state_durations(x, thr, sample_ms=1.0)
    for k in range(6):
        want = _rle_numpy(x[:, k], thr)
        assert got[0][k] == want[0] and got[2][k] == want[2]
        assert got[1][k] == pytest.approx(want[1], rel=1e-12) and got[3][k] == pytest.approx(want[3], rel=1e-12)
    # invariant: counted samples + the two cut runs = all samples; UP and DOWN episodes alternate
    for k in range(6):
        assert abs(got[0][k] - got[2][k]) <= 1

"""Pins against the small text fixtures of tests/golden/ (each line carries its citation):
paper_constants.txt   -- numbers PAPER.md prints (Table 1, figure captions)
oracle_regression.txt -- FP64 oracle outputs written by tests/golden/make_golden.py (oracle/ only)."""
import importlib.util
import os
import re

import numpy as np
import pytest

import workloads as wl
from oracle import oracle as orc

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(scope="module", autouse=True)
def _built():
    import paper_2311_13337_b200 as tvbx
    tvbx.build()
    orc.build()


def paper_constants():
    out = {}
    for line in open(os.path.join(GOLD, "paper_constants.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split()
            out[k] = float(v)
    return out


def regression():
    out = {}
    for line in open(os.path.join(GOLD, "oracle_regression.txt")):
        if not line.startswith("#"):
            k, v = line.rsplit(" : ", 1)
            out[k] = float(v)
    return out


def _value(name):
    m = re.fullmatch(r"poly_([ei])\[(\d)\]", name)
    if m:
        return (wl.POLY_RS if m.group(1) == "e" else wl.POLY_FS)[int(m.group(2))]
    return wl.DEFAULTS[name]


def test_inputs_carry_the_numbers_the_paper_prints():
    pc = paper_constants()
    assert len(pc) == 31
    for name, want in pc.items():
        assert _value(name) == want, name
    # the flat parameter vector both sides receive ends with the two Table-1 rows in the printed order
    vec = wl.param_vector()
    np.testing.assert_array_equal(vec[-20:-10], [pc[f"poly_e[{i}]"] for i in range(10)])
    np.testing.assert_array_equal(vec[-10:], [pc[f"poly_i[{i}]"] for i in range(10)])


def test_library_defaults_carry_the_numbers_the_paper_prints():
    import paper_2311_13337_b200 as tvbx
    d = tvbx.default_params()
    pc = paper_constants()
    for name, want in pc.items():
        m = re.fullmatch(r"poly_([ei])\[(\d)\]", name)
        if m:
            got = d[len(wl.PARAM_NAMES) + (0 if m.group(1) == "e" else 10) + int(m.group(2))]
        else:
            got = d[wl.PARAM_NAMES.index(name)]
        assert got == want, name


def test_oracle_reproduces_its_frozen_outputs():
    """A change to the oracle's arithmetic shows up here (and as a diff of oracle_regression.txt)."""
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(GOLD, "make_golden.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    gold = regression()
    rows = mg.rows()
    assert len(rows) == len(gold)
    for k, v in rows:
        assert v == pytest.approx(gold[k], rel=1e-12, abs=1e-300), k


def test_frozen_fixed_points_agree_with_the_surveys_probe():
    """SURVEY.md section 8(c) A3 quotes a scratch probe of the isolated node (first-order equations, the same
    defaults, Table 1 as printed): E = 0.53, 0.42, 0.35 Hz and I = 1.85, 1.57, 1.41 Hz for b_e = 0, 60, 120 pA.
    The second-order terms are O(1e-3) relative at kappa = 1e-3, so the oracle's rates must land on those
    two-digit values -- an end-to-end check (transfer function, Eqs. 1-3, units) from outside the oracle."""
    gold = regression()
    for b_e, (E_hz, I_hz) in {0: (0.53, 1.85), 60: (0.42, 1.57), 120: (0.35, 1.41)}.items():
        assert 1e3 * gold[f"node b_e={b_e} step=20000 E"] == pytest.approx(E_hz, abs=0.006)
        assert 1e3 * gold[f"node b_e={b_e} step=20000 I"] == pytest.approx(I_hz, abs=0.006)


@pytest.mark.gpu
def test_cuda_path_against_the_frozen_oracle_outputs():
    """The CUDA path against stored oracle values (no live oracle in this test): cfg-1 state at step 1,000 with
    the noise off (FP32, 1e-3 relative to the variable's scale) and the isolated-node rates after 2 s."""
    import paper_2311_13337_b200 as tvbx
    gold = regression()
    names = ("E", "I", "C_ee", "C_ei", "C_ii", "W_e", "W_i")
    cfg = wl.config(1)
    W, L = wl.config_connectome(cfg)
    _, sw = tvbx.sweep_from_config(cfg, W, L)
    sw.run(1000, cfg["dt"], noise_on=False, ds=10)
    y, _ = sw.state()
    for s in (0, 7):
        for k in (0, 33, 67):
            for q, nm in enumerate(names):
                want = gold[f"cfg1 noise=0 sim={s} region={k} step=1000 {nm}"]
                scale = max(abs(gold[f"cfg1 noise=0 sim={s} region={kk} step=1000 {nm}"]) for kk in (0, 33, 67))
                assert abs(float(y[s][q][k]) - want) <= 1e-3 * scale + 1e-30, (s, k, nm)
    for b_e in (0.0, 60.0, 120.0):
        conn = tvbx.Connectome(np.zeros((2, 2)), np.zeros((2, 2)))
        sw = tvbx.Sweep(conn, [], params=dict(G=0.0, b_e=b_e))
        sw.run(20000, 0.1, noise_on=False, ds=0)
        y, _ = sw.state()
        for q, nm in enumerate(names[:2]):
            assert float(y[0][q][0]) == pytest.approx(gold[f"node b_e={b_e:g} step=20000 {nm}"], rel=1e-3)


def test_connectome_hashes():
    """The seeded generator reproduces the recorded inputs bit for bit (tests/golden/connectome_sha256.txt)."""
    import hashlib
    want = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "connectome_sha256.txt")):
        if line.strip() and not line.startswith("#"):
            parts = line.split()
            want[parts[0]] = parts[-1]
    for key, cid in (("cfg1-4", 1), ("cfg5", 5)):
        W, L = wl.config_connectome(wl.config(cid))
        assert W.dtype == np.float64 and W.flags.c_contiguous
        assert hashlib.sha256(W.tobytes() + L.tobytes()).hexdigest() == want[key]
    for cid in (2, 3, 4):                       # the same 68-region connectome
        W, L = wl.config_connectome(wl.config(cid))
        assert hashlib.sha256(W.tobytes() + L.tobytes()).hexdigest() == want["cfg1-4"]

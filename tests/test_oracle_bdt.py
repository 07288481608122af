"""Pins of oracle/bdt.py: a hand-worked forest, a pure-Python per-event walk, depth-1
stumps as a closed form, forests that send every event to one known leaf, the logistic output."""
import os

import numpy as np

import synth
from oracle import bdt

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(line, dtype):
    return np.array([[float(v) for v in part.split()] for part in line.split(":", 1)[1].split("|")]).astype(dtype)


def test_worked_example():
    d = {}
    for line in open(os.path.join(GOLD, "bdt_worked_example.txt")):
        if line.startswith("#") or ":" not in line:
            continue
        d[line.split(":")[0]] = line
    f, t, l, x = _rows(d["feature"], np.int32), _rows(d["threshold"], np.float32), _rows(d["leaf"], np.float32), _rows(d["x"], np.float32)
    want = _rows(d["margin"], np.float64)[0]
    m = bdt.margins(f, t, l, x)
    assert np.abs(m - want).max() < 1e-6            # leaves are fp32 roundings of the decimals
    # the logistic output and its column order, pinned to the golden file's decimal-arithmetic values and to scipy's expit
    # (the leaves are fp32 roundings of the decimals, so the margins differ from the decimals by ~1e-8)
    from scipy.special import expit
    p = bdt.predict(f, t, l, x)
    prob = _rows(d["prob"], np.float64)[0]
    assert p.shape == (5, 2)
    assert np.abs(p[:, 1] - prob).max() < 1e-7 and np.abs(p[:, 0] - (1.0 - prob)).max() < 1e-7
    assert np.abs(p[:, 1] - expit(m)).max() < 1e-15 and np.abs(p[:, 0] - expit(-m)).max() < 1e-15
    assert (p[:, 1] > 0.5).tolist() == [True, False, True, True, False]        # positive margin -> second column wins


def test_logistic_special_cases():
    """margin 0 -> (0.5, 0.5) exactly; a large positive margin puts all the mass on the SECOND column, a large negative one on
    the first (a swapped column order or a wrong sign in the exponent fails here)"""
    f = np.zeros((1, 1), np.int32); t = np.zeros((1, 1), np.float32)
    x = np.array([[-1.0], [1.0]], np.float32)                                   # first event goes left, second right
    p = bdt.predict(f, t, np.array([[0.0, 0.0]], np.float32), x)
    assert np.array_equal(p, np.full((2, 2), 0.5))
    p = bdt.predict(f, t, np.array([[40.0, -40.0]], np.float32), x)
    assert p[0, 1] > 1 - 1e-15 and p[0, 0] < 1e-15 and p[1, 0] > 1 - 1e-15 and p[1, 1] < 1e-15


def walk(feature, threshold, leaf, x):
    """one event, one tree at a time, plain Python"""
    T, n_int = feature.shape
    out = []
    for e in range(x.shape[0]):
        m = 0.0
        for t in range(T):
            node = 0
            while node < n_int:
                node = 2 * node + 1 if x[e, feature[t, node]] < threshold[t, node] else 2 * node + 2
            m += float(leaf[t, node - n_int])
        out.append(m)
    return np.array(out)


def test_against_per_event_walk():
    for depth, T, F in ((1, 3, 2), (3, 7, 5), (6, 100, 20)):
        f, t, l = synth.make_bdt(seed=depth, n_trees=T, depth=depth, n_features=F)
        x = synth.make_bdt_events(300, F, seed=9)
        x[::17, 0] = np.nan
        assert np.abs(bdt.margins(f, t, l, x) - walk(f, t, l, x)).max() < 1e-12


def test_stumps_closed_form():
    """depth 1: margin = sum_t (leaf[t, 0] if x[f_t] < thr_t else leaf[t, 1])"""
    f, t, l = synth.make_bdt(seed=4, n_trees=50, depth=1, n_features=20)
    x = synth.make_bdt_events(1000)
    left = x[:, f[:, 0]] < t[:, 0][None, :]
    want = np.where(left, l[:, 0][None, :].astype(np.float64), l[:, 1][None, :].astype(np.float64)).sum(1)
    assert np.abs(bdt.margins(f, t, l, x) - want).max() < 1e-12


def test_forced_paths():
    f, t, l = synth.make_bdt(seed=5, n_trees=10, depth=4, n_features=20)
    x = synth.make_bdt_events(64)
    hi = np.full_like(t, np.inf); lo = np.full_like(t, -np.inf)
    assert np.allclose(bdt.margins(f, hi, l, x), l[:, 0].astype(np.float64).sum())        # always left: first leaf
    assert np.allclose(bdt.margins(f, lo, l, x), l[:, -1].astype(np.float64).sum())       # always right: last leaf

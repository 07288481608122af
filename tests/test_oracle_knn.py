"""Pins for the oracle's kNN (oracle.c knn_jet; readings R3-R6).  CPU only."""
import os
import numpy as np
import pytest
import oracle
from np_restatement import knn_lexsort

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _lattice_cases():
    for line in open(os.path.join(GOLD, "knn_lattices.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        name, pts, k, q, s = [t.strip() for t in line.split("|")]
        P = np.array([[float(v) for v in p.split(",")] for p in pts.split(";")])
        yield name, P, int(k), int(q), sorted(int(v) for v in s.split(","))


@pytest.mark.parametrize("name,P,k,q,expect", list(_lattice_cases()))
def test_lattice_tie_breaks(name, P, k, q, expect):
    """Worked examples with exact ties: lower index wins (north_star (1)); self excluded by index (R4)."""
    idx, _, _ = oracle.knn(P, np.array([0, len(P)], np.int32), k)
    assert sorted(idx[q].tolist()) == expect


def test_brute_force_random_jets():
    """Brute force on tiny jets: full lexsort of (d, j) pairs, 1000 jets, n in [1,24], D in {2,5,64}, k in {1,4,16}."""
    rng = np.random.default_rng(11)
    for trial in range(1000):
        n = int(rng.integers(1, 25)); D = int(rng.choice([2, 5, 64])); k = int(rng.choice([1, 4, 16]))
        s = rng.normal(0, 1, (n, D))
        if trial % 7 == 0:                      # force exact ties: integer lattice
            s = rng.integers(0, 3, (n, D)).astype(np.float64)
        idx, dk, dk1 = oracle.knn(s, np.array([0, n], np.int32), k)
        ref, d = knn_lexsort(s, k)
        assert np.array_equal(idx, ref), (trial, n, D, k)
        for i in range(n):
            sel = idx[i][idx[i] >= 0]
            if sel.size:
                assert dk[i] == d[i, sel].max()
            rest = [j for j in range(n) if j != i and j not in sel]
            assert dk1[i] == (min(d[i, rest]) if rest else np.inf)


def test_invariants_and_order():
    rng = np.random.default_rng(3)
    counts = [1, 2, 5, 16, 17, 18, 40, 100, 128, 0, 7]
    off = np.zeros(len(counts) + 1, np.int32); off[1:] = np.cumsum(counts)
    s = rng.normal(0, 1, (off[-1], 3))
    k = 16
    idx, dk, dk1 = oracle.knn(s, off, k)
    for b, n in enumerate(counts):
        for i in range(n):
            row = idx[off[b] + i]
            sel = row[row >= 0]
            assert sel.size == min(k, n - 1)                       # R6: k_eff
            assert (row[sel.size:] == -1).all()
            assert len(set(sel.tolist())) == sel.size and i not in sel
            assert ((sel >= 0) & (sel < n)).all()                  # jet-local, inside the jet
            d = ((s[off[b] + i] - s[off[b]:off[b + 1]]) ** 2).sum(1)
            keys = [(d[j], j) for j in sel]
            assert keys == sorted(keys)                            # (d, j) order
            rest = [(d[j], j) for j in range(n) if j != i and j not in sel]
            if rest and keys:
                assert max(keys) < min(rest)


def test_translation_invariance_exact():
    """Coordinates on a 2^-10 grid translated by an exactly representable constant: identical sets and distances."""
    rng = np.random.default_rng(5)
    s = rng.integers(-400, 400, (60, 2)) / 1024.0
    off = np.array([0, 25, 60], np.int32)
    i0, d0, e0 = oracle.knn(s, off, 16)
    i1, d1, e1 = oracle.knn(s + np.array([0.5, -0.25]), off, 16)
    assert np.array_equal(i0, i1) and np.array_equal(d0, d1) and np.array_equal(e0, e1)


def test_duplicates_are_legitimate_neighbours():
    """R4: a duplicate of particle i sits at distance 0 and is selected first (lowest (d, j))."""
    s = np.array([[0.0, 0.0], [1.0, 0.0], [0.0, 0.0], [5.0, 5.0]])
    idx, dk, _ = oracle.knn(s, np.array([0, 4], np.int32), 2)
    assert idx[0].tolist() == [2, 1] and idx[2].tolist() == [0, 1]

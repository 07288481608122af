"""TEST INFRASTRUCTURE ONLY (never imported by the product): fp64 oracle of the boosted-decision-tree workload
(section 4.1: "a small boosted decision tree (BDT) with 20 input features and 100 trees"; Table C2:
input shape 20, output shape 2).  The paper names XGBoost and prints no tree; the form below is DESIGN.md readings B1-B4:
complete binary trees of one depth, internal node i tests x[feature[i]] < threshold[i] (true -> child 2 i + 1, false or NaN
-> child 2 i + 2), margin = sum of the reached leaves, p = 1 / (1 + exp(-margin)), output (1 - p, p).

The walk is written level by level over all events at once with numpy indexing; nothing else is vectorised or reordered.
Pins (tests/test_oracle_bdt.py): a pure-Python per-event walk, the hand-worked forest of tests/golden/bdt_worked_example.txt,
depth-1 stumps as a closed form, forests whose thresholds send every event to one known leaf; predict(): the golden file's
decimal-arithmetic probabilities, scipy.special.expit, margin 0 and +-40 (column order and sign)."""
import numpy as np


def margins(feature, threshold, leaf, x):
    """feature, threshold [T, 2^d - 1]; leaf [T, 2^d]; x [N, F] -> margin [N] in fp64 (comparisons on the fp32 values)."""
    feature = np.asarray(feature); threshold = np.asarray(threshold, np.float32); leaf = np.asarray(leaf, np.float64)
    x = np.asarray(x, np.float32)
    T, n_int = feature.shape
    depth = int(np.log2(n_int + 1))
    assert (1 << depth) - 1 == n_int and leaf.shape == (T, 1 << depth)
    rows = np.arange(x.shape[0])
    m = np.zeros(x.shape[0], np.float64)
    for t in range(T):
        node = np.zeros(x.shape[0], np.int64)
        for _ in range(depth):
            goes_left = x[rows, feature[t, node]] < threshold[t, node]          # NaN -> False -> right
            node = 2 * node + np.where(goes_left, 1, 2)
        m += leaf[t, node - n_int]
    return m


def predict(feature, threshold, leaf, x):
    """[N, 2] = (1 - p, p), p = 1 / (1 + exp(-margin)), fp64."""
    p = 1.0 / (1.0 + np.exp(-margins(feature, threshold, leaf, x)))
    return np.stack([1.0 - p, p], axis=1)

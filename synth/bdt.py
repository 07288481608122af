"""Seeded synthetic forest and events for the BDT workload (20 input features, 100 trees; the paper's trained
XGBoost model is not available, so the trees are random: no arithmetic of the method lives here)."""
import numpy as np


def make_bdt(seed: int = 2001, n_trees: int = 100, depth: int = 6, n_features: int = 20):
    """feature int32 [T, 2^d - 1] ~ uniform{0..F-1}; threshold fp32 ~ N(0, 1); leaf fp32 [T, 2^d] ~ N(0, 0.1)."""
    rng = np.random.default_rng(seed)
    n_int = (1 << depth) - 1
    feature = rng.integers(0, n_features, (n_trees, n_int)).astype(np.int32)
    threshold = rng.normal(0.0, 1.0, (n_trees, n_int)).astype(np.float32)
    leaf = rng.normal(0.0, 0.1, (n_trees, 1 << depth)).astype(np.float32)
    return feature, threshold, leaf


def make_bdt_events(n: int, n_features: int = 20, seed: int = 2002) -> np.ndarray:
    """x fp32 [n, F] ~ N(0, 1) (the paper's perf_analyzer requests are randomly generated, L279)."""
    return np.random.default_rng(seed).standard_normal((n, n_features), dtype=np.float32)

"""-m gpu parity tests of the PRODUCTION kNN path (GNN_BF16 mode): the grouped kernels of csrc/knn_group.cu -- several jets
per 128-row tile, Gram distances on fp16 operands (fp32 accumulate) on the tensor cores for the feature spaces (D = 64 / 128 / 256), exact direct
differences for the coordinates, 32-bit selection keys (d to 16 mantissa bits | j) -- against the fp64 oracle's kNN,
through gnn_debug_knn on a GNN_BF16 model (which runs exactly what that model's forward runs).

BASELINE.json north_star sets no neighbour-set bar in this mode (R20), so the bars here are the ones DESIGN.md
section 2 (R28) derives from the arithmetic:
  * every point whose oracle gap (d^(k+1) - d^(k)) / d^(k+1) is >= 1e-2 (features) / >= 1e-4 (coordinates) must have the
    IDENTICAL neighbour set;
  * the overall set-mismatch rate on feature spaces shaped like x^1 / x^2 (the oracle's own block outputs of configs[1])
    stays below 1.5 % of the points (the oracle's gap distribution has ~10 % of the points below 1e-2 and ~1 % below 1e-3);
  * integer lattices are reproduced bit for bit by the coordinates kernel (integer distances below 2^16 are exact in
    16 mantissa bits); in the Gram kernel centring makes exact ties a matter of rounding noise (gap 0 = ambiguous).
"""
import os

import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2312_06838_b200 as gnn
from gpu_util import dev, make_model, compare_sets

pytestmark = pytest.mark.gpu
GOLD = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def pn():
    a = synth.ARCHS["particlenet"]
    w = synth.make_weights(a)
    return a, w, make_model(a, w, precision=gnn.BF16, max_batch_jets=1024, max_particles=128)


@pytest.fixture(scope="module")
def dumps():
    """The oracle's per-block outputs on the first 256 jets of configs[1]: spaces with the real magnitudes of x^1 / x^2."""
    a = synth.ARCHS["particlenet"]
    b = synth.make_particlenet_batch(n_jets=256)
    return b, oracle.forward(a, synth.make_weights(a), b.feats, b.coords, b.offsets, dumps=True)


def rel_gap(dk, dk1):
    with np.errstate(divide="ignore", invalid="ignore"):
        g = (dk1 - dk) / dk1
    return np.where(np.isfinite(dk1) & (dk1 > 0), g, np.where(np.isfinite(dk1), 0.0, np.inf))


def run_knn(m, space, off, k):
    idx = m.debug_knn(dev(space.astype(np.float32)), dev(off), k)
    torch.cuda.synchronize()
    assert m.status_check() == 0
    return idx.cpu().numpy()


def check_structure(idx, ref, off):
    """what is unique whatever the arithmetic: k_eff entries, -1 padding behind them, all inside the jet, none equal to i"""
    assert ((idx >= 0).sum(1) == (ref >= 0).sum(1)).all()
    n = np.repeat(np.diff(off), np.diff(off))
    i = np.arange(idx.shape[0]) - np.repeat(off[:-1], np.diff(off))
    valid = idx >= 0
    assert (np.where(valid, idx, 0) < n[:, None]).all()
    assert not (valid & (idx == i[:, None])).any()
    srt = np.sort(np.where(valid, idx, 10 ** 6 + np.arange(idx.shape[1])[None, :]), axis=1)
    assert (np.diff(srt, axis=1) > 0).all()                    # distinct


@pytest.mark.parametrize("block", [1, 2])
def test_feature_space_knn_against_oracle(pn, dumps, block, record_property):
    """kNN of block `block` + 1 on the oracle's x^block (fp64 -> fp32): identical sets at gap >= 1e-2, mismatch rate <= 1.5 %."""
    a, _, m = pn
    b, r = dumps
    space = r["x"][block - 1]
    idx = run_knn(m, space, b.offsets, a.k)
    ref, dk, dk1 = oracle.knn(space.astype(np.float32), b.offsets, a.k)
    check_structure(idx, ref, b.offsets)
    gap = rel_gap(dk, dk1)
    _, _, diff = compare_sets(idx, ref, np.zeros(len(gap), bool))
    rate = diff.mean()
    record_property("set_mismatch_rate_block%d" % (block + 1), float(rate))
    print("block %d (D = %d): %d / %d points differ (%.3f %%), largest gap among them %.2e" %
          (block + 1, space.shape[1], diff.sum(), diff.size, 100 * rate, gap[diff].max() if diff.any() else 0.0))
    assert not (diff & (gap >= 1e-2)).any(), "a point with a clear gap has a different neighbour set"
    assert rate <= 0.015


def test_coordinate_knn_against_oracle(pn):
    """Block 1 (exact direct differences, 32-bit keys): identical sets wherever the oracle's gap is >= 1e-4."""
    a, _, m = pn
    b = synth.make_particlenet_batch(n_jets=1024)
    idx = run_knn(m, b.coords, b.offsets, a.k)
    ref, dk, dk1 = oracle.knn(b.coords, b.offsets, a.k)
    check_structure(idx, ref, b.offsets)
    gap = rel_gap(dk, dk1)
    _, _, diff = compare_sets(idx, ref, np.zeros(len(gap), bool))
    print("coordinates: %d / %d points differ, largest gap among them %.2e" % (diff.sum(), diff.size, gap[diff].max() if diff.any() else 0.0))
    assert not (diff & (gap >= 1e-4)).any()
    assert diff.mean() <= 2e-3


def test_lattices_bit_exact_through_32bit_keys(pn):
    """Integer coordinates: distances are small integers, exact in fp32, in tf32 products and in 16 mantissa bits, so the
    tie-break (lower index) must come out exactly as the hand-derived sets and as the oracle's order."""
    _, _, m = pn
    for line in open(os.path.join(GOLD, "knn_lattices.txt")):
        if not line.strip() or line.startswith("#"):
            continue
        name, pts, k, q, s = [t.strip() for t in line.split("|")]
        P = np.array([[float(v) for v in p.split(",")] for p in pts.split(";")], np.float32)
        idx = run_knn(m, P, np.array([0, len(P)], np.int32), int(k))
        assert sorted(idx[int(q)].tolist()) == sorted(int(v) for v in s.split(",")), name
    rng = np.random.default_rng(0)
    off = np.array([0, 37, 37, 100, 228], np.int32)
    for D in (2, 3, 4):                                          # the coordinates kernel: order included
        P = rng.integers(0, 4, (228, D)).astype(np.float32)
        idx = run_knn(m, P, off, 16)
        ref, _, _ = oracle.knn(P, off, 16)
        assert np.array_equal(idx, ref), D
    # Gram kernel: centring makes the products inexact, so exact ties are broken by rounding noise (the oracle's gap is 0
    # there: ambiguous by definition); every point with a clear gap still has the identical set
    P = rng.integers(0, 4, (228, 64)).astype(np.float32)
    idx = run_knn(m, P, off, 16)
    ref, dk, dk1 = oracle.knn(P, off, 16)
    _, _, diff = compare_sets(idx, ref, np.zeros(228, bool))
    assert not (diff & (rel_gap(dk, dk1) >= 1e-2)).any()


@pytest.mark.parametrize("D,k", [(2, 16), (64, 16), (128, 16), (256, 16), (2, 4), (64, 4), (2, 1), (128, 2), (64, 8), (2, 32), (128, 32)])
def test_group_schedule_and_k(pn, D, k):
    """Multiplicities that stress the group schedule (runs of empty and one-particle jets longer than a group may hold,
    jets of exactly 128, a group boundary inside a chunk of 32 jets and across chunks) and every selection width."""
    _, _, m = pn
    rng = np.random.default_rng(D * 100 + k)
    counts = ([1] * 40 + [0] * 35 + [128, 128, 1, 127, 2, 126] + [3, 5, 2, 1] * 12 + [64, 64, 65, 63] +
              list(rng.integers(5, 101, 70)) + [0, 128, 0])
    off = np.zeros(len(counts) + 1, np.int32); off[1:] = np.cumsum(counts)
    s = rng.normal(0, 1, (off[-1], D)).astype(np.float32)
    if D > 8:
        s = np.maximum(s, 0)
    idx = run_knn(m, s, off, k)
    ref, dk, dk1 = oracle.knn(s, off, k)
    check_structure(idx, ref, off)
    gap = rel_gap(dk, dk1)
    _, _, diff = compare_sets(idx, ref, np.zeros(len(gap), bool))
    assert not (diff & (gap >= (1e-4 if D <= 4 else 1e-2))).any()
    assert diff.mean() <= 0.02


def test_jet_result_independent_of_group_mates(pn):
    """Per-jet centring and per-row selection: a jet's neighbours do not depend on which jets share its tile (bitwise)."""
    a, _, m = pn
    rng = np.random.default_rng(5)
    counts = list(rng.integers(5, 60, 40))
    off = np.zeros(len(counts) + 1, np.int32); off[1:] = np.cumsum(counts)
    s = np.maximum(rng.normal(0.5, 1, (off[-1], 64)), 0).astype(np.float32)
    full = run_knn(m, s, off, 16)
    for j in (0, 7, 39):
        lo, hi = off[j], off[j + 1]
        alone = run_knn(m, s[lo:hi], np.array([0, hi - lo], np.int32), 16)
        assert np.array_equal(alone, full[lo:hi])


# ---- the pooling EdgeConv epilogue (steps a6 + a7 in one kernel) -------------------------------------------------------
def test_edgeconv_pool_stage_given_oracle_indices(pn):
    """gnn_debug_edgeconv_pool: last block with the epilogue that adds the block output into per-jet channel sums instead of
    storing it.  Against mean over particles of oracle.edgeconv; and bitwise equal whatever the batch mates are."""
    a, w, m = pn
    rng = np.random.default_rng(11)
    counts = [1, 2, 17, 40, 100, 0, 5, 16, 61, 40, 40, 33, 128, 3, 0] + list(rng.integers(5, 101, 80))
    off = np.zeros(len(counts) + 1, np.int32); off[1:] = np.cumsum(counts)
    x = np.maximum(rng.normal(0, 1, (off[-1], a.block_in(2))), 0).astype(np.float32)
    idx, _, _ = oracle.knn(x, off, a.k)
    g = m.debug_edgeconv_pool(dev(x), dev(idx), dev(off)).cpu().numpy()
    assert m.status_check() == 0
    y = oracle.edgeconv(a, w, 2, x, idx, off)
    ref = np.stack([y[off[j]:off[j + 1]].mean(0) if off[j + 1] > off[j] else np.zeros(y.shape[1]) for j in range(len(counts))])
    assert np.abs(g - ref).max() < 3e-3 * max(1.0, np.abs(ref).max())
    # the stored-output kernel + plain mean gives the same numbers to fp32 rounding of the mean
    ys = m.debug_edgeconv(2, dev(x), dev(idx), dev(off)).cpu().numpy().astype(np.float64)
    ref2 = np.stack([ys[off[j]:off[j + 1]].mean(0) if off[j + 1] > off[j] else np.zeros(ys.shape[1]) for j in range(len(counts))])
    assert np.abs(g - ref2).max() < 1e-5 * max(1.0, np.abs(ref2).max())
    # batch-composition invariance of the fixed-point sums: bitwise
    sel = [3, 12, 40, 4]
    xs = np.concatenate([x[off[j]:off[j + 1]] for j in sel]); ids = np.concatenate([idx[off[j]:off[j + 1]] for j in sel])
    o2 = np.zeros(len(sel) + 1, np.int32); o2[1:] = np.cumsum([counts[j] for j in sel])
    g2 = m.debug_edgeconv_pool(dev(xs), dev(ids), dev(o2)).cpu().numpy()
    assert np.array_equal(g2, g[sel])


def test_edgeconv_large_activations_do_not_overflow_fp16(pn):
    """E3 sums the k rows of relu(D1 + t3) in packed fp16 with 1/k folded into layer 3: activations of ~1e4 (sum over 16
    rows ~1.6e5, beyond fp16) must come out finite and right to bf16 accuracy."""
    a, w, m = pn
    rng = np.random.default_rng(12)
    counts = [40, 17, 5, 64]
    off = np.zeros(len(counts) + 1, np.int32); off[1:] = np.cumsum(counts)
    x = (np.maximum(rng.normal(0, 1, (off[-1], a.block_in(1))), 0) * 4e3).astype(np.float32)
    idx, _, _ = oracle.knn(x, off, a.k)
    y = m.debug_edgeconv(1, dev(x), dev(idx), dev(off)).cpu().numpy()
    ref = oracle.edgeconv(a, w, 1, x, idx, off)
    assert np.isfinite(y).all() and np.abs(ref).max() > 5e3
    assert np.abs(y - ref).max() < 8e-3 * np.abs(ref).max()

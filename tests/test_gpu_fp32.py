"""-m gpu parity tests, GNN_FP32_VALIDATION mode: the CUDA path against the fp64 oracle, through the C ABI.
Bar (BASELINE.json north_star): neighbour sets identical except where the oracle's k-th and (k+1)-th distances differ
by < 1e-5 relative; logits within 1e-4 absolute."""
import os

import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2312_06838_b200 as gnn
from gpu_util import dev, make_model, run_ragged, ambiguous_points, compare_sets, staged_fp32

pytestmark = pytest.mark.gpu
LOGIT_TOL = 1e-4
GOLD = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def pn():
    a = synth.ARCHS["particlenet"]
    w = synth.make_weights(a)
    return a, w, make_model(a, w, max_batch_jets=1024)


@pytest.fixture(scope="module")
def tiny():
    a = synth.ARCHS["tiny"]
    w = synth.make_weights(a)
    return a, w, make_model(a, w, max_batch_jets=64)


# ---- kNN stage --------------------------------------------------------------------------------------------------
def test_knn_lattices_bit_exact(pn):
    """Integer coordinates: exact in fp32, so the tie-break (lower index) must be reproduced exactly."""
    _, _, m = pn
    for line in open(os.path.join(GOLD, "knn_lattices.txt")):
        if not line.strip() or line.startswith("#"):
            continue
        name, pts, k, q, s = [t.strip() for t in line.split("|")]
        P = np.array([[float(v) for v in p.split(",")] for p in pts.split(";")], np.float32)
        idx = m.debug_knn(dev(P), dev(np.array([0, len(P)], np.int32)), int(k)).cpu().numpy()
        assert sorted(idx[int(q)].tolist()) == sorted(int(v) for v in s.split(","))
    # the oracle agrees element by element, order included, on a lattice with many ties
    rng = np.random.default_rng(0)
    P = rng.integers(0, 4, (100, 3)).astype(np.float32)
    off = np.array([0, 37, 37, 100], np.int32)
    idx = m.debug_knn(dev(P), dev(off), 16).cpu().numpy()
    ref, _, _ = oracle.knn(P, off, 16)
    assert np.array_equal(idx, ref)


@pytest.mark.parametrize("D,k", [(2, 16), (64, 16), (128, 16), (256, 16), (5, 4), (2, 1), (7, 32)])
def test_knn_random_spaces(pn, D, k):
    _, _, m = pn
    rng = np.random.default_rng(D * 100 + k)
    counts = [1, 2, 5, 16, 17, 18, 40, 100, 127, 128, 0, 33] + list(rng.integers(5, 101, 60))
    off = np.zeros(len(counts) + 1, np.int32); off[1:] = np.cumsum(counts)
    s = rng.normal(0, 1, (off[-1], D)).astype(np.float32)
    if D > 8:
        s = np.maximum(s, 0)                                   # post-ReLU-like features
    idx = m.debug_knn(dev(s), dev(off), k).cpu().numpy()
    ref, dk, dk1 = oracle.knn(s, off, k)
    bad, flips, _ = compare_sets(idx, ref, ambiguous_points(dk, dk1))
    assert bad == 0, "neighbour sets differ outside the 1e-5 near-tie band"
    assert flips <= 3
    assert ((idx >= 0).sum(1) == (ref >= 0).sum(1)).all()      # k_eff and the -1 padding


# ---- EdgeConv and pool/head stages ------------------------------------------------------------------------------
@pytest.mark.parametrize("block", [0, 1, 2])
def test_edgeconv_stage_given_oracle_indices(pn, block):
    a, w, m = pn
    rng = np.random.default_rng(block)
    counts = [1, 2, 17, 40, 100, 5, 16, 61]
    off = np.zeros(len(counts) + 1, np.int32); off[1:] = np.cumsum(counts)
    cin = a.block_in(block)
    x = rng.normal(0, 1, (off[-1], cin)).astype(np.float32)
    idx, _, _ = oracle.knn(x, off, a.k)
    y = m.debug_edgeconv(block, dev(x), dev(idx), dev(off)).cpu().numpy()
    ref = oracle.edgeconv(a, w, block, x, idx, off)
    assert np.abs(y - ref).max() < 2e-5 * max(1.0, np.abs(ref).max())


def test_pool_head_stage(pn):
    a, w, m = pn
    rng = np.random.default_rng(9)
    counts = [3, 0, 40, 1, 128]
    off = np.zeros(len(counts) + 1, np.int32); off[1:] = np.cumsum(counts)
    x = np.maximum(rng.normal(0, 1, (off[-1], 256)), 0).astype(np.float32)
    lg = m.debug_pool_head(dev(x), dev(off)).cpu().numpy()
    ref, _ = oracle.pool_head(a, w, x, off)
    assert np.abs(lg - ref).max() < 2e-5


# ---- whole network ----------------------------------------------------------------------------------------------
def test_tiny_end_to_end(tiny):
    a, w, m = tiny
    t = synth.make_tiny()
    lg, r, report, excluded = staged_fp32(m, a, w, t)
    assert all(bad == 0 for bad, _ in report)
    assert np.abs(lg - r["logits"])[~excluded].max() < LOGIT_TOL
    direct = run_ragged(m, t)
    assert np.array_equal(direct, lg)                          # gnn_infer == the staged entry points
    assert (np.argmax(direct, 1) == np.argmax(r["logits"], 1)).all()


def test_particlenet_end_to_end_256(pn):
    a, w, m = pn
    b = synth.make_particlenet_batch(n_jets=256)
    lg, r, report, excluded = staged_fp32(m, a, w, b)
    assert all(bad == 0 for bad, _ in report), report
    assert excluded.sum() <= 3
    assert np.abs(lg - r["logits"])[~excluded].max() < LOGIT_TOL
    assert np.array_equal(run_ragged(m, b), lg)


def test_particlenet_full_batch_1024(pn):
    """BASELINE configs[1] at its full size, in the launch configuration bench.py times (one gnn_infer).  R21 to the
    letter: the staged run gives the GPU's neighbour sets of every block; a jet may miss the 1e-4 bar only if it holds
    an ambiguous point (oracle gap < 1e-5 relative) whose GPU set actually differs, and every such jet is counted."""
    a, w, m = pn
    b = synth.make_particlenet_batch()
    staged, r, report, excluded = staged_fp32(m, a, w, b)
    assert all(bad == 0 for bad, _ in report), report          # no set differs outside the near-tie band
    lg = run_ragged(m, b)
    assert np.array_equal(lg, staged)                          # gnn_infer == the staged entry points, bitwise
    err = np.abs(lg - r["logits"]).max(1)
    print("fp32 B=1024: max |dlogit| over non-excluded jets %.2e, excluded jets %d, ambiguous flips per block %s" %
          (err[~excluded].max(), excluded.sum(), [f for _, f in report]))
    assert (err[~excluded] < LOGIT_TOL).all()
    assert excluded.sum() <= 8                                 # expected ~1-2e-4 of the points per block
    assert np.median(err) < 2e-5
    assert (np.argmax(lg, 1) == np.argmax(r["logits"], 1)).all()


def test_edge_case_set(pn):
    a, w, m = pn
    b = synth.make_edge_case_batch(a.in_features)
    lg, r, report, excluded = staged_fp32(m, a, w, b)
    assert all(bad == 0 for bad, _ in report)
    assert np.abs(lg - r["logits"])[~excluded].max() < LOGIT_TOL
    assert np.array_equal(run_ragged(m, b), lg)
    for sizes in [(1,), (0,), (128,), (0, 0, 0)]:             # B = 1 and all-empty batches
        bb = synth.make_edge_case_batch(a.in_features, sizes=sizes)
        ref = oracle.forward(a, w, bb.feats, bb.coords, bb.offsets)
        assert np.abs(run_ragged(m, bb) - ref).max() < LOGIT_TOL
    big = synth.make_edge_case_batch(a.in_features, sizes=(40, 7), scale=10.0)      # |x| ~ 10
    ref = oracle.forward(a, w, big.feats, big.coords, big.offsets)
    assert np.abs(run_ragged(m, big) - ref).max() < 1e-4 * max(1.0, np.abs(ref).max())
    z = synth.make_edge_case_batch(a.in_features, sizes=(12,))
    z.feats[:] = 0                                            # all features zero
    ref = oracle.forward(a, w, z.feats, z.coords, z.offsets)
    assert np.abs(run_ragged(m, z) - ref).max() < LOGIT_TOL
    d = synth.make_edge_case_batch(a.in_features, sizes=(20,))
    d.feats[10:] = d.feats[:10]; d.coords[10:] = d.coords[:10]   # duplicate particles: exact ties at d = 0
    ref = oracle.forward(a, w, d.feats, d.coords, d.offsets)
    assert np.abs(run_ragged(m, d) - ref).max() < LOGIT_TOL


def test_batch_composition_and_permutation_invariance(pn):
    a, w, m = pn
    b = synth.make_particlenet_batch(n_jets=64)
    full = run_ragged(m, b)
    sub = b.select([5, 2, 63, 7])
    assert np.array_equal(run_ragged(m, sub), full[[5, 2, 63, 7]])         # bitwise: what makes batching legal
    rng = np.random.default_rng(0)
    f, c = b.feats.copy(), b.coords.copy()
    for j in range(b.n_jets):
        s, e = b.offsets[j], b.offsets[j + 1]
        p = rng.permutation(e - s)
        f[s:e] = b.feats[s:e][p]; c[s:e] = b.coords[s:e][p]
    perm = synth.JetBatch(f, c, b.offsets)
    assert np.abs(run_ragged(m, perm) - full).max() < 5e-5


@pytest.mark.parametrize("P,interleave,garbage", [(100, False, np.nan), (100, True, 1e9), (128, True, np.nan), (101, True, np.nan)])
def test_padded_entry_is_padding_invariant(pn, P, interleave, garbage):
    a, w, m = pn
    b = synth.make_particlenet_batch(n_jets=48)
    ref = run_ragged(m, b)
    f, c, mk = synth.pad_batch(b, P, interleave=interleave, garbage=garbage)
    out = m.infer_padded(dev(f), dev(c), dev(mk))
    torch.cuda.synchronize()
    assert m.status_check() == 0
    assert np.array_equal(out.cpu().numpy().astype(np.float64), ref)       # same kernels on the same packed rows


def test_device_side_errors(pn):
    a, w, _ = pn
    m = make_model(a, w, max_batch_jets=16, max_particles=100)
    b = synth.make_particlenet_batch(n_jets=4)
    off = b.offsets.copy(); off[2] = off[1] - 1                            # not monotone
    out = m.infer(dev(b.feats), dev(b.coords), dev(off))
    torch.cuda.synchronize()
    assert torch.isnan(out).all()
    assert m.status_check() == -6 and m.status_check() == 0                 # sticky, then cleared
    big = synth.make_edge_case_batch(a.in_features, sizes=(10, 101, 12))   # 101 > max_particles = 100
    out = m.infer(dev(big.feats), dev(big.coords), dev(big.offsets)).cpu().numpy()
    assert m.status_check() == -7
    assert np.isnan(out[1]).all() and np.isfinite(out[[0, 2]]).all()
    ref = oracle.forward(a, w, big.feats, big.coords, big.offsets)
    assert np.abs(out[[0, 2]] - ref[[0, 2]]).max() < LOGIT_TOL               # batch mates are untouched
    ok = m.infer(dev(b.feats), dev(b.coords), dev(b.offsets))               # a good batch afterwards is clean
    torch.cuda.synchronize()
    assert torch.isfinite(ok).all() and m.status_check() == 0
    with pytest.raises(gnn.GnnError) as e:
        bb = synth.make_particlenet_batch(n_jets=17)
        m.infer(dev(bb.feats), dev(bb.coords), dev(bb.offsets))
    assert e.value.code == -4

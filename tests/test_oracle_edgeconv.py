"""Pins for the oracle's EdgeConv block and pool+head (oracle.c edgeconv_jet / pool_head_jet).  CPU only.
Each special case reduces the block to a textbook / library routine so that a dropped term, wrong sign, wrong
index or transposed operand in the oracle fails at least one of them."""
import numpy as np
import pytest
import oracle
import synth
from synth.arch import Arch
from np_restatement import split_blob


def _views(a, blob):
    """Writable views into the blob, in blob order (restated from include/gnn.h, not imported from anywhere)."""
    out, o = [], 0
    for l, (c1, c2, c3) in enumerate(a.channels):
        cin = a.block_in(l)
        blk = {}
        for name, (i, w) in zip(("l1", "l2", "l3"), ((2 * cin, c1), (c1, c2), (c2, c3))):
            blk[name] = (blob[o:o + w * i].reshape(w, i), blob[o + w * i:o + w * i + w], blob[o + w * i + w:o + w * i + 2 * w])
            o += w * i + 2 * w
        blk["sc"] = (blob[o:o + c3 * cin].reshape(c3, cin), blob[o + c3 * cin:o + c3 * cin + c3],
                     blob[o + c3 * cin + c3:o + c3 * cin + 2 * c3])
        o += c3 * cin + 2 * c3
        out.append(blk)
    return out


A = Arch(in_features=5, k=4, channels=((12, 10, 14),), fc_hidden=(6,), n_classes=3, max_particles=32)


def _dense_block(blk, x):
    h = x
    for name in ("l1", "l2", "l3"):
        W, s, t = [np.asarray(v, np.float64) for v in blk[name]]
        h = np.maximum((h @ W.T) * s + t, 0.0)
    return h


def test_zeroed_difference_half_is_a_dense_mlp():
    """(i) zero W1[:, C_in:]: output is independent of the neighbours = per-particle dense MLP (numpy matmul)."""
    rng = np.random.default_rng(1)
    blob = synth.make_weights(A, 3)
    blk = _views(A, blob)[0]
    blk["l1"][0][:, 5:] = 0.0
    x = rng.normal(0, 1, (9, 5)); off = np.array([0, 9], np.int32)
    idx, _, _ = oracle.knn(rng.normal(0, 1, (9, 2)), off, A.k)
    y = oracle.edgeconv(A, blob, 0, x, idx, off)
    W1 = np.asarray(blk["l1"][0], np.float64)
    e = np.concatenate([x, np.zeros_like(x)], 1)
    h = np.maximum((e @ W1.T) * blk["l1"][1] + blk["l1"][2], 0)
    for name in ("l2", "l3"):
        W, s, t = [np.asarray(v, np.float64) for v in blk[name]]
        h = np.maximum((h @ W.T) * s + t, 0)
    Ws, ss, ts = [np.asarray(v, np.float64) for v in blk["sc"]]
    ref = np.maximum(h + (x @ Ws.T) * ss + ts, 0)
    assert np.allclose(y, ref, rtol=0, atol=1e-12)


def test_identical_particles():
    """(ii) all particles equal: x_j - x_i = 0, same reduction with unmodified weights."""
    blob = synth.make_weights(A, 4)
    blk = _views(A, blob)[0]
    x0 = np.random.default_rng(2).normal(0, 1, 5)
    x = np.tile(x0, (7, 1)); off = np.array([0, 7], np.int32)
    idx, _, _ = oracle.knn(x, off, A.k)
    y = oracle.edgeconv(A, blob, 0, x, idx, off)
    e = np.concatenate([x, np.zeros_like(x)], 1)
    h = _dense_block(blk, e)
    Ws, ss, ts = [np.asarray(v, np.float64) for v in blk["sc"]]
    ref = np.maximum(h + (x @ Ws.T) * ss + ts, 0)
    assert np.allclose(y, ref, rtol=0, atol=1e-12)


def test_transparent_relus_closed_form():
    """(iii) scale=1, shift=0, W2=W3=I, W1a >= W1b >= 0, x >= 0, Ws >= 0: every ReLU is transparent and
    y_i = W1a x_i + W1b (centroid(N_i) - x_i) + Ws x_i.  Rectangular, asymmetric W1 catches transpositions."""
    a = Arch(in_features=5, k=3, channels=((8, 8, 8),), fc_hidden=(), n_classes=2)
    rng = np.random.default_rng(6)
    blob = np.zeros(synth.weight_count(a), np.float32)
    blk = _views(a, blob)[0]
    W1b = rng.uniform(0, 1, (8, 5)); W1a = W1b + rng.uniform(0, 1, (8, 5))
    blk["l1"][0][:, :5] = W1a; blk["l1"][0][:, 5:] = W1b
    for name in ("l1", "l2", "l3", "sc"):
        blk[name][1][:] = 1.0; blk[name][2][:] = 0.0
    blk["l2"][0][:] = np.eye(8); blk["l3"][0][:] = np.eye(8)
    blk["sc"][0][:] = rng.uniform(0, 1, (8, 5))
    W1a = blk["l1"][0][:, :5].astype(np.float64); W1b = blk["l1"][0][:, 5:].astype(np.float64)
    Ws = blk["sc"][0].astype(np.float64)
    x = rng.uniform(0, 2, (11, 5)); off = np.array([0, 11], np.int32)
    idx, _, _ = oracle.knn(x[:, :2], off, a.k)
    y = oracle.edgeconv(a, blob, 0, x, idx, off)
    cen = x[idx].mean(1)
    ref = x @ W1a.T + (cen - x) @ W1b.T + x @ Ws.T
    assert np.allclose(y, ref, rtol=0, atol=1e-12)


def test_folded_equals_unfolded():
    """(iv) folding scale into W (W' = diag(scale) W, scale' = 1) changes nothing beyond rounding (R8)."""
    a = synth.ARCHS["tiny"]
    blob = synth.make_weights(a, 0)
    t = synth.make_tiny(n_jets=4)
    ref = oracle.forward(a, blob, t.feats, t.coords, t.offsets)
    folded = blob.astype(np.float64)
    o = 0
    cin = a.in_features
    for (i, w) in ((2 * cin, 32), (32, 32), (32, 32), (cin, 32)):
        W = folded[o:o + w * i].reshape(w, i); s = folded[o + w * i:o + w * i + w]
        W *= s[:, None]; s[:] = 1.0
        o += w * i + 2 * w
    got = oracle.forward(a, folded.astype(np.float32), t.feats, t.coords, t.offsets)
    assert np.allclose(got, ref, rtol=0, atol=2e-6)      # fp32 rounding of the folded blob only


def test_all_pairs_special_case_and_single_particle():
    """k = n-1: every other particle is a neighbour, EdgeConv is an all-pairs mean that needs no kNN code (R6);
    n = 1: no neighbours, x = ReLU(shortcut)."""
    a = Arch(in_features=5, k=6, channels=((12, 10, 14),), fc_hidden=(), n_classes=2)
    blob = synth.make_weights(a, 9)
    blk = _views(a, blob)[0]
    rng = np.random.default_rng(8)
    n = 7
    x = rng.normal(0, 1, (n, 5)); off = np.array([0, n], np.int32)
    idx, _, _ = oracle.knn(rng.normal(0, 1, (n, 2)), off, a.k)
    y = oracle.edgeconv(a, blob, 0, x, idx, off)
    Ws, ss, ts = [np.asarray(v, np.float64) for v in blk["sc"]]
    for i in range(n):
        others = [j for j in range(n) if j != i]
        e = np.concatenate([np.tile(x[i], (n - 1, 1)), x[others] - x[i]], 1)
        ref = np.maximum(_dense_block(blk, e).mean(0) + (Ws @ x[i]) * ss + ts, 0)
        assert np.allclose(y[i], ref, rtol=0, atol=1e-12)
    # fewer than k others (n = 4 < k+1): mean divides by k_eff = 3
    n = 4
    x = rng.normal(0, 1, (n, 5)); off = np.array([0, n], np.int32)
    idx, _, _ = oracle.knn(x, off, a.k)
    assert (idx[:, 3:] == -1).all()
    y = oracle.edgeconv(a, blob, 0, x, idx, off)
    for i in range(n):
        others = [j for j in range(n) if j != i]
        e = np.concatenate([np.tile(x[i], (n - 1, 1)), x[others] - x[i]], 1)
        ref = np.maximum(_dense_block(blk, e).mean(0) + (Ws @ x[i]) * ss + ts, 0)
        assert np.allclose(y[i], ref, rtol=0, atol=1e-12)
    # n = 1
    x = rng.normal(0, 1, (1, 5)); off = np.array([0, 1], np.int32)
    idx, _, _ = oracle.knn(x, off, a.k)
    assert (idx == -1).all()
    y = oracle.edgeconv(a, blob, 0, x, idx, off)
    assert np.allclose(y[0], np.maximum((Ws @ x[0]) * ss + ts, 0), rtol=0, atol=1e-13)


def test_pool_head_is_mean_and_matmul():
    a = synth.ARCHS["particlenet"]
    blob = synth.make_weights(a, 0)
    _, fcs = split_blob(a, blob)
    rng = np.random.default_rng(4)
    counts = [3, 0, 40, 1]
    off = np.zeros(5, np.int32); off[1:] = np.cumsum(counts)
    x = rng.normal(0, 1, (off[-1], 256))
    logits, g = oracle.pool_head(a, blob, x, off)
    for b, n in enumerate(counts):
        gb = x[off[b]:off[b + 1]].mean(0) if n else np.zeros(256)      # R12
        z = np.maximum(fcs[0][0] @ gb + fcs[0][1], 0)
        z = fcs[1][0] @ z + fcs[1][1]
        assert np.allclose(g[b], gb, rtol=0, atol=1e-13)
        assert np.allclose(logits[b], z, rtol=0, atol=1e-12)

"""Pins for the whole oracle forward: independent numpy restatement, the survey's probe values, and the
invariances BASELINE.json north_star requires (permutation, padding) plus batch composition.  CPU only."""
import os
import numpy as np
import pytest
import oracle
import synth
from np_restatement import forward_np

GOLD = {}
for _line in open(os.path.join(os.path.dirname(__file__), "golden", "survey_probe_values.txt")):
    if _line.strip() and not _line.startswith("#"):
        _k, _v = _line.split("|")
        GOLD[_k.strip()] = np.array([float(t) for t in _v.split()])


def test_generator_is_the_normative_one():
    t = synth.make_tiny()
    assert np.allclose(t.coords[:3].ravel(), GOLD["tiny_jet0_coords"], atol=1e-6)
    assert synth.make_particlenet_batch(n_jets=128).n_particles == int(GOLD["pn128_n_particles"][0])
    for name, n in (("particlenet", 366146), ("wide", 1453186), ("tiny", 2754)):
        assert synth.weight_count(synth.ARCHS[name]) == n == oracle.blob_count(synth.ARCHS[name])


def test_tiny_matches_survey_probe_and_numpy_restatement():
    a = synth.ARCHS["tiny"]; w = synth.make_weights(a); t = synth.make_tiny()
    r = oracle.forward(a, w, t.feats, t.coords, t.offsets, dumps=True)
    lg = r["logits"]
    assert np.allclose(lg[0], GOLD["tiny_logits_jet0"], atol=2e-5)
    assert np.allclose(lg[31], GOLD["tiny_logits_jet31"], atol=2e-5)
    assert np.allclose(lg.mean(0), GOLD["tiny_logits_mean"], atol=2e-5)
    assert np.allclose(lg.std(0), GOLD["tiny_logits_std"], atol=2e-5)
    for i in range(4):
        assert sorted(r["nbr"][0, i].tolist()) == GOLD["tiny_jet0_nbr%d" % i].astype(int).tolist()
    assert np.allclose(lg, forward_np(a, w, t.feats, t.coords, t.offsets), rtol=0, atol=1e-10)


def test_particlenet_matches_survey_probe_and_numpy_restatement():
    a = synth.ARCHS["particlenet"]; w = synth.make_weights(a); b = synth.make_particlenet_batch(n_jets=128)
    lg = oracle.forward(a, w, b.feats, b.coords, b.offsets)
    assert np.allclose(lg.mean(0), GOLD["pn128_logits_mean"], atol=2e-4)
    assert np.allclose(lg.std(0), GOLD["pn128_logits_std"], atol=2e-4)
    gap = lg[:, 0] - lg[:, 1]
    assert np.allclose([gap.mean(), gap.std()], GOLD["pn128_gap_mean_std"], atol=1e-3)
    sub = b.head(6)
    assert np.allclose(lg[:6], forward_np(a, w, sub.feats, sub.coords, sub.offsets), rtol=0, atol=1e-10)


def test_wide_matches_survey_probe():
    a = synth.ARCHS["wide"]; w = synth.make_weights(a); b = synth.make_sweep_batch(n_jets=12)
    lg = oracle.forward(a, w, b.feats, b.coords, b.offsets)
    assert np.allclose(lg.mean(0), GOLD["wide12_logits_mean"], atol=2e-4)


def test_permutation_invariance():
    """north_star: logits invariant under particle reordering (no exact ties with continuous inputs, R5)."""
    a = synth.ARCHS["particlenet"]; w = synth.make_weights(a); b = synth.make_particlenet_batch(n_jets=6)
    ref = oracle.forward(a, w, b.feats, b.coords, b.offsets)
    rng = np.random.default_rng(0)
    f, c = b.feats.copy(), b.coords.copy()
    for j in range(b.n_jets):
        s, e = b.offsets[j], b.offsets[j + 1]
        p = rng.permutation(e - s)
        f[s:e] = b.feats[s:e][p]; c[s:e] = b.coords[s:e][p]
    got = oracle.forward(a, w, f, c, b.offsets)
    assert np.abs(got - ref).max() < 1e-11


@pytest.mark.parametrize("P,interleave,garbage", [(None, False, np.nan), (None, True, 1e9), (100, True, np.nan),
                                                  (128, True, np.nan), (128, False, 1e9)])
def test_padding_invariance(P, interleave, garbage):
    """north_star: extra masked particles must not change the output (R7) -- bitwise in the oracle."""
    a = synth.ARCHS["particlenet"]; w = synth.make_weights(a); b = synth.make_particlenet_batch(n_jets=5)
    ref = oracle.forward(a, w, b.feats, b.coords, b.offsets)
    P = P or int(b.counts().max()) + 1
    f, c, m = synth.pad_batch(b, P, interleave=interleave, garbage=garbage)
    got = oracle.forward_padded(a, w, f, c, m)
    assert np.array_equal(got, ref)


def test_batch_composition_invariance():
    """What makes dynamic batching legal: a jet's logits do not depend on its batch mates."""
    a = synth.ARCHS["particlenet"]; w = synth.make_weights(a); b = synth.make_particlenet_batch(n_jets=8)
    ref = oracle.forward(a, w, b.feats, b.coords, b.offsets)
    sub = b.select([5, 2, 7])
    got = oracle.forward(a, w, sub.feats, sub.coords, sub.offsets)
    assert np.array_equal(got, ref[[5, 2, 7]])
    assert np.array_equal(oracle.forward(a, w, b.feats, b.coords, b.offsets, nthreads=1), ref)   # thread count


def test_edge_case_set_runs_and_empty_jet_is_head_of_zero():
    a = synth.ARCHS["particlenet"]; w = synth.make_weights(a)
    b = synth.make_edge_case_batch(a.in_features, sizes=(0, 1, 2, 3, 16, 17, 0))
    r = oracle.forward(a, w, b.feats, b.coords, b.offsets, dumps=True)
    assert np.isfinite(r["logits"]).all()
    assert np.array_equal(r["logits"][0], r["logits"][6])          # both empty: head(0) (R12)
    zero_logits, _ = oracle.pool_head(a, w, np.zeros((0, 256)), np.array([0, 0], np.int32))
    assert np.array_equal(r["logits"][0], zero_logits[0])
    ref = forward_np(a, w, b.feats, b.coords, b.offsets)
    assert np.allclose(r["logits"], ref, rtol=0, atol=1e-10)


def test_softmax_against_library_and_closed_form():
    """oracle.softmax (SURVEY 8(f) variants): scipy's routine, rows summing to one, the two-class closed form
    p_0 = 1 / (1 + exp(z_1 - z_0)), shift invariance."""
    from scipy.special import softmax as sp_softmax
    rng = np.random.default_rng(3)
    z = rng.normal(0, 5, (200, 2))
    p = oracle.softmax(z)
    assert np.abs(p - sp_softmax(z, axis=1)).max() < 1e-14
    assert np.abs(p.sum(1) - 1).max() < 1e-14
    assert np.abs(p[:, 0] - 1.0 / (1.0 + np.exp(z[:, 1] - z[:, 0]))).max() < 1e-13
    assert np.abs(oracle.softmax(z + 1000.0) - p).max() < 1e-12
    z5 = rng.normal(0, 3, (50, 5))
    assert np.abs(oracle.softmax(z5) - sp_softmax(z5, axis=1)).max() < 1e-14

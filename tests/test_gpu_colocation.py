"""-m gpu test of multi-model co-location (section 4.3, Figs. 10-11: several models
served from one GPU at once).  Four models of the ParticleNet shape with DIFFERENT weights (seeds 0-3), each behind its own
batcher and stream, are loaded at the same time by their own client threads.  Sharing the device must not leak anything
between them: every ticket of every model is bitwise what that model returns alone, and within the bf16 bars (5e-2 absolute,
argmax) of the fp64 oracle run with THAT model's weights."""
import threading

import numpy as np
import pytest

import oracle
import synth
import paper_2312_06838_b200 as gnn
from gpu_util import make_model, run_ragged

pytestmark = pytest.mark.gpu
N_MODELS, CLIENTS_PER_MODEL, ROUNDS = 4, 4, 6


def test_colocated_models_return_their_own_logits():
    a = synth.ARCHS["particlenet"]
    weights = [synth.make_weights(a, seed=s) for s in range(N_MODELS)]
    assert not np.array_equal(weights[0], weights[1])
    models = [make_model(a, w, precision=gnn.BF16, max_batch_jets=1024, slices=2, max_particles=100) for w in weights]
    # every (model, client) pair walks its own requests of 16 jets
    pools = [[synth.make_client_pool(10 * i + c, n_requests=ROUNDS) for c in range(CLIENTS_PER_MODEL)] for i in range(N_MODELS)]
    solo = [[[run_ragged(models[i], r) for r in pools[i][c]] for c in range(CLIENTS_PER_MODEL)] for i in range(N_MODELS)]
    # the oracle with each model's own weights, on the first client's requests
    for i in range(N_MODELS):
        for r, lg in zip(pools[i][0], solo[i][0]):
            ref = oracle.forward(a, weights[i], r.feats, r.coords, r.offsets)
            assert np.abs(lg - ref).max() < 5e-2
            assert (lg.argmax(1) == ref.argmax(1)).all() or np.abs(ref[:, 0] - ref[:, 1]).min() < 0.1
    # the same requests through model 0 and model 1 differ: the models really are different functions
    assert np.abs(run_ragged(models[1], pools[0][0][0]) - solo[0][0][0]).max() > 1e-2
    batchers = [gnn.Batcher(m, max_batch_jets=1024, max_queue_delay_us=500, n_instances=2) for m in models]
    errors, done = [], []
    start = threading.Barrier(N_MODELS * CLIENTS_PER_MODEL)

    def client(i, c):
        try:
            start.wait(30)
            for rnd, r in enumerate(pools[i][c]):
                t, out = batchers[i].submit(r.feats, r.coords, r.offsets)
                rc, _, _ = batchers[i].wait(t)
                assert rc == 0, rc
                assert np.array_equal(out.astype(np.float64), solo[i][c][rnd]), (i, c, rnd)
            done.append((i, c))
        except Exception as e:                                             # noqa: BLE001
            errors.append(repr(e))

    th = [threading.Thread(target=client, args=(i, c)) for i in range(N_MODELS) for c in range(CLIENTS_PER_MODEL)]
    [t.start() for t in th]
    [t.join(180) for t in th]
    assert not errors, errors[:3]
    assert len(done) == N_MODELS * CLIENTS_PER_MODEL
    for i, b in enumerate(batchers):
        st = b.stats()
        assert st["n_requests"] == CLIENTS_PER_MODEL * ROUNDS and st["n_jets"] == CLIENTS_PER_MODEL * ROUNDS * 16
        b.close()
    for m in models:
        m.close()

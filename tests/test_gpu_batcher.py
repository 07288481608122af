"""-m gpu tests of the host dynamic batcher (PAPER.md L53 dynamic batching): results independent of coalescing,
every ticket completes exactly once, deadline honoured."""
import threading
import time

import numpy as np
import pytest
import torch

import synth
import paper_2312_06838_b200 as gnn
from gpu_util import make_model, run_ragged

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def served():
    a = synth.ARCHS["particlenet"]
    w = synth.make_weights(a)
    m = make_model(a, w, max_batch_jets=1024, slices=3, max_particles=100)
    return a, w, m


def test_tickets_equal_direct_inference(served):
    a, w, m = served
    pool = synth.make_client_pool(0, n_requests=12)
    direct = [run_ragged(m, r) for r in pool]
    bt = gnn.Batcher(m, max_batch_jets=64, max_queue_delay_us=2000, n_instances=2)
    tickets = [bt.submit(r.feats, r.coords, r.offsets) for r in pool]
    for (t, out), ref in zip(tickets, direct):
        rc, q_us, c_us = bt.wait(t)
        assert rc == 0 and q_us >= 0 and c_us > 0
        assert np.array_equal(out.astype(np.float64), ref)                 # bitwise: batch-composition invariance
    st = bt.stats()
    assert st["n_requests"] == 12 and st["n_jets"] == 12 * 16 and 1 <= st["n_launches"] <= 12
    assert bt.wait(tickets[0][0])[0] == -11                                # already collected
    bt.close()


def test_many_client_threads_no_lost_or_duplicated_tickets(served):
    a, w, m = served
    bt = gnn.Batcher(m, max_batch_jets=1024, max_queue_delay_us=1000, n_instances=3)
    n_clients, n_rounds = 32, 6
    pools = [synth.make_client_pool(c, n_requests=n_rounds) for c in range(n_clients)]
    refs = [[run_ragged(m, r) for r in p] for p in pools[:4]]
    errors, done = [], [0] * n_clients

    def client(c):
        try:
            for i, r in enumerate(pools[c]):
                t, out = bt.submit(r.feats, r.coords, r.offsets)
                rc, _, _ = bt.wait(t)
                assert rc == 0
                assert np.isfinite(out).all()
                if c < 4:
                    assert np.array_equal(out.astype(np.float64), refs[c][i])
                done[c] += 1
        except Exception as e:                                             # noqa: BLE001
            errors.append(repr(e))

    th = [threading.Thread(target=client, args=(c,)) for c in range(n_clients)]
    [t.start() for t in th]
    [t.join(120) for t in th]
    assert not errors, errors[:3]
    assert done == [n_rounds] * n_clients
    st = bt.stats()
    assert st["n_requests"] == n_clients * n_rounds
    assert st["mean_batch_jets"] > 16                                      # requests really were coalesced
    bt.close()


def test_deadline_and_host_validation(served):
    a, w, m = served
    bt = gnn.Batcher(m, max_batch_jets=1024, max_queue_delay_us=1000, n_instances=1)
    r = synth.make_client_pool(1, n_requests=1)[0]
    bt.wait(bt.submit(r.feats, r.coords, r.offsets)[0])                    # warm
    t0 = time.perf_counter()
    t, out = bt.submit(r.feats, r.coords, r.offsets)
    rc, q_us, c_us = bt.wait(t)
    dt = time.perf_counter() - t0
    assert rc == 0 and 900 <= q_us < 20000 and dt < 0.1                    # idle GPU: delay + one forward
    bad = r.offsets.copy(); bad[3] = bad[2] - 1
    with pytest.raises(gnn.GnnError) as e:
        bt.submit(r.feats, r.coords, bad)
    assert e.value.code == -6
    big = synth.make_edge_case_batch(a.in_features, sizes=(101,))
    with pytest.raises(gnn.GnnError) as e:
        bt.submit(big.feats, big.coords, big.offsets)
    assert e.value.code == -7
    rc, _, _ = bt.wait(bt.submit(r.feats, r.coords, r.offsets)[0], timeout_us=0)
    assert rc in (0, -9)
    bt.close()                                                             # drains the pending ticket


def test_request_time_split_and_load_generator(served):
    """gnn_batcher_wait_ex: the device-side parts (host <-> device copies, forward; CUDA events on the instance's stream) lie
    inside the host-clock compute time; gnn_loadgen_run: closed-loop native clients, every request of the pool answered, the
    reported split consistent (queue / network / inference per request)."""
    a, w, m = served
    bt = gnn.Batcher(m, max_batch_jets=256, max_queue_delay_us=500, n_instances=2)
    r = synth.make_client_pool(3, n_requests=1)[0]
    t, out = bt.submit(r.feats, r.coords, r.offsets)
    rc, tm = bt.wait_ex(t)
    assert rc == 0 and np.array_equal(out.astype(np.float64), run_ragged(m, r))
    assert tm["transfer_us"] > 0 and tm["inference_us"] > 0
    assert tm["transfer_us"] + tm["inference_us"] <= tm["compute_us"] * 1.05 + 20
    assert 400 <= tm["queue_us"] < 50000                                   # one lonely request waits out the queue delay
    big = synth.make_particlenet_batch(seed=77, n_jets=512)
    rfj = np.arange(0, 513, 16, dtype=np.int32)
    res = bt.loadgen(big.feats, big.coords, big.offsets, rfj, n_clients=8, warmup_ms=50, run_ms=300)
    assert res["n_requests"] > 50 and res["n_jets"] == 16 * res["n_requests"]
    assert res["p50_us"] <= res["p90_us"] <= res["p99_us"]
    assert abs(res["queue_us_mean"] + res["compute_us_mean"] - res["mean_us"]) < 0.25 * res["mean_us"] + 50
    assert 0 < res["transfer_us_mean"] + res["inference_us_mean"] <= res["compute_us_mean"] * 1.05 + 20
    assert 16 <= res["mean_batch_jets"] <= 256
    bt.close()

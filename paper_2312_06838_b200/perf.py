"""perf_analyzer-style measurement of the batcher (App. C, Table C2 / Fig. C3) and the multi-model
co-location experiment (section 4.3, Figs. 10-11), on top of the library's native closed-loop load
generator (gnn_loadgen_run).  Host-side orchestration only: every inference runs through gnn_batcher / gnn_infer_slice.

The paper scanned concurrency 1-4 (simultaneous synchronous requests) x batch size {128, 256, 512, 1024} for ParticleNet
and split the request time into network latency, inference time and queue time, each normalised by the number of FP32
inputs of a request (inputs per item x batch size).  Here the "network" is PCIe: the host <-> device copies of the
coalesced batch (gnn_request_times.transfer_us).
"""
import threading

import numpy as np

from . import binding as gnn


def normalised_us(time_us: float, inputs_per_item: int, batch: int) -> float:
    """Time per FP32 input ("a BDT with 25 FP32 inputs, batch size of 500, and a total network latency of
    14,800 us, would have a normalized value of 1.184 us")."""
    return float(time_us) / (float(inputs_per_item) * float(batch))


def request_pool(batch, jets_per_request: int):
    """Cuts one ragged JetBatch into requests of `jets_per_request` consecutive jets: the request_first_jet array of
    gnn_loadgen_pool (a trailing remainder is dropped)."""
    n_req = batch.n_jets // jets_per_request
    return np.arange(n_req + 1, dtype=np.int32) * jets_per_request


def sweep(model, batch, inputs_per_item: int, batch_sizes=(128, 256, 512, 1024), concurrencies=(1, 2, 3, 4),
          n_instances: int = 1, max_queue_delay_us: int = 1000, warmup_ms: int = 200, run_ms: int = 800):
    """One row per (batch size, concurrency): requests of `batch size` jets, `concurrency` synchronous clients, the batcher
    at max_batch_jets = max(batch_sizes) (the paper's preferred batch size, L268)."""
    rows = []
    for bs in batch_sizes:
        rfj = request_pool(batch, bs)
        for conc in concurrencies:
            bt = gnn.Batcher(model, max_batch_jets=max(batch_sizes), max_queue_delay_us=max_queue_delay_us, n_instances=n_instances)
            r = bt.loadgen(batch.feats, batch.coords, batch.offsets, rfj, min(conc, rfj.size - 1), warmup_ms, run_ms)
            bt.close()
            total = r["mean_us"]
            row = {"batch": bs, "concurrency": conc, "jets_per_s": r["jets_per_s"], "requests": int(r["n_requests"]),
                   "total_us": total, "p50_us": r["p50_us"], "p99_us": r["p99_us"], "queue_us": r["queue_us_mean"],
                   "transfer_us": r["transfer_us_mean"], "inference_us": r["inference_us_mean"],
                   "mean_coalesced_batch_jets": r["mean_batch_jets"]}
            for k in ("queue", "transfer", "inference"):
                row[k + "_us_per_input"] = normalised_us(row[k + "_us"], inputs_per_item, bs)
                row[k + "_fraction"] = row[k + "_us"] / total if total > 0 else 0.0
            rows.append(row)
    return rows


def colocation(make_model, batch, n_models=(1, 2, 4, 8), clients_per_model: int = 16, jets_per_request: int = 64,
               warmup_ms: int = 300, run_ms: int = 1000):
    """PAPER.md section 4.3 on one GPU: n models of the same architecture with different weights ("background models"), each
    behind its own batcher instance and stream, all loaded at once by their own closed-loop clients.  Returns per n: the
    aggregate jets/s, the per-model jets/s and the ratio of the per-model mean to throughput(1) / n (the 1/n law of Fig. 10:
    1.0 = the models share the device exactly; the paper saw it break by memory thrashing on a MIG slice, here the question
    is SM contention on a whole B200).  make_model(i) -> gnn.Model with weights of seed i."""
    rfj = request_pool(batch, jets_per_request)
    out = []
    base = None
    for n in n_models:
        models = [make_model(i) for i in range(n)]
        batchers = [gnn.Batcher(m, max_batch_jets=1024, max_queue_delay_us=1000, n_instances=1) for m in models]
        res = [None] * n

        def run(i):
            res[i] = batchers[i].loadgen(batch.feats, batch.coords, batch.offsets, rfj, clients_per_model, warmup_ms, run_ms)

        th = [threading.Thread(target=run, args=(i,)) for i in range(n)]
        for t in th:
            t.start()
        for t in th:
            t.join()
        for b in batchers:
            b.close()
        for m in models:
            m.close()
        per = [r["jets_per_s"] for r in res]
        if base is None:
            base = per[0]
        out.append({"n_models": n, "aggregate_jets_per_s": float(sum(per)), "per_model_jets_per_s": per,
                    "per_model_p50_us": [r["p50_us"] for r in res],
                    "per_model_over_one_nth": float(np.mean(per)) / (base / n)})
    return out

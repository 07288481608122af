// loadgen.cu -- closed-loop load generator for the host dynamic batcher (host code only).
//
// PAPER.md L279 (App. C): the paper measures its server with perf_analyzer in synchronous mode -- every client sends a
// request, waits for the answer, sends the next -- at a given concurrency and batch size, and splits the request time
// into queue and compute (Fig. C3).  This is that client side for BASELINE.json configs[3] (64 request streams x 16 jets)
// and for the concurrency x batch sweep of Table C2: n_clients native threads, each cycling through its own requests of a
// caller-supplied pool, submit -> wait -> next, against a gnn_batcher.  Native threads, so the numbers are the batcher's
// and the GPU's, not an interpreter's.
#include "gnn_internal.h"
#include <algorithm>
#include <atomic>
#include <chrono>
#include <thread>

namespace {

using Clock = std::chrono::steady_clock;

struct ClientLog {
    std::vector<float> total_us, queue_us, compute_us;
    double transfer_us = 0.0, inference_us = 0.0;
    uint64_t jets = 0;
    int status = GNN_OK;
};

double percentile(std::vector<float>& v, double q) {
    if (v.empty()) return 0.0;
    const size_t i = std::min(v.size() - 1, (size_t)(q * (double)(v.size() - 1) + 0.5));
    std::nth_element(v.begin(), v.begin() + i, v.end());
    return v[i];
}

}  // namespace

extern "C" int gnn_loadgen_run(gnn_batcher* b, const gnn_loadgen_pool* pool, const gnn_loadgen_opts* opts,
                               gnn_loadgen_result* out) {
    if (!b || !pool || !opts || !out) return GNN_ERR_NULL;
    if (!pool->offsets_host || !pool->request_first_jet || pool->n_requests < 1 || pool->n_classes < 1 ||
        pool->in_features < 1 || pool->coord_dims < 1)
        return GNN_ERR_BAD_ARG;
    if (opts->n_clients < 1 || opts->n_clients > pool->n_requests || opts->run_ms < 1 || opts->warmup_ms < 0) return GNN_ERR_BAD_ARG;
    const int nc = opts->n_clients;
    std::vector<ClientLog> logs(nc);
    std::atomic<int> phase{0};                  // 0 warm-up, 1 measured, 2 stop
    auto client = [&](int c) {
        ClientLog& L = logs[c];
        // this client's requests: c, c + nc, c + 2 nc, ... of the pool
        std::vector<int32_t> rel;
        std::vector<float> logits;
        for (int r = c;; r += nc) {
            if (r >= pool->n_requests) r = c;
            const int ph = phase.load(std::memory_order_acquire);
            if (ph == 2) break;
            const int j0 = pool->request_first_jet[r], j1 = pool->request_first_jet[r + 1];
            const int nj = j1 - j0, p0 = pool->offsets_host[j0];
            rel.resize(nj + 1);
            for (int j = 0; j <= nj; ++j) rel[j] = pool->offsets_host[j0 + j] - p0;
            logits.resize((size_t)nj * pool->n_classes);
            const auto t0 = Clock::now();
            gnn_ticket tk;
            int rc = gnn_batcher_submit(b, pool->feats_host + (size_t)p0 * pool->in_features,
                                        pool->coords_host + (size_t)p0 * pool->coord_dims, rel.data(), nj, logits.data(), &tk);
            gnn_request_times tm{};
            if (rc == GNN_OK) rc = gnn_batcher_wait_ex(b, tk, -1, &tm);
            const auto t1 = Clock::now();
            if (rc != GNN_OK) { L.status = rc; break; }
            if (ph == 1 && phase.load(std::memory_order_acquire) == 1) {
                L.total_us.push_back(std::chrono::duration<float, std::micro>(t1 - t0).count());
                L.queue_us.push_back((float)tm.queue_us);
                L.compute_us.push_back((float)tm.compute_us);
                L.transfer_us += tm.transfer_us; L.inference_us += tm.inference_us;
                L.jets += (uint64_t)nj;
            }
        }
    };
    uint64_t req0 = 0, jets0 = 0, launches0 = 0, req1 = 0, jets1 = 0, launches1 = 0;
    std::vector<std::thread> th;
    th.reserve(nc);
    for (int c = 0; c < nc; ++c) th.emplace_back(client, c);
    std::this_thread::sleep_for(std::chrono::milliseconds(opts->warmup_ms));
    gnn_batcher_stats(b, &req0, &jets0, &launches0, nullptr);
    const auto ta = Clock::now();
    phase.store(1, std::memory_order_release);
    std::this_thread::sleep_for(std::chrono::milliseconds(opts->run_ms));
    phase.store(2, std::memory_order_release);
    const auto tb = Clock::now();
    gnn_batcher_stats(b, &req1, &jets1, &launches1, nullptr);
    for (auto& t : th) t.join();
    std::vector<float> all, q, cu;
    uint64_t jets = 0;
    int status = GNN_OK;
    double tr = 0.0, inf = 0.0;
    for (auto& L : logs) {
        tr += L.transfer_us; inf += L.inference_us;
        all.insert(all.end(), L.total_us.begin(), L.total_us.end());
        q.insert(q.end(), L.queue_us.begin(), L.queue_us.end());
        cu.insert(cu.end(), L.compute_us.begin(), L.compute_us.end());
        jets += L.jets;
        if (L.status != GNN_OK) status = L.status;
    }
    auto mean = [](const std::vector<float>& v) { double s = 0.0; for (float x : v) s += x; return v.empty() ? 0.0 : s / (double)v.size(); };
    out->n_requests = all.size();
    out->n_jets = jets;
    out->seconds = std::chrono::duration<double>(tb - ta).count();
    out->jets_per_s = out->seconds > 0 ? (double)jets / out->seconds : 0.0;
    out->mean_us = mean(all);
    out->queue_us_mean = mean(q);
    out->compute_us_mean = mean(cu);
    out->transfer_us_mean = all.empty() ? 0.0 : tr / (double)all.size();
    out->inference_us_mean = all.empty() ? 0.0 : inf / (double)all.size();
    out->p50_us = percentile(all, 0.50);
    out->p90_us = percentile(all, 0.90);
    out->p99_us = percentile(all, 0.99);
    out->mean_batch_jets = launches1 > launches0 ? (double)(jets1 - jets0) / (double)(launches1 - launches0) : 0.0;
    return status;
}

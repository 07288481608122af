// Host-only harness for tests/test_batcher_host.py: csrc/batcher.cu and csrc/loadgen.cu compiled as plain C++ with
// -fsanitize=thread against the stand-ins below (no GPU, no CUDA runtime library): the CUDA calls the batcher makes become
// host memory operations and gnn_infer_slice becomes a function of its inputs that a client can check, so the run exercises
// exactly the batcher's own threading -- queue, coalescing, per-request completion, instance workers, load-generator
// clients -- under ThreadSanitizer, and verifies that every request gets the logits of ITS jets.
#include "../../paper_2312_06838_b200/csrc/gnn_internal.h"
#include <chrono>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <thread>

// ---- stand-ins for the CUDA runtime entry points batcher.cu uses ------------------------------------------------------------
extern "C" {
cudaError_t cudaSetDevice(int) { return cudaSuccess; }
cudaError_t cudaStreamCreateWithFlags(cudaStream_t* s, unsigned) { *s = nullptr; return cudaSuccess; }
cudaError_t cudaStreamDestroy(cudaStream_t) { return cudaSuccess; }
cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
cudaError_t cudaMallocHost(void** p, size_t n) { *p = std::malloc(n ? n : 1); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
cudaError_t cudaHostAlloc(void** p, size_t n, unsigned) { *p = std::malloc(n ? n : 1); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
cudaError_t cudaMalloc(void** p, size_t n) { *p = std::malloc(n ? n : 1); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
cudaError_t cudaFreeHost(void* p) { std::free(p); return cudaSuccess; }
cudaError_t cudaFree(void* p) { std::free(p); return cudaSuccess; }
cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, cudaMemcpyKind, cudaStream_t) { std::memcpy(d, s, n); return cudaSuccess; }
const char* cudaGetErrorString(cudaError_t) { return "stub"; }
cudaError_t cudaEventCreate(cudaEvent_t* e) { *e = reinterpret_cast<cudaEvent_t>(std::malloc(1)); return cudaSuccess; }
cudaError_t cudaEventDestroy(cudaEvent_t e) { std::free(e); return cudaSuccess; }
cudaError_t cudaEventRecord(cudaEvent_t, cudaStream_t) { return cudaSuccess; }
cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t, cudaEvent_t) { *ms = 0.05f; return cudaSuccess; }

// stand-in forward: logit c of jet j = (c + 1) * sum of the jet's first feature + number of particles; takes a little while
int gnn_infer_slice(gnn_model* m, int32_t, const float* feats, const float*, const int32_t* offsets, int32_t B, int32_t N,
                    float* logits, void*) {
    if (offsets[B] != N) return GNN_ERR_BAD_OFFSETS;
    const int F = m->arch.in_features, NC = m->arch.n_classes;
    for (int j = 0; j < B; ++j) {
        double s = 0.0;
        for (int p = offsets[j]; p < offsets[j + 1]; ++p) s += feats[(size_t)p * F];
        for (int c = 0; c < NC; ++c) logits[(size_t)j * NC + c] = (float)((c + 1) * s + (offsets[j + 1] - offsets[j]));
    }
    std::this_thread::sleep_for(std::chrono::microseconds(200));
    return GNN_OK;
}
}

int main() {
    gnn_model m;
    m.arch.in_features = 3; m.arch.coord_dims = 2; m.arch.n_classes = 2; m.arch.max_particles = 32; m.arch.max_batch_jets = 256;
    m.ws.resize(4);
    gnn_batcher_opts o{256, 500, 4, 0};
    gnn_batcher* b = nullptr;
    if (gnn_batcher_create(&m, &o, &b) != GNN_OK) { std::printf("create failed\n"); return 1; }
    // pool: 96 requests of 1..8 jets with 0..32 particles
    const int R = 96;
    std::vector<int32_t> rfj(R + 1, 0), off(1, 0);
    std::vector<float> feats, coords;
    unsigned rng = 12345u;
    auto next = [&] { rng = rng * 1664525u + 1013904223u; return rng >> 8; };
    for (int r = 0; r < R; ++r) {
        const int nj = 1 + (int)(next() % 8);
        for (int j = 0; j < nj; ++j) {
            const int n = (int)(next() % 33);
            for (int p = 0; p < n; ++p) {
                for (int f = 0; f < 3; ++f) feats.push_back((float)(next() % 100) * 0.25f);
                coords.push_back(0.f); coords.push_back(0.f);
            }
            off.push_back(off.back() + n);
        }
        rfj[r + 1] = rfj[r] + nj;
    }
    // (1) direct submit / wait from several threads, results checked against the stand-in forward
    int bad = 0;
    std::vector<std::thread> th;
    std::mutex mu;
    for (int t = 0; t < 12; ++t)
        th.emplace_back([&, t] {
            for (int it = 0; it < 40; ++it) {
                const int r = (t * 7 + it * 5) % R, j0 = rfj[r], nj = rfj[r + 1] - j0, p0 = off[j0];
                std::vector<int32_t> rel(nj + 1);
                for (int j = 0; j <= nj; ++j) rel[j] = off[j0 + j] - p0;
                std::vector<float> lg((size_t)nj * 2, -1.f);
                gnn_ticket tk;
                int rc = gnn_batcher_submit(b, feats.data() + (size_t)p0 * 3, coords.data() + (size_t)p0 * 2, rel.data(), nj, lg.data(), &tk);
                if (rc == GNN_OK) rc = gnn_batcher_wait(b, tk, (it % 4 == 0) ? 5000000 : -1, nullptr, nullptr);
                int wrong = rc != GNN_OK;
                for (int j = 0; j < nj && !wrong; ++j) {
                    double s = 0.0;
                    for (int p = off[j0 + j]; p < off[j0 + j + 1]; ++p) s += feats[(size_t)p * 3];
                    const int n = off[j0 + j + 1] - off[j0 + j];
                    if (lg[2 * j] != (float)(s + n) || lg[2 * j + 1] != (float)(2 * s + n)) wrong = 1;
                }
                if (wrong) { std::lock_guard<std::mutex> lk(mu); ++bad; }
            }
        });
    for (auto& t : th) t.join();
    // (2) the closed-loop load generator
    gnn_loadgen_pool pool{feats.data(), coords.data(), off.data(), rfj.data(), R, 3, 2, 2};
    gnn_loadgen_opts lo{24, 100, 600};
    gnn_loadgen_result res{};
    const int rc = gnn_loadgen_run(b, &pool, &lo, &res);
    uint64_t nreq = 0, njets = 0, nl = 0; double mb = 0;
    gnn_batcher_stats(b, &nreq, &njets, &nl, &mb);
    gnn_batcher_destroy(b);
    std::printf("batcher host harness: wrong results %d, loadgen rc %d, %llu requests at %.0f jets/s, p50 %.0f us, mean coalesced batch %.1f jets, %llu launches\n",
                bad, rc, (unsigned long long)res.n_requests, res.jets_per_s, res.p50_us, res.mean_batch_jets, (unsigned long long)nl);
    return (bad == 0 && rc == GNN_OK && res.n_requests > 0) ? 0 : 1;
}

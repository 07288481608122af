// batcher.cu -- step a9: host-side dynamic batcher (host code only; compiled by nvcc for the CUDA runtime calls).
//
// the server's dynamic batching "concatenate[s] small requests, run[s], split[s] results"; L268: preferred
// batch size 1024; L271: one model instance per MIG slice.  The single-GPU analogue (BASELINE.json north_star): many
// client threads submit small ragged requests; n_instances worker threads -- each owning a CUDA stream, a workspace
// slice of the model and pinned staging buffers -- coalesce whole requests up to max_batch_jets or until the oldest
// queued request is max_queue_delay_us old, run ONE gnn_infer_slice over the coalesced batch and scatter the logits
// back.  Jets are independent (batch-composition invariance), which is what makes coalescing legal.
#include "gnn_internal.h"
#include <chrono>
#include <condition_variable>
#include <cstring>
#include <deque>
#include <memory>
#include <mutex>
#include <thread>
#include <unordered_map>

namespace {

using Clock = std::chrono::steady_clock;

// One allocation per request: [feats | coords | offsets] copied once at submit.  Completion is per request (its own mutex
// and condition variable): a finished batch wakes exactly the clients whose tickets were in it, and a waking client takes
// the batcher's mutex only to erase its ticket.
struct Request {
    uint64_t id = 0;
    int n_jets = 0, n_particles = 0;
    std::unique_ptr<unsigned char[]> store;
    const float* feats = nullptr;
    const float* coords = nullptr;
    const int32_t* offsets = nullptr;  // [n_jets + 1], relative to the request
    float* out = nullptr;
    Clock::time_point t_submit, t_launch, t_done;
    float transfer_us = 0.0f, inference_us = 0.0f;   // device-side times of the batch the request rode in
    std::mutex mu;
    std::condition_variable cv;
    bool done = false;
    int status = GNN_OK;
};

struct Instance {
    cudaStream_t stream = nullptr;
    float *h_feats = nullptr, *h_coords = nullptr, *h_logits = nullptr;   // pinned
    int32_t* h_offsets = nullptr;
    float *d_feats = nullptr, *d_coords = nullptr, *d_logits = nullptr;
    int32_t* d_offsets = nullptr;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};   // before H2D, after H2D, after the forward, after D2H
    std::thread worker;
};

}  // namespace

struct gnn_batcher {
    gnn_model* m = nullptr;
    gnn_batcher_opts opts{};
    std::mutex mu;
    std::condition_variable cv_work;
    std::deque<Request*> queue;
    int queued_jets = 0;
    std::unordered_map<uint64_t, Request*> tickets;
    uint64_t next_id = 1;
    bool stop = false;
    std::vector<Instance> inst;
    uint64_t n_requests = 0, n_jets = 0, n_launches = 0;
};

namespace {

void finish(gnn_batcher* b, std::vector<Request*>& batch, int status, Clock::time_point t_launch, float transfer_us, float inference_us) {
    (void)b;
    auto now = Clock::now();
    for (Request* r : batch) {
        // notify under the request's lock: once it is released the waiter may delete r, so r is not touched again
        std::lock_guard<std::mutex> lk(r->mu);
        r->status = status; r->t_launch = t_launch; r->t_done = now; r->transfer_us = transfer_us; r->inference_us = inference_us;
        r->done = true;
        r->cv.notify_one();
    }
}

void worker_main(gnn_batcher* b, int wi) {
    cudaSetDevice(b->m->device);
    Instance& I = b->inst[wi];
    const gnn_arch& a = b->m->arch;
    const int F = a.in_features, CD = a.coord_dims, NC = a.n_classes;
    const auto delay = std::chrono::microseconds(b->opts.max_queue_delay_us);
    std::vector<Request*> batch;
    for (;;) {
        batch.clear();
        {
            std::unique_lock<std::mutex> lk(b->mu);
            b->cv_work.wait(lk, [&] { return b->stop || !b->queue.empty(); });
            if (b->queue.empty()) return;                       // stop requested and nothing left to drain
            // coalesce: wait until the batch is full or the oldest request has aged max_queue_delay
            while (!b->stop && b->queued_jets < b->opts.max_batch_jets) {
                auto deadline = b->queue.front()->t_submit + delay;
                if (Clock::now() >= deadline) break;
                b->cv_work.wait_until(lk, deadline);
                if (b->queue.empty()) break;                    // another instance took everything
            }
            if (b->queue.empty()) continue;
            int jets = 0;
            while (!b->queue.empty() && jets + b->queue.front()->n_jets <= b->opts.max_batch_jets) {
                Request* r = b->queue.front();
                b->queue.pop_front();
                jets += r->n_jets;
                batch.push_back(r);
            }
            b->queued_jets -= jets;
            b->n_launches += 1;
            if (!b->queue.empty()) b->cv_work.notify_one();     // leftovers: wake another instance
        }
        // pack whole requests back to back into the pinned staging buffers
        int B = 0, N = 0;
        I.h_offsets[0] = 0;
        for (Request* r : batch) {
            std::memcpy(I.h_feats + (size_t)N * F, r->feats, (size_t)r->n_particles * F * sizeof(float));
            std::memcpy(I.h_coords + (size_t)N * CD, r->coords, (size_t)r->n_particles * CD * sizeof(float));
            for (int j = 0; j < r->n_jets; ++j) I.h_offsets[B + j + 1] = N + r->offsets[j + 1];
            B += r->n_jets; N += r->n_particles;
        }
        auto t_launch = Clock::now();
        int rc = GNN_OK;
        cudaError_t e = cudaEventRecord(I.ev[0], I.stream);
        if (e == cudaSuccess && N > 0) {
            e = cudaMemcpyAsync(I.d_feats, I.h_feats, (size_t)N * F * sizeof(float), cudaMemcpyHostToDevice, I.stream);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(I.d_coords, I.h_coords, (size_t)N * CD * sizeof(float), cudaMemcpyHostToDevice, I.stream);
        }
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(I.d_offsets, I.h_offsets, (size_t)(B + 1) * sizeof(int32_t), cudaMemcpyHostToDevice, I.stream);
        if (e == cudaSuccess) e = cudaEventRecord(I.ev[1], I.stream);
        if (e == cudaSuccess) rc = gnn_infer_slice(b->m, wi, I.d_feats, I.d_coords, I.d_offsets, B, N, I.d_logits, I.stream);
        if (e == cudaSuccess && rc == GNN_OK) e = cudaEventRecord(I.ev[2], I.stream);
        if (e == cudaSuccess && rc == GNN_OK)
            e = cudaMemcpyAsync(I.h_logits, I.d_logits, (size_t)B * NC * sizeof(float), cudaMemcpyDeviceToHost, I.stream);
        if (e == cudaSuccess && rc == GNN_OK) e = cudaEventRecord(I.ev[3], I.stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(I.stream);
        if (e != cudaSuccess) rc = GNN_ERR_CUDA;
        float transfer_us = 0.0f, inference_us = 0.0f;
        if (rc == GNN_OK) {
            float h2d = 0.0f, fw = 0.0f, d2h = 0.0f;             // milliseconds on the instance's stream
            if (cudaEventElapsedTime(&h2d, I.ev[0], I.ev[1]) == cudaSuccess && cudaEventElapsedTime(&fw, I.ev[1], I.ev[2]) == cudaSuccess &&
                cudaEventElapsedTime(&d2h, I.ev[2], I.ev[3]) == cudaSuccess) {
                transfer_us = (h2d + d2h) * 1e3f;
                inference_us = fw * 1e3f;
            }
        }
        if (rc == GNN_OK) {
            int j0 = 0;
            for (Request* r : batch) {
                std::memcpy(r->out, I.h_logits + (size_t)j0 * NC, (size_t)r->n_jets * NC * sizeof(float));
                j0 += r->n_jets;
            }
        }
        finish(b, batch, rc, t_launch, transfer_us, inference_us);
    }
}

void free_instance(Instance& I) {
    if (I.h_feats) cudaFreeHost(I.h_feats);
    if (I.h_coords) cudaFreeHost(I.h_coords);
    if (I.h_logits) cudaFreeHost(I.h_logits);
    if (I.h_offsets) cudaFreeHost(I.h_offsets);
    if (I.d_feats) cudaFree(I.d_feats);
    if (I.d_coords) cudaFree(I.d_coords);
    if (I.d_logits) cudaFree(I.d_logits);
    if (I.d_offsets) cudaFree(I.d_offsets);
    for (cudaEvent_t e : I.ev) if (e) cudaEventDestroy(e);
    if (I.stream) cudaStreamDestroy(I.stream);
}

}  // namespace

extern "C" {

int gnn_batcher_create(gnn_model* m, const gnn_batcher_opts* opts, gnn_batcher** out) {
    if (!m || !opts || !out) return GNN_ERR_NULL;
    *out = nullptr;
    if (opts->max_batch_jets < 1 || opts->max_batch_jets > m->arch.max_batch_jets || opts->max_queue_delay_us < 0 ||
        opts->n_instances < 1 || opts->n_instances > (int)m->ws.size() || opts->max_pending_requests < 0)
        return GNN_ERR_BAD_ARG;
    GNN_CUDA_TRY(cudaSetDevice(m->device));
    gnn_batcher* b = new (std::nothrow) gnn_batcher();
    if (!b) return GNN_ERR_CUDA;
    b->m = m;
    b->opts = *opts;
    if (b->opts.max_pending_requests == 0) b->opts.max_pending_requests = 65536;
    const gnn_arch& a = m->arch;
    size_t Bm = (size_t)opts->max_batch_jets, Nm = Bm * a.max_particles;
    b->inst.resize(opts->n_instances);
    bool ok = true;
    for (auto& I : b->inst) {
        ok = ok && cudaStreamCreateWithFlags(&I.stream, cudaStreamNonBlocking) == cudaSuccess;
        for (auto& e : I.ev) ok = ok && cudaEventCreate(&e) == cudaSuccess;
        ok = ok && cudaMallocHost(&I.h_feats, Nm * a.in_features * sizeof(float)) == cudaSuccess;
        ok = ok && cudaMallocHost(&I.h_coords, Nm * a.coord_dims * sizeof(float)) == cudaSuccess;
        ok = ok && cudaMallocHost(&I.h_logits, Bm * a.n_classes * sizeof(float)) == cudaSuccess;
        ok = ok && cudaMallocHost(&I.h_offsets, (Bm + 1) * sizeof(int32_t)) == cudaSuccess;
        ok = ok && cudaMalloc(&I.d_feats, Nm * a.in_features * sizeof(float)) == cudaSuccess;
        ok = ok && cudaMalloc(&I.d_coords, Nm * a.coord_dims * sizeof(float)) == cudaSuccess;
        ok = ok && cudaMalloc(&I.d_logits, Bm * a.n_classes * sizeof(float)) == cudaSuccess;
        ok = ok && cudaMalloc(&I.d_offsets, (Bm + 1) * sizeof(int32_t)) == cudaSuccess;
    }
    if (!ok) {
        for (auto& I : b->inst) free_instance(I);
        delete b;
        return GNN_ERR_CUDA;
    }
    for (int i = 0; i < opts->n_instances; ++i) b->inst[i].worker = std::thread(worker_main, b, i);
    *out = b;
    return GNN_OK;
}

int gnn_batcher_submit(gnn_batcher* b, const float* feats_host, const float* coords_host, const int32_t* offsets_host,
                       int32_t n_jets, float* logits_host_out, gnn_ticket* out) {
    if (!b || !offsets_host || !logits_host_out || !out) return GNN_ERR_NULL;
    if (n_jets < 1 || n_jets > b->opts.max_batch_jets) return GNN_ERR_BAD_ARG;
    const gnn_arch& a = b->m->arch;
    if (offsets_host[0] != 0) return GNN_ERR_BAD_OFFSETS;
    for (int j = 0; j < n_jets; ++j) {
        int n = offsets_host[j + 1] - offsets_host[j];
        if (n < 0) return GNN_ERR_BAD_OFFSETS;
        if (n > a.max_particles) return GNN_ERR_JET_TOO_LARGE;
    }
    int N = offsets_host[n_jets];
    if (N > 0 && (!feats_host || !coords_host)) return GNN_ERR_NULL;
    Request* r = new (std::nothrow) Request();
    if (!r) return GNN_ERR_CUDA;
    r->n_jets = n_jets; r->n_particles = N; r->out = logits_host_out;
    const size_t fb = (size_t)N * a.in_features * sizeof(float), cb = (size_t)N * a.coord_dims * sizeof(float);
    const size_t ob = (size_t)(n_jets + 1) * sizeof(int32_t);
    r->store.reset(new (std::nothrow) unsigned char[fb + cb + ob]);
    if (!r->store) { delete r; return GNN_ERR_CUDA; }
    if (fb) std::memcpy(r->store.get(), feats_host, fb);
    if (cb) std::memcpy(r->store.get() + fb, coords_host, cb);
    std::memcpy(r->store.get() + fb + cb, offsets_host, ob);
    r->feats = reinterpret_cast<const float*>(r->store.get());
    r->coords = reinterpret_cast<const float*>(r->store.get() + fb);
    r->offsets = reinterpret_cast<const int32_t*>(r->store.get() + fb + cb);
    {
        std::lock_guard<std::mutex> lk(b->mu);
        if (b->stop || (int)b->tickets.size() >= b->opts.max_pending_requests) {
            delete r;
            return GNN_ERR_QUEUE_FULL;
        }
        r->id = b->next_id++;
        r->t_submit = Clock::now();
        b->tickets[r->id] = r;
        b->queue.push_back(r);
        b->queued_jets += n_jets;
        b->n_requests += 1; b->n_jets += (uint64_t)n_jets;
        out->id = r->id;
    }
    b->cv_work.notify_one();
    return GNN_OK;
}

int gnn_batcher_wait_ex(gnn_batcher* b, gnn_ticket t, int64_t timeout_us, gnn_request_times* times) {
    if (!b) return GNN_ERR_NULL;
    Request* r = nullptr;
    {
        std::lock_guard<std::mutex> lk(b->mu);
        auto it = b->tickets.find(t.id);
        if (it == b->tickets.end()) return GNN_ERR_BAD_TICKET;
        r = it->second;
        if (r->id == 0) return GNN_ERR_BAD_TICKET;             // another thread is already waiting on this ticket
        r->id = 0;                                             // claimed: a ticket has one waiter
    }
    int status;
    {
        std::unique_lock<std::mutex> lk(r->mu);
        if (timeout_us < 0) r->cv.wait(lk, [&] { return r->done; });
        else if (!r->cv.wait_for(lk, std::chrono::microseconds(timeout_us), [&] { return r->done; })) {
            lk.unlock();
            std::lock_guard<std::mutex> g(b->mu);
            r->id = t.id;                                      // unclaimed again: the ticket can be waited on later
            return GNN_ERR_TIMEOUT;
        }
        using us = std::chrono::duration<double, std::micro>;
        if (times) {
            times->queue_us = us(r->t_launch - r->t_submit).count();
            times->compute_us = us(r->t_done - r->t_launch).count();
            times->transfer_us = r->transfer_us;
            times->inference_us = r->inference_us;
        }
        status = r->status;
    }
    {
        std::lock_guard<std::mutex> lk(b->mu);
        b->tickets.erase(t.id);
    }
    delete r;
    return status;
}

int gnn_batcher_wait(gnn_batcher* b, gnn_ticket t, int64_t timeout_us, double* queue_us, double* compute_us) {
    gnn_request_times tm{};
    const int rc = gnn_batcher_wait_ex(b, t, timeout_us, &tm);
    if (rc != GNN_ERR_BAD_TICKET && rc != GNN_ERR_TIMEOUT && rc != GNN_ERR_NULL) {
        if (queue_us) *queue_us = tm.queue_us;
        if (compute_us) *compute_us = tm.compute_us;
    }
    return rc;
}

int gnn_batcher_stats(gnn_batcher* b, uint64_t* n_requests, uint64_t* n_jets, uint64_t* n_launches, double* mean_batch_jets) {
    if (!b) return GNN_ERR_NULL;
    std::lock_guard<std::mutex> lk(b->mu);
    if (n_requests) *n_requests = b->n_requests;
    if (n_jets) *n_jets = b->n_jets;
    if (n_launches) *n_launches = b->n_launches;
    if (mean_batch_jets) *mean_batch_jets = b->n_launches ? (double)b->n_jets / (double)b->n_launches : 0.0;
    return GNN_OK;
}

void gnn_batcher_destroy(gnn_batcher* b) {
    if (!b) return;
    {
        std::lock_guard<std::mutex> lk(b->mu);
        b->stop = true;                       // workers drain the queue (no more coalescing delay), then exit
    }
    b->cv_work.notify_all();
    for (auto& I : b->inst)
        if (I.worker.joinable()) I.worker.join();
    cudaSetDevice(b->m->device);
    for (auto& I : b->inst) free_instance(I);
    for (auto& kv : b->tickets) delete kv.second;     // uncollected tickets
    delete b;
}

}  // extern "C"

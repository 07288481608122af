// api.cu -- the C ABI of include/gnn.h: model creation (BN fold, transposition, packing), workspace slices, and the
// launch plan of one forward pass.  Host code only enqueues kernels; every step of the path runs on the GPU.
#include "gnn_internal.h"
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>

int edgeconv_bf16_prepare(gnn_model& m, const float* blob_host);       // edgeconv_bf16.cu
void edgeconv_bf16_release(gnn_model& m);
int launch_edgeconv_bf16(gnn_model& m, int block, const float* x, const int32_t* idx, int N, float* y, Workspace& w,
                         cudaStream_t s);
int launch_pre_bf16(gnn_model& m, int block, const float* x, int N, Workspace& w, cudaStream_t s, int dep);
bool pre_bf16_single_wave(const gnn_model& m, int block);
int launch_edge_bf16(gnn_model& m, int block, const int32_t* idx, int N, float* y, Workspace& w, cudaStream_t s);
bool edgeconv_bf16_can_pool(const gnn_model& m, int block);

namespace {

size_t blob_count(const gnn_arch& a) {
    size_t n = 0;
    for (int l = 0; l < a.n_blocks; ++l) {
        size_t cin = block_in(a, l), c1 = a.channels[l][0], c2 = a.channels[l][1], c3 = a.channels[l][2];
        n += c1 * 2 * cin + 2 * c1 + c2 * c1 + 2 * c2 + c3 * c2 + 2 * c3 + c3 * cin + 2 * c3;
    }
    size_t in = a.channels[a.n_blocks - 1][2];
    for (int i = 0; i <= a.n_fc_hidden; ++i) {
        size_t out = (i < a.n_fc_hidden) ? a.fc_hidden[i] : a.n_classes;
        n += out * in + out;
        in = out;
    }
    return n;
}

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

int check_arch(const gnn_arch& a) {
    if (a.n_blocks < 1 || a.n_blocks > GNN_MAX_BLOCKS) return GNN_ERR_BAD_ARCH;
    if (a.in_features < 1 || a.in_features > 1024) return GNN_ERR_BAD_ARCH;
    if (a.coord_dims < 1 || a.coord_dims > 8) return GNN_ERR_BAD_ARCH;
    if (a.k < 1 || a.k > GNN_MAX_K) return GNN_ERR_BAD_ARCH;
    if (a.n_fc_hidden < 0 || a.n_fc_hidden > GNN_MAX_FC) return GNN_ERR_BAD_ARCH;
    if (a.n_classes < 1 || a.n_classes > 64) return GNN_ERR_BAD_ARCH;
    if (a.max_particles < 1 || a.max_particles > GNN_MAX_PARTICLES) return GNN_ERR_BAD_ARCH;
    if (a.max_batch_jets < 1) return GNN_ERR_BAD_ARCH;
    if (a.workspace_slices < 0 || a.workspace_slices > GNN_MAX_SLICES) return GNN_ERR_BAD_ARCH;
    if (a.precision != GNN_FP32_VALIDATION && a.precision != GNN_BF16) return GNN_ERR_BAD_ARCH;
    for (int l = 0; l < a.n_blocks; ++l)
        for (int i = 0; i < 3; ++i) {
            int c = a.channels[l][i];
            if (c < 8 || c > 1024 || (c % 8) != 0) return GNN_ERR_BAD_ARCH;
        }
    for (int i = 0; i < a.n_fc_hidden; ++i)
        if (a.fc_hidden[i] < 1 || a.fc_hidden[i] > 1024) return GNN_ERR_BAD_ARCH;
    if (a.channels[a.n_blocks - 1][2] > 1024) return GNN_ERR_BAD_ARCH;
    if (a.precision == GNN_BF16) {
        if (!is_pow2(a.k)) return GNN_ERR_BAD_ARCH;
        for (int l = 0; l < a.n_blocks; ++l) {
            int c = a.channels[l][0];
            if (a.channels[l][1] != c || a.channels[l][2] != c) return GNN_ERR_BAD_ARCH;
            if (c != 32 && c != 64 && c != 128 && c != 256 && c != 512) return GNN_ERR_BAD_ARCH;
        }
    }
    return GNN_OK;
}

template <typename T>
int dev_alloc(gnn_model* m, T** p, size_t count) {
    void* q = nullptr;
    if (count == 0) count = 1;
    GNN_CUDA_TRY(cudaMalloc(&q, count * sizeof(T)));
    m->allocs.push_back(q);
    *p = static_cast<T*>(q);
    return GNN_OK;
}

// fold scale into W (fp32), transpose to Wt[Kp][N] with zero rows up to Kp, upload
int upload_linear(gnn_model* m, const float* W, const float* scale, const float* shift_or_bias, int K, int N, LinF32* out) {
    int Kp = (K + 3) & ~3;
    int Np = (N + 3) & ~3;              // column padding keeps float4 loads of the SIMT kernels in bounds
    std::vector<float> wt((size_t)Kp * Np, 0.0f), sh((size_t)Np, 0.0f);
    for (int o = 0; o < N; ++o) {
        float sc = scale ? scale[o] : 1.0f;
        for (int c = 0; c < K; ++c) wt[(size_t)c * Np + o] = sc * W[(size_t)o * K + c];
        sh[o] = shift_or_bias[o];
    }
    float *dW = nullptr, *dS = nullptr;
    int rc;
    if ((rc = dev_alloc(m, &dW, wt.size())) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &dS, sh.size())) != GNN_OK) return rc;
    GNN_CUDA_TRY(cudaMemcpy(dW, wt.data(), wt.size() * sizeof(float), cudaMemcpyHostToDevice));
    GNN_CUDA_TRY(cudaMemcpy(dS, sh.data(), sh.size() * sizeof(float), cudaMemcpyHostToDevice));
    out->Wt = dW; out->shift = dS; out->K = K; out->Kp = Kp; out->N = N; out->ld = Np;
    return GNN_OK;
}

int build_model(gnn_model* m, const float* blob) {
    const gnn_arch& a = m->arch;
    const float* p = blob;
    int rc;
    for (int l = 0; l < a.n_blocks; ++l) {
        BlockDev& b = m->blocks[l];
        b.cin = block_in(a, l); b.c1 = a.channels[l][0]; b.c2 = a.channels[l][1]; b.c3 = a.channels[l][2];
        const int ins[3] = {2 * b.cin, b.c1, b.c2}, outs[3] = {b.c1, b.c2, b.c3};
        LinF32* dst[3] = {&b.l1, &b.l2, &b.l3};
        for (int i = 0; i < 3; ++i) {
            const float* W = p; p += (size_t)outs[i] * ins[i];
            const float* sc = p; p += outs[i];
            const float* sh = p; p += outs[i];
            if ((rc = upload_linear(m, W, sc, sh, ins[i], outs[i], dst[i])) != GNN_OK) return rc;
        }
        const float* W = p; p += (size_t)b.c3 * b.cin;
        const float* sc = p; p += b.c3;
        const float* sh = p; p += b.c3;
        if ((rc = upload_linear(m, W, sc, sh, b.cin, b.c3, &b.sc)) != GNN_OK) return rc;
    }
    int in = a.channels[a.n_blocks - 1][2];
    m->n_fc = 0;
    for (int i = 0; i <= a.n_fc_hidden; ++i) {
        int out = (i < a.n_fc_hidden) ? a.fc_hidden[i] : a.n_classes;
        const float* W = p; p += (size_t)out * in;
        const float* bias = p; p += out;
        if ((rc = upload_linear(m, W, nullptr, bias, in, out, &m->fc[m->n_fc])) != GNN_OK) return rc;
        ++m->n_fc;
        in = out;
    }
    return GNN_OK;
}

int alloc_workspace(gnn_model* m, Workspace& w) {
    const gnn_arch& a = m->arch;
    int rc;
    size_t Nmax = (size_t)m->Nmax, Bmax = (size_t)a.max_batch_jets;
    if ((rc = dev_alloc(m, &w.xa, Nmax * m->Cmax)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.xb, Nmax * m->Cmax)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.idx, Nmax * a.k)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.pjet, Nmax)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.dm, Nmax * (size_t)((a.max_particles + 3) & ~3))) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.jet_start, Bmax)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.jet_n, Bmax)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.status, 1)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.meta, 4)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.groups, Bmax)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.pjid, Nmax)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.pool, Bmax * (size_t)a.channels[a.n_blocks - 1][2])) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.pfeats, Nmax * a.in_features)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.pcoords, Nmax * a.coord_dims)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.poffsets, Bmax + 1)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.pcounts, Bmax)) != GNN_OK) return rc;
    if ((rc = dev_alloc(m, &w.hlogits, Bmax * a.n_classes)) != GNN_OK) return rc;
    GNN_CUDA_TRY(cudaMemset(w.pool, 0, Bmax * (size_t)a.channels[a.n_blocks - 1][2] * sizeof(unsigned long long)));
    GNN_CUDA_TRY(cudaMallocHost(reinterpret_cast<void**>(&w.h_status), sizeof(unsigned)));
    *w.h_status = 0u;
    GNN_CUDA_TRY(cudaMemset(w.status, 0, sizeof(unsigned)));
    GNN_CUDA_TRY(cudaMemset(w.meta, 0, 4 * sizeof(int32_t)));
    return GNN_OK;
}

// stage timing: one event before the first stage and one after each stage, on the caller's stream
struct StageTimer {
    Workspace& w; cudaStream_t s; bool on; int stage = 0; size_t base = 0;
    StageTimer(Workspace& w_, cudaStream_t s_, int n_stages) : w(w_), s(s_) {
        on = w.prof_on && w.prof_forwards < PROF_MAX_FORWARDS;
        if (!on) return;
        if (w.prof_stages != n_stages) { w.prof_stages = n_stages; w.prof_names.assign(n_stages, ""); w.prof_forwards = 0; }
        base = (size_t)w.prof_forwards * (n_stages + 1);
        while (w.prof_events.size() < base + n_stages + 1) {
            cudaEvent_t e = nullptr;
            if (cudaEventCreate(&e) != cudaSuccess) { on = false; return; }
            w.prof_events.push_back(e);
        }
        cudaEventRecord(w.prof_events[base], s);
    }
    void mark(const char* name, int l = -1) {
        if (!on) return;
        if (w.prof_names[stage].empty()) w.prof_names[stage] = l < 0 ? std::string(name) : std::string(name) + std::to_string(l);
        cudaEventRecord(w.prof_events[base + stage + 1], s);
        ++stage;
    }
    ~StageTimer() { if (on) ++w.prof_forwards; }
};

// the launch plan of one forward (SURVEY.md call stack (4)): ingest -> per block [kNN, EdgeConv] -> pool + head
int forward(gnn_model* m, Workspace& w, const float* feats, const float* coords, const int32_t* offsets,
            const int32_t* counts, int B, int N_exact, int N_upper, float* logits, cudaStream_t s, int* n_launches_out = nullptr) {
    const gnn_arch& a = m->arch;
    int n = 0, rc;
    StageTimer tm(w, s, 2 + 2 * a.n_blocks);
    if ((rc = launch_ingest(offsets, counts, B, N_exact, (int)m->Nmax, a.max_particles, w, s)) < 0) return rc;
    n += rc;
    tm.mark("ingest");
    const float* x = feats;
    float* bufs[2] = {w.xa, w.xb};
    const bool bf16 = a.precision == GNN_BF16;
    // bf16 mode: the last block adds its output straight into the per-jet channel sums (step a7 inside E3 of step a6).  The
    // sums are zero between forwards: the head kernel that reads them clears them (head_split_kernel), else they are cleared here.
#ifdef GNN_DEV_KNOBS                              // developer builds only (build.py: GNN_NVCC_DEFS=-DGNN_DEV_KNOBS): A/B of the pooling epilogue
    static const bool no_fuse = std::getenv("GNN_NO_POOL_FUSE") != nullptr;
#else
    constexpr bool no_fuse = false;               // the shipped library's launch plan does not depend on the environment
#endif
    // The pooling epilogue finds a particle's jet in w.pjid, and only the grouped kNN kernels write that map: the epilogue is
    // used only if some block of THIS forward takes the grouped path (otherwise -- coord_dims > 4 with no 64 / 128 / 256-wide
    // feature space, or max_particles beyond a tile -- the last block stores its output and pool_head_kernel pools it).
    bool pjid_written = false;
    for (int l = 0; l < a.n_blocks; ++l)
        pjid_written = pjid_written || knn_group_supported(l == 0 ? a.coord_dims : block_in(a, l), a.max_particles);
    const bool fuse_pool = bf16 && !no_fuse && pjid_written && edgeconv_bf16_can_pool(*m, a.n_blocks - 1);
    if (fuse_pool && !w.pool_self_cleaning &&
        cudaMemsetAsync(w.pool, 0, (size_t)B * a.channels[a.n_blocks - 1][2] * sizeof(unsigned long long), s) != cudaSuccess)
        return GNN_ERR_CUDA;
    for (int l = 0; l < a.n_blocks; ++l) {
        const float* space = (l == 0) ? coords : x;
        int D = (l == 0) ? a.coord_dims : block_in(a, l);
        float* y = (fuse_pool && l == a.n_blocks - 1) ? nullptr : bufs[l & 1];
        if (bf16) {
            // One stream, programmatic dependent launches.  u, v and the shortcut of a block depend on x only, as does its kNN,
            // so the two kernels run SIDE BY SIDE as a primary / secondary pair (gnn_internal.h, DEP_*); the primary is the one
            // whose CTAs are all resident at once: the tensor-core pre kernel (blocks >= 2), else the grouped kNN kernel.  The
            // primary's prologue (weights, TMEM) runs under the tail of the kernel before it.  edge_l is itself launched as a
            // dependent of the secondary (launch_edge_t passes the attribute): its prologue may start while the secondary
            // drains, and its grid_dep_wait returns when the secondary -- whose CTA 0 waits for the primary -- has completed,
            // i.e. when the pair has.
            int rc_pre, rc_knn;
            if (N_upper == 0 || !knn_group_supported(D, a.max_particles)) {          // no pair: ordinary launches
                if ((rc_pre = launch_pre_bf16(*m, l, x, N_upper, w, s, DEP_NONE)) < 0) return rc_pre;
                if ((rc_knn = launch_knn(space, D, a.k, B, a.max_particles, w, w.idx, 0, 1, s)) < 0) return rc_knn;
            } else if (pre_bf16_single_wave(*m, l)) {
                if ((rc_pre = launch_pre_bf16(*m, l, x, N_upper, w, s, DEP_PRIMARY)) < 0) return rc_pre;
                if ((rc_knn = launch_knn(space, D, a.k, B, a.max_particles, w, w.idx, 0, 1, s, DEP_SECONDARY)) < 0) return rc_knn;
            } else {
                if ((rc_knn = launch_knn(space, D, a.k, B, a.max_particles, w, w.idx, 0, 1, s, DEP_PRIMARY)) < 0) return rc_knn;
                if ((rc_pre = launch_pre_bf16(*m, l, x, N_upper, w, s, DEP_SECONDARY)) < 0) return rc_pre;
            }
            n += rc_pre + rc_knn;
            tm.mark("knn", l);
            rc = launch_edge_bf16(*m, l, w.idx, N_upper, y, w, s);
        } else {
            const int rc_knn = launch_knn(space, D, a.k, B, a.max_particles, w, w.idx, 0, 0, s);
            if (rc_knn < 0) return rc_knn;
            n += rc_knn;
            tm.mark("knn", l);
            rc = launch_edgeconv_f32(m->blocks[l], a.k, x, w.idx, N_upper, y, w, s);
        }
        if (rc < 0) return rc;
        n += rc;
        tm.mark("edgeconv", l);
        x = y;
    }
    if ((rc = launch_pool_head(*m, x, B, w, logits, s, bf16)) < 0) return rc;
    n += rc;
    tm.mark("pool_head");
    if (n_launches_out) *n_launches_out = n;
    else m->launches.fetch_add(n, std::memory_order_relaxed);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        std::fprintf(stderr, "libgnn: launch failed: %s\n", cudaGetErrorString(e));
        return GNN_ERR_CUDA;
    }
    return GNN_OK;
}

// gnn_infer_slice through the slice's graph cache.  A call is replayed from a graph if its arguments (pointers, B, N) equal
// an earlier call's; the graph is captured the SECOND time a set of arguments is seen, so one-off calls never pay for a
// capture.  Not used while stage timing is on (events between the kernels) or while the caller's stream is itself being
// captured (the forward is then simply recorded into the caller's graph: one stream, no host synchronisation).
int forward_cached(gnn_model* m, Workspace& w, const float* feats, const float* coords, const int32_t* offsets, int B, int N,
                   float* logits, cudaStream_t s) {
#ifdef GNN_DEV_KNOBS
    static const bool no_graphs = std::getenv("GNN_NO_GRAPHS") != nullptr;
#else
    constexpr bool no_graphs = false;
#endif
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (no_graphs || w.prof_on || cudaStreamIsCapturing(s, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone)
        return forward(m, w, feats, coords, offsets, nullptr, B, N, N, logits, s);
    Workspace::ForwardGraph* hit = nullptr;
    for (auto& g : w.graphs)
        if (g.feats == feats && g.coords == coords && g.offsets == offsets && g.logits == logits && g.B == B && g.N == N) { hit = &g; break; }
    if (hit && hit->exec) {
        hit->last_use = ++w.graph_clock;
        GNN_CUDA_TRY(cudaGraphLaunch(hit->exec, s));
        m->launches.fetch_add(hit->n_launches, std::memory_order_relaxed);
        return GNN_OK;
    }
    if (!hit) {                                                  // first sighting: remember the arguments, run normally
        if ((int)w.graphs.size() < GNN_MAX_FORWARD_GRAPHS) w.graphs.emplace_back();
        else {
            hit = &w.graphs[0];
            for (auto& g : w.graphs) if (g.last_use < hit->last_use) hit = &g;
            if (hit->exec) cudaGraphExecDestroy(hit->exec);
            *hit = Workspace::ForwardGraph();
        }
        Workspace::ForwardGraph& g = hit ? *hit : w.graphs.back();
        g.feats = feats; g.coords = coords; g.offsets = offsets; g.logits = logits; g.B = B; g.N = N;
        g.last_use = ++w.graph_clock;
        return forward(m, w, feats, coords, offsets, nullptr, B, N, N, logits, s);
    }
    // second sighting: capture, instantiate, launch
    hit->last_use = ++w.graph_clock;
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        return forward(m, w, feats, coords, offsets, nullptr, B, N, N, logits, s);
    }
    int n = 0;
    const int rc = forward(m, w, feats, coords, offsets, nullptr, B, N, N, logits, s, &n);
    const cudaError_t ec = cudaStreamEndCapture(s, &graph);
    if (rc != GNN_OK || ec != cudaSuccess || graph == nullptr) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        if (rc != GNN_OK) return rc;
        *hit = Workspace::ForwardGraph();                        // capture not possible here: keep launching directly
        return forward(m, w, feats, coords, offsets, nullptr, B, N, N, logits, s);
    }
    cudaGraphExec_t exec = nullptr;
    const cudaError_t ei = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ei != cudaSuccess || exec == nullptr) {
        cudaGetLastError();
        *hit = Workspace::ForwardGraph();
        return forward(m, w, feats, coords, offsets, nullptr, B, N, N, logits, s);
    }
    hit->exec = exec; hit->n_launches = n;
    GNN_CUDA_TRY(cudaGraphLaunch(exec, s));
    m->launches.fetch_add(n, std::memory_order_relaxed);
    return GNN_OK;
}

}  // namespace

bool gnn_pdl_enabled() {
#ifdef GNN_DEV_KNOBS
    static const bool on = std::getenv("GNN_NO_PDL") == nullptr;
    return on;
#else
    return true;
#endif
}

extern "C" {

int gnn_weights_bytes(const gnn_arch* arch, size_t* out_bytes) {
    if (!arch || !out_bytes) return GNN_ERR_NULL;
    int rc = check_arch(*arch);
    if (rc != GNN_OK) return rc;
    *out_bytes = blob_count(*arch) * sizeof(float);
    return GNN_OK;
}

int gnn_create(const void* weights_host, size_t bytes, const gnn_arch* arch, int device, gnn_model** out) {
    if (!weights_host || !arch || !out) return GNN_ERR_NULL;
    *out = nullptr;
    int rc = check_arch(*arch);
    if (rc != GNN_OK) return rc;
    if (bytes != blob_count(*arch) * sizeof(float)) return GNN_ERR_BAD_BLOB_SIZE;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        std::fprintf(stderr, "libgnn: no usable CUDA device %d (found %d); there is no CPU fallback\n", device, ndev);
        return GNN_ERR_CUDA;
    }
    GNN_CUDA_TRY(cudaSetDevice(device));
    gnn_model* m = new (std::nothrow) gnn_model();
    if (!m) return GNN_ERR_CUDA;
    m->arch = *arch;
    if (m->arch.workspace_slices == 0) m->arch.workspace_slices = 1;
    m->device = device;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) m->n_sms = prop.multiProcessorCount;
    m->Nmax = (int64_t)arch->max_batch_jets * arch->max_particles;
    m->Cmax = 8;
    for (int l = 0; l < arch->n_blocks; ++l) m->Cmax = std::max(m->Cmax, arch->channels[l][2]);
    if ((rc = knn_configure()) != GNN_OK || (rc = pool_head_configure()) != GNN_OK || (rc = knn_group_configure()) != GNN_OK || (rc = edgeconv_f32_configure()) != GNN_OK ||
        (rc = build_model(m, static_cast<const float*>(weights_host))) != GNN_OK) {
        gnn_destroy(m);
        return rc;
    }
    m->ws.resize(m->arch.workspace_slices);
    for (auto& w : m->ws) {
        if ((rc = alloc_workspace(m, w)) != GNN_OK) { gnn_destroy(m); return rc; }
        w.pool_self_cleaning = head_clears_pool(*m);
    }
    if (m->arch.precision == GNN_BF16 &&
        (rc = edgeconv_bf16_prepare(*m, static_cast<const float*>(weights_host))) != GNN_OK) {
        gnn_destroy(m);
        return rc;
    }
    GNN_CUDA_TRY(cudaDeviceSynchronize());
    *out = m;
    return GNN_OK;
}

void gnn_destroy(gnn_model* m) {
    if (!m) return;
    cudaSetDevice(m->device);
    cudaDeviceSynchronize();
    for (void* p : m->allocs) cudaFree(p);
    edgeconv_bf16_release(*m);
    for (auto& w : m->ws) {
        for (auto& g : w.graphs) if (g.exec) cudaGraphExecDestroy(g.exec);
        if (w.h_status) cudaFreeHost(w.h_status);
        for (cudaEvent_t e : w.prof_events) cudaEventDestroy(e);
    }
    delete m;
}

int gnn_infer_slice(gnn_model* m, int32_t slice, const float* feats_dev, const float* coords_dev,
                    const int32_t* offsets_dev, int32_t B, int32_t N, float* logits_dev, void* cuda_stream) {
    if (!m) return GNN_ERR_NULL;
    if (B < 0 || N < 0) return GNN_ERR_BAD_ARG;
    if (slice < 0 || slice >= (int)m->ws.size()) return GNN_ERR_BATCH_TOO_LARGE;
    if (B > m->arch.max_batch_jets || (int64_t)N > m->Nmax) return GNN_ERR_BATCH_TOO_LARGE;
    if (B == 0) return GNN_OK;
    if (!offsets_dev || !logits_dev || (N > 0 && (!feats_dev || !coords_dev))) return GNN_ERR_NULL;
    return forward_cached(m, m->ws[slice], feats_dev, coords_dev, offsets_dev, B, N, logits_dev, static_cast<cudaStream_t>(cuda_stream));
}

int gnn_infer(gnn_model* m, const float* feats_dev, const float* coords_dev, const int32_t* offsets_dev, int32_t B,
              int32_t N, float* logits_dev, void* cuda_stream) {
    return gnn_infer_slice(m, 0, feats_dev, coords_dev, offsets_dev, B, N, logits_dev, cuda_stream);
}

int gnn_infer_padded_slice(gnn_model* m, int32_t slice, const float* feats_dev, const float* coords_dev, const float* mask_dev,
                           int32_t B, int32_t P, float* logits_dev, void* cuda_stream) {
    if (!m) return GNN_ERR_NULL;
    if (B < 0 || P < 0) return GNN_ERR_BAD_ARG;
    if (slice < 0 || slice >= (int)m->ws.size()) return GNN_ERR_BATCH_TOO_LARGE;
    if (B > m->arch.max_batch_jets || (int64_t)B * P > (int64_t)m->arch.max_batch_jets * GNN_MAX_PARTICLES)
        return GNN_ERR_BATCH_TOO_LARGE;
    if (B == 0) return GNN_OK;
    if (!logits_dev || (P > 0 && (!feats_dev || !coords_dev || !mask_dev))) return GNN_ERR_NULL;
    Workspace& w = m->ws[slice];
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    int rc = launch_compact_padded(feats_dev, coords_dev, mask_dev, B, P, m->arch.in_features, m->arch.coord_dims,
                                   m->arch.max_particles, w, s);
    if (rc < 0) return rc;
    m->launches.fetch_add(rc, std::memory_order_relaxed);
    int64_t upper = std::min<int64_t>((int64_t)B * std::min<int>(P, m->arch.max_particles), m->Nmax);
    return forward(m, w, w.pfeats, w.pcoords, w.poffsets, w.pcounts, B, -1, (int)upper, logits_dev, s);
}

int gnn_infer_channel_first(gnn_model* m, int32_t slice, const float* points_dev, const float* features_dev, const float* mask_dev,
                            int32_t B, int32_t P, int32_t softmax, float* out_dev, void* cuda_stream) {
    if (!m) return GNN_ERR_NULL;
    if (B < 0 || P < 0) return GNN_ERR_BAD_ARG;
    if (slice < 0 || slice >= (int)m->ws.size()) return GNN_ERR_BATCH_TOO_LARGE;
    if (B > m->arch.max_batch_jets || (int64_t)B * P > (int64_t)m->arch.max_batch_jets * GNN_MAX_PARTICLES)
        return GNN_ERR_BATCH_TOO_LARGE;
    if (B == 0) return GNN_OK;
    if (!out_dev || (P > 0 && (!features_dev || !points_dev || !mask_dev))) return GNN_ERR_NULL;
    Workspace& w = m->ws[slice];
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    int rc = launch_compact_padded(features_dev, points_dev, mask_dev, B, P, m->arch.in_features, m->arch.coord_dims,
                                   m->arch.max_particles, w, s, true);
    if (rc < 0) return rc;
    m->launches.fetch_add(rc, std::memory_order_relaxed);
    int64_t upper = std::min<int64_t>((int64_t)B * std::min<int>(P, m->arch.max_particles), m->Nmax);
    rc = forward(m, w, w.pfeats, w.pcoords, w.poffsets, w.pcounts, B, -1, (int)upper, out_dev, s);
    if (rc != GNN_OK || !softmax) return rc;
    if ((rc = launch_softmax(out_dev, B, m->arch.n_classes, out_dev, s)) < 0) return rc;
    m->launches.fetch_add(rc, std::memory_order_relaxed);
    return cudaGetLastError() == cudaSuccess ? GNN_OK : GNN_ERR_CUDA;
}

int gnn_softmax(const float* logits_dev, int32_t B, int32_t n_classes, float* probs_dev, void* cuda_stream) {
    if (B < 0 || n_classes < 1) return GNN_ERR_BAD_ARG;
    if (B == 0) return GNN_OK;
    if (!logits_dev || !probs_dev) return GNN_ERR_NULL;
    if (launch_softmax(logits_dev, B, n_classes, probs_dev, static_cast<cudaStream_t>(cuda_stream)) < 0) return GNN_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? GNN_OK : GNN_ERR_CUDA;
}

int gnn_infer_padded(gnn_model* m, const float* feats_dev, const float* coords_dev, const float* mask_dev, int32_t B,
                     int32_t P, float* logits_dev, void* cuda_stream) {
    return gnn_infer_padded_slice(m, 0, feats_dev, coords_dev, mask_dev, B, P, logits_dev, cuda_stream);
}

int gnn_infer_host_begin(gnn_model* m, int32_t slice, const float* feats_host, const float* coords_host,
                         const int32_t* offsets_host, int32_t B, int32_t N, float* logits_host, void* cuda_stream) {
    if (!m) return GNN_ERR_NULL;
    if (B < 0 || N < 0) return GNN_ERR_BAD_ARG;
    if (slice < 0 || slice >= (int)m->ws.size()) return GNN_ERR_BATCH_TOO_LARGE;
    if (B > m->arch.max_batch_jets || (int64_t)N > m->Nmax) return GNN_ERR_BATCH_TOO_LARGE;
    Workspace& w = m->ws[slice];
    w.host_pending = false;
    if (B == 0) return GNN_OK;
    if (!offsets_host || !logits_host || (N > 0 && (!feats_host || !coords_host))) return GNN_ERR_NULL;
    const gnn_arch& a = m->arch;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (N > 0) {
        GNN_CUDA_TRY(cudaMemcpyAsync(w.pfeats, feats_host, (size_t)N * a.in_features * sizeof(float), cudaMemcpyHostToDevice, s));
        GNN_CUDA_TRY(cudaMemcpyAsync(w.pcoords, coords_host, (size_t)N * a.coord_dims * sizeof(float), cudaMemcpyHostToDevice, s));
    }
    GNN_CUDA_TRY(cudaMemcpyAsync(w.poffsets, offsets_host, (size_t)(B + 1) * sizeof(int32_t), cudaMemcpyHostToDevice, s));
    int rc = forward(m, w, w.pfeats, w.pcoords, w.poffsets, nullptr, B, N, N, w.hlogits, s);
    if (rc != GNN_OK) return rc;
    GNN_CUDA_TRY(cudaMemcpyAsync(logits_host, w.hlogits, (size_t)B * a.n_classes * sizeof(float), cudaMemcpyDeviceToHost, s));
    // the sticky status word rides the same stream into pinned memory of the slice: gnn_infer_host_end needs one synchronisation
    GNN_CUDA_TRY(cudaMemcpyAsync(w.h_status, w.status, sizeof(unsigned), cudaMemcpyDeviceToHost, s));
    w.host_pending = true;
    return GNN_OK;
}

int gnn_infer_host_end(gnn_model* m, int32_t slice, void* cuda_stream) {
    if (!m) return GNN_ERR_NULL;
    if (slice < 0 || slice >= (int)m->ws.size()) return GNN_ERR_BATCH_TOO_LARGE;
    Workspace& w = m->ws[slice];
    if (!w.host_pending) return GNN_OK;                          // nothing in flight (B = 0, or already collected)
    w.host_pending = false;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    GNN_CUDA_TRY(cudaStreamSynchronize(s));
    const unsigned st = *w.h_status;
    if (st) {
        GNN_CUDA_TRY(cudaMemsetAsync(w.status, 0, sizeof(unsigned), s));
        GNN_CUDA_TRY(cudaStreamSynchronize(s));
    }
    if (st & GNN_DEV_BAD_OFFSETS) return GNN_ERR_BAD_OFFSETS;
    if (st & GNN_DEV_JET_TOO_LARGE) return GNN_ERR_JET_TOO_LARGE;
    return GNN_OK;
}

int gnn_infer_host(gnn_model* m, int32_t slice, const float* feats_host, const float* coords_host,
                   const int32_t* offsets_host, int32_t B, int32_t N, float* logits_host, void* cuda_stream) {
    const int rc = gnn_infer_host_begin(m, slice, feats_host, coords_host, offsets_host, B, N, logits_host, cuda_stream);
    return rc != GNN_OK ? rc : gnn_infer_host_end(m, slice, cuda_stream);
}

int gnn_profile_enable(gnn_model* m, int32_t slice, int32_t on) {
    if (!m) return GNN_ERR_NULL;
    if (slice < 0 || slice >= (int)m->ws.size()) return GNN_ERR_BAD_ARG;
    m->ws[slice].prof_on = on != 0;
    if (on) m->ws[slice].prof_forwards = 0;
    return GNN_OK;
}

int gnn_profile_read(gnn_model* m, int32_t slice, int32_t max_stages, float* ms_mean_out, int32_t* n_stages_out,
                     int32_t* n_forwards_out) {
    if (!m || !ms_mean_out || !n_stages_out || !n_forwards_out) return GNN_ERR_NULL;
    if (slice < 0 || slice >= (int)m->ws.size()) return GNN_ERR_BAD_ARG;
    Workspace& w = m->ws[slice];
    const int S = w.prof_stages, R = w.prof_forwards;
    *n_stages_out = S; *n_forwards_out = R;
    if (S > max_stages) return GNN_ERR_BAD_ARG;
    for (int i = 0; i < S; ++i) ms_mean_out[i] = 0.0f;
    if (R == 0) return GNN_OK;
    for (int r = 0; r < R; ++r) {
        size_t base = (size_t)r * (S + 1);
        GNN_CUDA_TRY(cudaEventSynchronize(w.prof_events[base + S]));
        for (int i = 0; i < S; ++i) {
            float ms = 0.0f;
            GNN_CUDA_TRY(cudaEventElapsedTime(&ms, w.prof_events[base + i], w.prof_events[base + i + 1]));
            ms_mean_out[i] += ms;
        }
    }
    for (int i = 0; i < S; ++i) ms_mean_out[i] /= (float)R;
    return GNN_OK;
}

const char* gnn_profile_stage_name(gnn_model* m, int32_t slice, int32_t stage) {
    if (!m || slice < 0 || slice >= (int)m->ws.size()) return nullptr;
    Workspace& w = m->ws[slice];
    if (stage < 0 || stage >= (int)w.prof_names.size()) return nullptr;
    return w.prof_names[stage].c_str();
}

int gnn_status_check(gnn_model* m, int32_t slice, void* cuda_stream) {
    if (!m) return GNN_ERR_NULL;
    if (slice < 0 || slice >= (int)m->ws.size()) return GNN_ERR_BATCH_TOO_LARGE;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    unsigned st = 0;
    GNN_CUDA_TRY(cudaMemcpyAsync(&st, m->ws[slice].status, sizeof(unsigned), cudaMemcpyDeviceToHost, s));
    GNN_CUDA_TRY(cudaStreamSynchronize(s));
    if (st) {
        GNN_CUDA_TRY(cudaMemsetAsync(m->ws[slice].status, 0, sizeof(unsigned), s));
        GNN_CUDA_TRY(cudaStreamSynchronize(s));
    }
    if (st & GNN_DEV_BAD_OFFSETS) return GNN_ERR_BAD_OFFSETS;
    if (st & GNN_DEV_JET_TOO_LARGE) return GNN_ERR_JET_TOO_LARGE;
    return GNN_OK;
}

const char* gnn_strerror(int status) {
    switch (status) {
        case GNN_OK: return "ok";
        case GNN_ERR_NULL: return "null pointer";
        case GNN_ERR_BAD_ARCH: return "architecture field out of range";
        case GNN_ERR_BAD_BLOB_SIZE: return "weight blob size does not match the architecture";
        case GNN_ERR_BATCH_TOO_LARGE: return "batch exceeds the workspace (max_batch_jets / max_particles / slice)";
        case GNN_ERR_CUDA: return "CUDA runtime error (or no CUDA device: there is no CPU fallback)";
        case GNN_ERR_BAD_OFFSETS: return "offsets are not a valid CSR (offsets[0] != 0, not monotone, or offsets[B] != N)";
        case GNN_ERR_JET_TOO_LARGE: return "a jet has more than max_particles particles";
        case GNN_ERR_BAD_ARG: return "bad argument";
        case GNN_ERR_TIMEOUT: return "timed out";
        case GNN_ERR_QUEUE_FULL: return "batcher queue full";
        case GNN_ERR_BAD_TICKET: return "unknown or already collected ticket";
        default: return "unknown status";
    }
}

int64_t gnn_launch_count(const gnn_model* m) { return m ? m->launches.load(std::memory_order_relaxed) : 0; }

// ---- per-stage entry points ------------------------------------------------------------------------------------
int gnn_debug_knn(gnn_model* m, const float* space_dev, int32_t D, const int32_t* offsets_dev, int32_t B, int32_t N,
                  int32_t k, int32_t* idx_dev, void* cuda_stream) {
    if (!m) return GNN_ERR_NULL;
    if (B < 0 || N < 0 || D < 1 || D > 1024 || k < 1 || k > GNN_MAX_K) return GNN_ERR_BAD_ARG;
    if (B > m->arch.max_batch_jets || (int64_t)N > m->Nmax) return GNN_ERR_BATCH_TOO_LARGE;
    if (B == 0) return GNN_OK;
    if (!offsets_dev || !idx_dev || (N > 0 && !space_dev)) return GNN_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    Workspace& w = m->ws[0];
    int n = 0, rc;
    if ((rc = launch_ingest(offsets_dev, nullptr, B, N, (int)m->Nmax, m->arch.max_particles, w, s)) < 0) return rc;
    n += rc;
    // a GNN_BF16 model runs what its forward runs (grouped kernels: Gram distances for D = 64 / 128 / 256, 32-bit keys)
    if ((rc = launch_knn(space_dev, D, k, B, m->arch.max_particles, w, idx_dev, 1, m->arch.precision == GNN_BF16 ? 1 : 0, s)) < 0) return rc;
    n += rc;
    m->launches.fetch_add(n, std::memory_order_relaxed);
    return cudaGetLastError() == cudaSuccess ? GNN_OK : GNN_ERR_CUDA;
}

int gnn_debug_edgeconv(gnn_model* m, int32_t block, const float* x_dev, const int32_t* idx_dev,
                       const int32_t* offsets_dev, int32_t B, int32_t N, float* y_dev, void* cuda_stream) {
    if (!m) return GNN_ERR_NULL;
    if (block < 0 || block >= m->arch.n_blocks || B < 0 || N < 0) return GNN_ERR_BAD_ARG;
    if (B > m->arch.max_batch_jets || (int64_t)N > m->Nmax) return GNN_ERR_BATCH_TOO_LARGE;
    if (B == 0 || N == 0) return GNN_OK;
    if (!offsets_dev || !idx_dev || !x_dev || !y_dev) return GNN_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    Workspace& w = m->ws[0];
    int n = 0, rc;
    if ((rc = launch_ingest(offsets_dev, nullptr, B, N, (int)m->Nmax, m->arch.max_particles, w, s)) < 0) return rc;
    n += rc;
    if ((rc = launch_globalize_idx(idx_dev, m->arch.k, B, w, w.idx, s)) < 0) return rc;
    n += rc;
    if (m->arch.precision == GNN_BF16) rc = launch_edgeconv_bf16(*m, block, x_dev, w.idx, N, y_dev, w, s);
    else rc = launch_edgeconv_f32(m->blocks[block], m->arch.k, x_dev, w.idx, N, y_dev, w, s);
    if (rc < 0) return rc;
    n += rc;
    m->launches.fetch_add(n, std::memory_order_relaxed);
    return cudaGetLastError() == cudaSuccess ? GNN_OK : GNN_ERR_CUDA;
}

int gnn_debug_edgeconv_pool(gnn_model* m, const float* x_dev, const int32_t* idx_dev, const int32_t* offsets_dev, int32_t B,
                            int32_t N, float* g_dev, void* cuda_stream) {
    if (!m) return GNN_ERR_NULL;
    if (B < 0 || N < 0) return GNN_ERR_BAD_ARG;
    if (B > m->arch.max_batch_jets || (int64_t)N > m->Nmax) return GNN_ERR_BATCH_TOO_LARGE;
    const int block = m->arch.n_blocks - 1;
    if (m->arch.precision != GNN_BF16 || !edgeconv_bf16_can_pool(*m, block)) return GNN_ERR_BAD_ARG;
    if (B == 0) return GNN_OK;
    if (!offsets_dev || !g_dev || (N > 0 && (!idx_dev || !x_dev))) return GNN_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    Workspace& w = m->ws[0];
    const int C = m->arch.channels[block][2];
    int n = 0, rc;
    if ((rc = launch_ingest(offsets_dev, nullptr, B, N, (int)m->Nmax, m->arch.max_particles, w, s)) < 0) return rc;
    n += rc;
    GNN_CUDA_TRY(cudaMemsetAsync(w.pool, 0, (size_t)B * C * sizeof(unsigned long long), s));
    if (N > 0) {
        if ((rc = launch_globalize_idx(idx_dev, m->arch.k, B, w, w.idx, s)) < 0) return rc;
        n += rc;
        if ((rc = launch_pre_bf16(*m, block, x_dev, N, w, s, DEP_NONE)) < 0) return rc;
        n += rc;
        if ((rc = launch_edge_bf16(*m, block, w.idx, N, nullptr, w, s)) < 0) return rc;
        n += rc;
    }
    if ((rc = launch_pooled_mean(*m, B, w, g_dev, s)) < 0) return rc;
    n += rc;
    GNN_CUDA_TRY(cudaMemsetAsync(w.pool, 0, (size_t)B * C * sizeof(unsigned long long), s));   // the sums are zero between calls
    m->launches.fetch_add(n, std::memory_order_relaxed);
    return cudaGetLastError() == cudaSuccess ? GNN_OK : GNN_ERR_CUDA;
}

int gnn_debug_pool_head(gnn_model* m, const float* x_dev, const int32_t* offsets_dev, int32_t B, int32_t N,
                        float* logits_dev, void* cuda_stream) {
    if (!m) return GNN_ERR_NULL;
    if (B < 0 || N < 0) return GNN_ERR_BAD_ARG;
    if (B > m->arch.max_batch_jets || (int64_t)N > m->Nmax) return GNN_ERR_BATCH_TOO_LARGE;
    if (B == 0) return GNN_OK;
    if (!offsets_dev || !logits_dev || (N > 0 && !x_dev)) return GNN_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    Workspace& w = m->ws[0];
    int n = 0, rc;
    if ((rc = launch_ingest(offsets_dev, nullptr, B, N, (int)m->Nmax, m->arch.max_particles, w, s)) < 0) return rc;
    n += rc;
    if ((rc = launch_pool_head(*m, x_dev, B, w, logits_dev, s)) < 0) return rc;
    n += rc;
    m->launches.fetch_add(n, std::memory_order_relaxed);
    return cudaGetLastError() == cudaSuccess ? GNN_OK : GNN_ERR_CUDA;
}

}  // extern "C"

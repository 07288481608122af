// bdt.cu -- the paper's second workload: inference of a small boosted decision tree, "20 input features
// and 100 trees" (section 4.1, Fig. 6; Table C2: input shape 20, output shape 2, batches of 10 K ...
// 2.56 M).  The paper's point is that this model is NOT worth a GPU server once transfers are counted; bench.py measures both
// sides of that statement: device-resident events/s and the same through host buffers.
//
// Model (readings B1-B4; the paper only names XGBoost): n_trees complete binary trees of depth `depth`; internal
// node i of a tree tests x[feature[i]] < threshold[i]: true -> child 2 i + 1, false -> child 2 i + 2 (NaN compares false: goes
// right); the margin is the sum of the reached leaves over the trees IN TREE ORDER (fp32 here), p = 1 / (1 + exp(-margin)),
// output row = (1 - p, p).
//
// Kernel: the whole forest lives in shared memory (100 trees x (63 nodes x 8 B + 64 leaves x 4 B) = 76 KB), one thread per
// event, events staged through shared memory in tiles so that the global reads are whole 128-byte lines (rows are 80 bytes)
// and a thread's feature lookups x[f] are shared-memory reads at a row pitch of F + 1 words (conflict-free across a warp).
// Every thread walks the same instruction stream (the path is data, not control), so there is no divergence.  Per event:
// n_trees x depth dependent (node load, feature load, compare) steps = 600 for the paper's model against 88 bytes of HBM
// traffic: the kernel is bound by shared-memory / ALU issue, not by HBM (bench.py reports both).
#include "gnn_internal.h"
#include <cmath>
#include <cstring>
#include <new>

struct gnn_bdt {
    int device = 0, n_trees = 0, depth = 0, n_features = 0, n_sms = 148;
    uint2* nodes = nullptr;        // [n_trees][2^depth - 1] (feature, threshold bits)
    float* leaves = nullptr;       // [n_trees][2^depth]
    float* x_stage = nullptr;      // gnn_bdt_infer_host staging
    float* out_stage = nullptr;
    int64_t stage_events = 0;
    size_t smem = 0;
};

namespace {

constexpr int BDT_THREADS = 256;
constexpr int BDT_MAX_SMEM = 200 * 1024;   // largest forest + staging a CTA may ask for (one CTA per SM then)

__global__ void __launch_bounds__(BDT_THREADS)
bdt_kernel(const uint2* __restrict__ nodes, const float* __restrict__ leaves, int n_trees, int depth, int F,
           const float* __restrict__ x, long long N, float* __restrict__ out) {
    extern __shared__ __align__(16) unsigned char smem_bdt[];
    const int n_int = (1 << depth) - 1, n_leaf = 1 << depth;
    uint2* nd = reinterpret_cast<uint2*>(smem_bdt);                                   // [n_trees][n_int]
    float* lf = reinterpret_cast<float*>(nd + (size_t)n_trees * n_int);               // [n_trees][n_leaf]
    float* xs = lf + (size_t)n_trees * n_leaf;                                        // [BDT_THREADS][F + 1]
    for (int i = threadIdx.x; i < n_trees * n_int; i += BDT_THREADS) nd[i] = nodes[i];
    for (int i = threadIdx.x; i < n_trees * n_leaf; i += BDT_THREADS) lf[i] = leaves[i];
    const int pitch = F + 1;
    for (long long e0 = (long long)blockIdx.x * BDT_THREADS; e0 < N; e0 += (long long)gridDim.x * BDT_THREADS) {
        __syncthreads();                                         // forest loaded / previous tile consumed
        const long long n_here = min((long long)BDT_THREADS, N - e0);
        const float* src = x + e0 * F;                           // the tile's rows are contiguous: coalesced word loads
        for (int i = threadIdx.x; i < (int)n_here * F; i += BDT_THREADS) xs[(i / F) * pitch + (i % F)] = __ldg(src + i);
        __syncthreads();
        if (threadIdx.x < n_here) {
            const float* xr = xs + threadIdx.x * pitch;
            float margin = 0.0f;
            for (int t = 0; t < n_trees; ++t) {
                const uint2* tn = nd + t * n_int;
                int node = 0;
                for (int l = 0; l < depth; ++l) {
                    const uint2 nv = tn[node];
                    node = 2 * node + ((xr[nv.x] < __uint_as_float(nv.y)) ? 1 : 2);
                }
                margin += lf[t * n_leaf + (node - n_int)];       // tree order, fp32
            }
            const float p = 1.0f / (1.0f + expf(-margin));
            reinterpret_cast<float2*>(out)[e0 + threadIdx.x] = make_float2(1.0f - p, p);
        }
    }
}

}  // namespace

extern "C" {

int gnn_bdt_create(const int32_t* feature_host, const float* threshold_host, const float* leaf_host, int32_t n_trees,
                   int32_t depth, int32_t n_features, int device, gnn_bdt** out) {
    if (!feature_host || !threshold_host || !leaf_host || !out) return GNN_ERR_NULL;
    *out = nullptr;
    if (n_trees < 1 || n_trees > 4096 || depth < 1 || depth > 12 || n_features < 1 || n_features > 1024) return GNN_ERR_BAD_ARCH;
    const size_t n_int = ((size_t)1 << depth) - 1, n_leaf = (size_t)1 << depth;
    const size_t smem = (size_t)n_trees * (n_int * sizeof(uint2) + n_leaf * sizeof(float)) + (size_t)BDT_THREADS * (n_features + 1) * sizeof(float);
    if (smem > (size_t)BDT_MAX_SMEM) return GNN_ERR_BAD_ARCH;              // the forest must fit one SM's shared memory
    for (size_t i = 0; i < (size_t)n_trees * n_int; ++i)
        if (feature_host[i] < 0 || feature_host[i] >= n_features) return GNN_ERR_BAD_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        std::fprintf(stderr, "libgnn: no usable CUDA device %d (found %d); there is no CPU fallback\n", device, ndev);
        return GNN_ERR_CUDA;
    }
    GNN_CUDA_TRY(cudaSetDevice(device));
    gnn_bdt* b = new (std::nothrow) gnn_bdt();
    if (!b) return GNN_ERR_CUDA;
    b->device = device; b->n_trees = n_trees; b->depth = depth; b->n_features = n_features; b->smem = smem;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) b->n_sms = prop.multiProcessorCount;
    std::vector<uint2> nd((size_t)n_trees * n_int);
    for (size_t i = 0; i < nd.size(); ++i) {
        uint32_t bits;
        std::memcpy(&bits, &threshold_host[i], 4);
        nd[i] = make_uint2((uint32_t)feature_host[i], bits);
    }
    bool ok = cudaMalloc(&b->nodes, nd.size() * sizeof(uint2)) == cudaSuccess &&
              cudaMalloc(&b->leaves, (size_t)n_trees * n_leaf * sizeof(float)) == cudaSuccess &&
              cudaMemcpy(b->nodes, nd.data(), nd.size() * sizeof(uint2), cudaMemcpyHostToDevice) == cudaSuccess &&
              cudaMemcpy(b->leaves, leaf_host, (size_t)n_trees * n_leaf * sizeof(float), cudaMemcpyHostToDevice) == cudaSuccess &&
              // the attribute belongs to the kernel on this device, not to this forest: always the 200 KB ceiling checked
              // above, so that creating a smaller forest later never lowers the cap under an earlier, larger one
              cudaFuncSetAttribute(bdt_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, BDT_MAX_SMEM) == cudaSuccess;
    if (!ok) { gnn_bdt_destroy(b); return GNN_ERR_CUDA; }
    *out = b;
    return GNN_OK;
}

void gnn_bdt_destroy(gnn_bdt* b) {
    if (!b) return;
    cudaSetDevice(b->device);
    cudaDeviceSynchronize();
    if (b->nodes) cudaFree(b->nodes);
    if (b->leaves) cudaFree(b->leaves);
    if (b->x_stage) cudaFree(b->x_stage);
    if (b->out_stage) cudaFree(b->out_stage);
    delete b;
}

int gnn_bdt_infer(gnn_bdt* b, const float* x_dev, int64_t N, float* out_dev, void* cuda_stream) {
    if (!b) return GNN_ERR_NULL;
    if (N < 0) return GNN_ERR_BAD_ARG;
    if (N == 0) return GNN_OK;
    if (!x_dev || !out_dev) return GNN_ERR_NULL;
    if ((reinterpret_cast<uintptr_t>(out_dev) & 7u) != 0) return GNN_ERR_BAD_ARG;   // rows are stored as float2
    const long long tiles = (N + BDT_THREADS - 1) / BDT_THREADS;
    const int per_sm = std::max(1, (int)((220 * 1024) / b->smem));
    const int grid = (int)std::min<long long>(tiles, (long long)b->n_sms * per_sm);
    bdt_kernel<<<grid, BDT_THREADS, b->smem, static_cast<cudaStream_t>(cuda_stream)>>>(b->nodes, b->leaves, b->n_trees, b->depth,
                                                                                      b->n_features, x_dev, (long long)N, out_dev);
    return cudaGetLastError() == cudaSuccess ? GNN_OK : GNN_ERR_CUDA;
}

int gnn_bdt_infer_host(gnn_bdt* b, const float* x_host, int64_t N, float* out_host, void* cuda_stream) {
    if (!b) return GNN_ERR_NULL;
    if (N < 0) return GNN_ERR_BAD_ARG;
    if (N == 0) return GNN_OK;
    if (!x_host || !out_host) return GNN_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (N > b->stage_events) {                                   // staging grows to the largest batch seen (not per call)
        GNN_CUDA_TRY(cudaStreamSynchronize(s));
        if (b->x_stage) cudaFree(b->x_stage);
        if (b->out_stage) cudaFree(b->out_stage);
        b->x_stage = nullptr; b->out_stage = nullptr; b->stage_events = 0;
        GNN_CUDA_TRY(cudaMalloc(&b->x_stage, (size_t)N * b->n_features * sizeof(float)));
        GNN_CUDA_TRY(cudaMalloc(&b->out_stage, (size_t)N * 2 * sizeof(float)));
        b->stage_events = N;
    }
    GNN_CUDA_TRY(cudaMemcpyAsync(b->x_stage, x_host, (size_t)N * b->n_features * sizeof(float), cudaMemcpyHostToDevice, s));
    const int rc = gnn_bdt_infer(b, b->x_stage, N, b->out_stage, cuda_stream);
    if (rc != GNN_OK) return rc;
    GNN_CUDA_TRY(cudaMemcpyAsync(out_host, b->out_stage, (size_t)N * 2 * sizeof(float), cudaMemcpyDeviceToHost, s));
    GNN_CUDA_TRY(cudaStreamSynchronize(s));
    return GNN_OK;
}

}  // extern "C"

// pool_head.cu -- steps a7/a8: masked global average pool over the particles of a jet and the FC head
// ("two fully connected layers with 256 nodes and 0.1 dropout rate to two nodes"; L270 inference mode
// => dropout is the identity; BASELINE.json north_star (3)).  fp32 in every precision mode (R19).
// Ragged input makes the "mask" implicit: only the n_b real particles of jet b are ever stored (R7, R12).
//
// One CTA per jet: thread c sums channel c over the jet's rows (coalesced: consecutive threads read consecutive
// channels of one row), then the FC layers run as coalesced mat-vecs on the transposed weights Wt[in][out].
#include "gnn_internal.h"

namespace {

constexpr int PH_THREADS = 256;
constexpr int PH_MAXW = 1024;

struct HeadParams {
    LinF32 fc[GNN_MAX_FC + 1];
    int n_fc;
    int C;
    int n_classes;
};

__global__ void __launch_bounds__(PH_THREADS)
pool_head_kernel(const float* __restrict__ x, const int32_t* __restrict__ jet_start, const int32_t* __restrict__ jet_n,
                 const int32_t* __restrict__ meta, HeadParams hp, float* __restrict__ logits) {
    __shared__ float z0[PH_MAXW], z1[PH_MAXW];
    const int b = blockIdx.x;
    const int n = jet_n[b];
    if (meta[0] || n < 0) {                       // poisoned batch or offending jet: NaN logits (include/gnn.h)
        for (int o = threadIdx.x; o < hp.n_classes; o += PH_THREADS) logits[(size_t)b * hp.n_classes + o] = __int_as_float(0x7fc00000);
        return;
    }
    const int C = hp.C;
    const float* xb = x + (size_t)jet_start[b] * C;
    for (int c = threadIdx.x; c < C; c += PH_THREADS) {
        float s = 0.0f;
        for (int i = 0; i < n; ++i) s += xb[(size_t)i * C + c];
        z0[c] = (n > 0) ? s / (float)n : 0.0f;    // R12: empty jet pools to 0
    }
    __syncthreads();
    float* zin = z0; float* zout = z1;
    for (int l = 0; l < hp.n_fc; ++l) {
        const LinF32 L = hp.fc[l];
        const bool last = (l == hp.n_fc - 1);
        for (int o = threadIdx.x; o < L.N; o += PH_THREADS) {
            float acc = 0.0f;
            for (int c = 0; c < L.K; ++c) acc = fmaf(zin[c], __ldg(L.Wt + (size_t)c * L.ld + o), acc);
            acc += __ldg(L.shift + o);
            if (last) logits[(size_t)b * hp.n_classes + o] = acc;
            else zout[o] = fmaxf(acc, 0.0f);
        }
        __syncthreads();
        float* t = zin; zin = zout; zout = t;
    }
}

}  // namespace

int launch_pool_head(const gnn_model& m, const float* x, int B, const Workspace& w, float* logits, cudaStream_t s) {
    if (B == 0) return 0;
    HeadParams hp;
    hp.n_fc = m.n_fc;
    for (int i = 0; i < m.n_fc; ++i) hp.fc[i] = m.fc[i];
    hp.C = m.arch.channels[m.arch.n_blocks - 1][2];
    hp.n_classes = m.arch.n_classes;
    pool_head_kernel<<<B, PH_THREADS, 0, s>>>(x, w.jet_start, w.jet_n, w.meta, hp, logits);
    return 1;
}

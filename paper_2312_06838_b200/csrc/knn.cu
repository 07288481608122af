// knn.cu -- steps a1/a3/a5: exact per-jet k nearest neighbours ("k=16 nearest neighbors", L97
// "dynamic graph"; BASELINE.json north_star (1): pairwise distances in shared memory, top-k with ties broken by the
// lower index; on (eta, phi) for block 1 and on the features for later blocks).
//
// One CTA per jet.  Readings: R3 squared Euclidean, direct differences (R18: no Gram form -- its
// cancellation error exceeds the 1e-5 near-tie band); R4 self excluded by index; R5 strict order on (d, j); R6
// k_eff = min(k, n-1).  fp32 arithmetic, d = fma(t, t, d) with t = s_i - s_j, dimensions summed in index order.
//
// Phase 1 (ALU-bound): each thread owns 4x4 (query x candidate) register tiles; rows of the space are staged in
//   shared memory with a row stride of D+4 floats so that the eight lanes of a quarter-warp reading eight
//   consecutive rows with LDS.128 hit eight different 16-byte bank groups.  Distances go to a [n][n+1] matrix in
//   shared memory with d_ii = +inf.
// Phase 2: one thread per query walks its row and keeps the k smallest 64-bit keys (float bits of d << 32 | j) in a
//   sorted register list -- d >= 0, so unsigned order on the bits is numeric order and equal distances fall back
//   to the lower index for free.  (The paper-era "warp-level top-k" is replaced by this: see DESIGN.md.)
#include "gnn_internal.h"
#include <cfloat>

namespace {

constexpr int KNN_THREADS = 256;

template <int K>
__device__ __forceinline__ void topk_insert(unsigned long long (&best)[K], unsigned long long key) {
    // best[] ascending; key < best[K-1] is known
#pragma unroll
    for (int m = K - 1; m >= 0; --m) {
        unsigned long long lo = (m > 0) ? best[m - 1] : 0ull;
        bool shift = (m > 0) && (key < lo);
        bool place = (key < best[m]) && !shift;
        if (shift) best[m] = lo;
        else if (place) best[m] = key;
    }
}

template <int K>
__global__ void __launch_bounds__(KNN_THREADS)
knn_kernel(const float* __restrict__ space, int D, int k, const int32_t* __restrict__ jet_start,
           const int32_t* __restrict__ jet_n, const int32_t* __restrict__ meta, int32_t* __restrict__ idx_out,
           int local_out) {
    extern __shared__ __align__(16) float smem[];
    if (meta[0]) return;
    const int b = blockIdx.x;
    const int n = jet_n[b];
    const int start = jet_start[b];
    if (n < -1) {                             // offending ragged jet (jet_n = -multiplicity): its packed rows exist and
        for (int e = threadIdx.x; e < -n * k; e += KNN_THREADS)   // the point-tiled EdgeConv walks them: no neighbours
            idx_out[(size_t)start * k + e] = -1;
        return;
    }
    if (n <= 0) return;                       // empty jet (or offending padded jet, which owns no rows)
    const int Dp = (D + 3) & ~3;
    const int ld = Dp + 4;                    // row stride in floats
    const int n4 = (n + 3) & ~3;
    float* S = smem;                          // [n4][ld]
    float* Dm = smem + (size_t)n4 * ld;       // [n][n+1]
    const int ldd = n + 1;

    // stage rows (coalesced over the contiguous [n, D] span of the jet), zero the padding
    const float* src = space + (size_t)start * D;
    for (int e = threadIdx.x; e < n4 * Dp; e += KNN_THREADS) {
        int r = e / Dp, c = e - r * Dp;
        S[r * ld + c] = (r < n && c < D) ? src[(size_t)r * D + c] : 0.0f;
    }
    __syncthreads();

    // phase 1: 4x4 register tiles.  Thread-tile (ig, jg) covers query rows ig + nG*r and candidate rows jg + nG*r.
    const int nG = n4 >> 2;
    for (int t = threadIdx.x; t < nG * nG; t += KNN_THREADS) {
        const int ig = t / nG, jg = t - ig * nG;
        float acc[4][4];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[a][c] = 0.0f;
        const float* pi = S + ig * ld;
        const float* pj = S + jg * ld;
        for (int c0 = 0; c0 < Dp; c0 += 4) {
            float4 qi[4], qj[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                qi[r] = *reinterpret_cast<const float4*>(pi + (size_t)r * nG * ld + c0);
                qj[r] = *reinterpret_cast<const float4*>(pj + (size_t)r * nG * ld + c0);
            }
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    float t0 = qi[a].x - qj[c].x; acc[a][c] = fmaf(t0, t0, acc[a][c]);
                    float t1 = qi[a].y - qj[c].y; acc[a][c] = fmaf(t1, t1, acc[a][c]);
                    float t2 = qi[a].z - qj[c].z; acc[a][c] = fmaf(t2, t2, acc[a][c]);
                    float t3 = qi[a].w - qj[c].w; acc[a][c] = fmaf(t3, t3, acc[a][c]);
                }
        }
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            int i = ig + nG * a;
            if (i >= n) continue;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                int j = jg + nG * c;
                if (j < n) Dm[i * ldd + j] = (i == j) ? INFINITY : acc[a][c];
            }
        }
    }
    __syncthreads();

    // phase 2: thread i selects for query i
    for (int i = threadIdx.x; i < n; i += KNN_THREADS) {
        unsigned long long best[K];
#pragma unroll
        for (int m = 0; m < K; ++m) best[m] = ~0ull;
        const float* row = Dm + i * ldd;
        for (int j = 0; j < n; ++j) {
            if (j == i) continue;                                       // R4: by index
            unsigned long long key = ((unsigned long long)__float_as_uint(row[j]) << 32) | (unsigned)j;
            if (key < best[K - 1]) topk_insert<K>(best, key);
        }
        int32_t* out = idx_out + (size_t)(start + i) * k;
        const int base = local_out ? 0 : start;
#pragma unroll
        for (int m = 0; m < K; ++m)
            if (m < k) out[m] = (best[m] == ~0ull) ? -1 : (int32_t)(best[m] & 0xffffffffull) + base;
    }
}

size_t knn_smem_bytes(int D, int P) {
    int Dp = (D + 3) & ~3, ld = Dp + 4, n4 = (P + 3) & ~3;
    return ((size_t)n4 * ld + (size_t)P * (P + 1)) * sizeof(float);
}

template <int K>
int launch_knn_t(const float* space, int D, int k, int B, int P, const Workspace& w, int32_t* idx_out, int local_out,
                 cudaStream_t s) {
    knn_kernel<K><<<B, KNN_THREADS, knn_smem_bytes(D, P), s>>>(space, D, k, w.jet_start, w.jet_n, w.meta, idx_out, local_out);
    return 1;
}

}  // namespace

int launch_knn(const float* space, int D, int k, int B, int max_particles, const Workspace& w, int32_t* idx_out,
               int local_out, cudaStream_t s) {
    if (B == 0) return 0;
    if (knn_smem_bytes(D, max_particles) > 227 * 1024) return GNN_ERR_BAD_ARG;
    if (k <= 4) return launch_knn_t<4>(space, D, k, B, max_particles, w, idx_out, local_out, s);
    if (k <= 8) return launch_knn_t<8>(space, D, k, B, max_particles, w, idx_out, local_out, s);
    if (k <= 16) return launch_knn_t<16>(space, D, k, B, max_particles, w, idx_out, local_out, s);
    return launch_knn_t<32>(space, D, k, B, max_particles, w, idx_out, local_out, s);
}

// debug entry: jet-local neighbour indices -> the global ones the EdgeConv kernels read (out-of-jet values -> -1)
__global__ void globalize_idx_kernel(const int32_t* __restrict__ idx_local, int k, const int32_t* __restrict__ jet_start,
                                     const int32_t* __restrict__ jet_n, const int32_t* __restrict__ meta,
                                     int32_t* __restrict__ idx_global) {
    if (meta[0]) return;
    const int b = blockIdx.x;
    int n = jet_n[b];
    const int start = jet_start[b];
    const int rows = n < -1 ? -n : n;
    for (int e = threadIdx.x; e < rows * k; e += blockDim.x) {
        int j = idx_local[(size_t)start * k + e];
        idx_global[(size_t)start * k + e] = (n > 0 && j >= 0 && j < n) ? j + start : -1;
    }
}

int launch_globalize_idx(const int32_t* idx_local, int k, int B, const Workspace& w, int32_t* idx_global, cudaStream_t s) {
    if (B == 0) return 0;
    globalize_idx_kernel<<<B, 128, 0, s>>>(idx_local, k, w.jet_start, w.jet_n, w.meta, idx_global);
    return 1;
}

// opt every instantiation into the full 227 KB of dynamic shared memory (called once from gnn_create)
int knn_configure() {
    const int lim = 227 * 1024;
    if (cudaFuncSetAttribute(knn_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) != cudaSuccess) return GNN_ERR_CUDA;
    if (cudaFuncSetAttribute(knn_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) != cudaSuccess) return GNN_ERR_CUDA;
    if (cudaFuncSetAttribute(knn_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) != cudaSuccess) return GNN_ERR_CUDA;
    if (cudaFuncSetAttribute(knn_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) != cudaSuccess) return GNN_ERR_CUDA;
    return GNN_OK;
}

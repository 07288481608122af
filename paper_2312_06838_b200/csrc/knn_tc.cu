// knn_tc.cu -- GNN_BF16 mode only: the pairwise squared distances of steps a3/a5 (kNN in the feature space of the previous
// block, D = 64 / 128 / 256) as a per-jet Gram matrix on the tensor cores.  BASELINE.json north_star sets no neighbour-set
// bar for this mode (R20: the features it ranks already carry the bf16 path's 2^-8 relative noise), so the
// distance may take the Gram form the fp32 validation mode must avoid (R18):
//     d(i, j) = G_ii + G_jj - 2 G_ij,   G = Xc Xc^T,   Xc = tf32(x - mean over the jet's particles)
// Centering keeps |Xc| at the spread of the jet, so the cancellation error of the Gram form (~2^-10 |Xc|^2) stays below
// the gaps between neighbour distances; the diagonal comes from the same product, so d(i, i) = 0 and d is symmetric
// bit for bit (knn_select_kernel reads d(j, i) for d(i, j)); d is clamped at 0 (the selection orders float bits).
// One CTA per jet: the jet is staged by cp.async, centred / rounded / swizzled in place into a K-major operand tile, one
// thread issues M = 128, N = n rounded up to 16, K = D tcgen05.mma kind::tf32 with A = B = that tile, 128 threads
// (thread = row = TMEM lane) turn G into d and store whole 128-byte segments of dm.  Latency is hidden by CTAs per SM.
#include "gnn_internal.h"
#include "tc05.cuh"

namespace {

using namespace tc05;

constexpr int KTC_THREADS = 160;         // warps 0-3: load + epilogue; warp 4: TMEM owner + MMA issuer

template <int D>
struct KnnTcCfg {
    static constexpr int KBD = D / 32;                         // K blocks of 32 tf32 (128 bytes per row)
    static constexpr int XK_BYTES = 128 * 128;
    static constexpr int SMEM_BYTES = KBD * XK_BYTES + D * 4 + 128 * 4 + 2 * 8 + 16;
};

template <int D>
__global__ void __launch_bounds__(KTC_THREADS)
knn_gram_kernel(const float* __restrict__ space, const int32_t* __restrict__ jet_start, const int32_t* __restrict__ jet_n,
                const int32_t* __restrict__ meta, float* __restrict__ dm, int pld, int2* __restrict__ pjet) {
    using Cfg = KnnTcCfg<D>;
    constexpr int KBD = Cfg::KBD;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    if (meta[0]) return;
    const int b = blockIdx.x;
    const int n = jet_n[b];
    const int start = jet_start[b];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (n < -1) {                             // offending ragged jet: owns -n rows; only the particle -> jet map is needed
        for (int r = tid; r < -n; r += KTC_THREADS) pjet[start + r] = make_int2(start, n);
        return;
    }
    if (n <= 0) return;
    uint8_t* X = smem_raw;                    // [KBD][128 rows][32 tf32], 128B-swizzled
    if ((smem_u32(X) & 1023u) != 0u) __trap();
    float* mean_s = reinterpret_cast<float*>(X + KBD * Cfg::XK_BYTES);   // [D]
    float* diag_s = mean_s + D;                                          // [128]
    uint64_t* bars = reinterpret_cast<uint64_t*>(diag_s + 128);
    uint64_t* d_full = bars;
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(bars + 2);
    if (tid == 0) { mbar_init(d_full, 1); fence_mbar_init(); }
    if (warp == 4) tmem_alloc(tmem_ptr, 128);
    if (tid < n) pjet[start + tid] = make_int2(start, n);
    const float* src = space + (size_t)start * D;
    // (1) the jet's rows, raw fp32, into the tile buffer with ONE round trip to memory: 16-byte cp.async per (row, chunk),
    //     all in flight (x of the previous block has usually left L2 by now: a dependent walk costs ~1 us per step)
    constexpr int CPR = D / 4;                                  // 16-byte chunks per row
    for (int e = tid; e < n * CPR; e += KTC_THREADS) {
        const int r = e / CPR, c = e - r * CPR;                  // chunk c of row r: K block c / 8, chunk c % 8 of its line
        const unsigned sa = smem_u32(X + (c >> 3) * Cfg::XK_BYTES + r * 128 + ((c & 7) << 4));
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(src + (size_t)r * D + 4 * c) : "memory");
    }
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_ptr;
    // (2) column means from shared memory (lanes = consecutive columns: conflict-free)
    for (int c = tid; c < D; c += KTC_THREADS) {
        const float* colp = reinterpret_cast<const float*>(X + (c >> 5) * Cfg::XK_BYTES) + (c & 31);
        float s0 = 0.0f, s1 = 0.0f;
        int r = 0;
        for (; r + 1 < n; r += 2) { s0 += colp[r * 32]; s1 += colp[(r + 1) * 32]; }
        if (r < n) s0 += colp[r * 32];
        mean_s[c] = (s0 + s1) / (float)n;
    }
    __syncthreads();
    // (3) in place: centre, round to tf32 (RNA), apply the 128-byte swizzle.  One thread owns a whole 128-byte line (row, K
    //     block): it reads the eight chunks, then writes them permuted.  Rows >= n keep whatever the buffer held: row i of
    //     A and row j of B only reach G_ij, and no entry with i >= n or j >= n is ever read back.
    for (int e = tid; e < n * KBD; e += KTC_THREADS) {
        const int r = e / KBD, kb = e - r * KBD;
        uint8_t* line = X + kb * Cfg::XK_BYTES + r * 128;
        uint4 o[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const float4 v = *reinterpret_cast<const float4*>(line + (c << 4));
            const float4 mu = *reinterpret_cast<const float4*>(mean_s + kb * 32 + 4 * c);
            asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(o[c].x) : "f"(v.x - mu.x));
            asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(o[c].y) : "f"(v.y - mu.y));
            asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(o[c].z) : "f"(v.z - mu.z));
            asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(o[c].w) : "f"(v.w - mu.w));
        }
#pragma unroll
        for (int c = 0; c < 8; ++c) *reinterpret_cast<uint4*>(line + ((c ^ (r & 7)) << 4)) = o[c];
    }
    fence_proxy_async();
    __syncthreads();
    const int n16 = (n + 15) & ~15;
    if (warp == 4 && lane == 0) {
        tc_fence_after();
        const uint32_t idesc = idesc_tf32_f32(128, n16);
        const uint32_t x_addr = smem_u32(X);
#pragma unroll
        for (int kb = 0; kb < KBD; ++kb)
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
                const uint64_t ad = desc_sw128(x_addr + kb * Cfg::XK_BYTES + ks * 32);
                mma_tf32_ss(tmem, ad, ad, idesc, (kb | ks) != 0);
            }
        mma_commit(d_full);
    }
    if (warp < 4) {
        // thread = row i = TMEM lane; diagonal first (G_ii sits in this thread's own row), then d(i, j) slab by slab
        mbar_wait(d_full, 0);
        tc_fence_after();
        const int i = 32 * warp + lane;
        const uint32_t tbase = tmem + ((uint32_t)(32 * warp) << 16);
        float gii = 0.0f;
        {
            float v[32];
            tmem_ld32(tbase + 32 * warp, v);   // columns 32*warp .. +31 hold the diagonal entries of this warp's rows
            tmem_ld_wait();
#pragma unroll
            for (int c = 0; c < 32; ++c) gii = (c == lane) ? v[c] : gii;
        }
        diag_s[i] = gii;
        asm volatile("bar.sync 1, 128;" ::: "memory");
        float* out = dm + (size_t)(start + i) * pld;
        for (int s = 0; s * 32 < n; ++s) {
            float v[32];
            tmem_ld32(tbase + s * 32, v);
            tmem_ld_wait();
            if (i < n) {
#pragma unroll
                for (int c = 0; c < 32; c += 4) {
                    const int j = s * 32 + c;
                    if (j < n && j < pld) {
                        const float4 gj = *reinterpret_cast<const float4*>(diag_s + j);
                        *reinterpret_cast<float4*>(out + j) =
                            make_float4(fmaxf(fmaf(-2.0f, v[c], gii + gj.x), 0.0f), fmaxf(fmaf(-2.0f, v[c + 1], gii + gj.y), 0.0f),
                                        fmaxf(fmaf(-2.0f, v[c + 2], gii + gj.z), 0.0f), fmaxf(fmaf(-2.0f, v[c + 3], gii + gj.w), 0.0f));
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 4) tmem_dealloc(tmem, 128);
}

template <int D>
int launch_gram(const float* space, int B, const Workspace& w, int pld, cudaStream_t s) {
    knn_gram_kernel<D><<<B, KTC_THREADS, KnnTcCfg<D>::SMEM_BYTES, s>>>(space, w.jet_start, w.jet_n, w.meta, w.dm, pld, w.pjet);
    return 1;
}

}  // namespace

// distances of every jet in `space` [N, D] into w.dm (and the particle -> jet map); returns 0 if D has no tensor-core form
int launch_knn_gram(const float* space, int D, int B, int max_particles, const Workspace& w, cudaStream_t s) {
    const int pld = (max_particles + 3) & ~3;
    switch (D) {
        case 64: return launch_gram<64>(space, B, w, pld, s);
        case 128: return launch_gram<128>(space, B, w, pld, s);
        case 256: return launch_gram<256>(space, B, w, pld, s);
        default: return 0;
    }
}

int knn_tc_configure() {
    if (cudaFuncSetAttribute(knn_gram_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, KnnTcCfg<64>::SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(knn_gram_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, KnnTcCfg<128>::SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(knn_gram_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, KnnTcCfg<256>::SMEM_BYTES) != cudaSuccess)
        return GNN_ERR_CUDA;
    return GNN_OK;
}

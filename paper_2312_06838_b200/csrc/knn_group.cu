// knn_group.cu -- steps a1/a3/a5 in GNN_BF16 mode: per-jet k nearest neighbours, distances and selection in ONE kernel,
// several jets per CTA ("k=16 nearest neighbors", L97 "dynamic graph"; BASELINE.json north_star (1):
// pairwise distances on chip, top-k with ties broken by the lower index; on (eta, phi) for block 1 and on the features
// for later blocks).
//
// Work unit = a GROUP of consecutive whole jets whose rows fit one 128-row tile (schedule built by ingest_kernel:
// ~3 jets of the configs' <n> = 40 per group, so ~110 of the 128 rows are busy instead of 40 with one jet per CTA).
// thread = row = one particle; its candidates are the columns [c0, c1) of its own jet inside the tile.
//   knn_group_gram_kernel<D, K>   feature spaces, D = 64 / 128 / 256 (R28): the tile's pairwise inner products as
//       ONE tcgen05.mma chain (kind::tf32, M = 128, N = rows rounded up to 16, K = D, A = B = the tile) into TMEM;
//       d(i, j) = G_ii + G_jj - 2 G_ij on rows centred on their JET's mean (centring keeps the cancellation error of the
//       Gram form below the neighbour gaps, and per-jet means keep a jet's result independent of its group mates, so
//       batch-composition invariance stays bitwise).  The distance matrix never leaves the SM: each thread reads its row
//       of G from TMEM 16 columns at a time and selects in registers.
//   knn_group_coords_kernel<K>    spaces of <= 4 dimensions (the coordinates of block 1): exact direct differences in
//       fp32 from shared memory, same selection.
// Selection: 32-bit keys (float bits of d with the low 7 mantissa bits replaced by the jet-local index j < 128: d to 16
// mantissa bits, ties and near-ties within 2^-16 relative go to the lower index).  Candidates arrive in chunks of K:
// a chunk is ordered by a bitonic network in registers and merged with the running best-K list as
// min(best[m], chunk[K-1-m]) + log2(K) half-cleaner stages -- ~15 data-independent instructions per candidate, no
// divergence, instead of ~40 for a sorted insert that some lane of the warp nearly always needs.
// Output: idx [N, k] GLOBAL row indices in ascending (d, j) order (R29), -1 = none (k_eff < k); pjid [N] = jet of a row.
#include "gnn_internal.h"
#include "tc05.cuh"

namespace {

using namespace tc05;

constexpr int KG_ROWS = 128;
constexpr int KG_MAX_JETS = 16;           // = GROUP_MAX_JETS of ingest.cu
constexpr unsigned KEY_NONE = 0xffffffffu;

template <int K>
__device__ __forceinline__ void bitonic_sort_asc(unsigned (&c)[K]) {
#pragma unroll
    for (int size = 2; size <= K; size <<= 1)
#pragma unroll
        for (int st = size >> 1; st > 0; st >>= 1)
#pragma unroll
            for (int m = 0; m < K; ++m) {
                const int o = m ^ st;
                if (o > m) {
                    const bool asc = (m & size) == 0;
                    const unsigned a = c[m], b = c[o];
                    const unsigned lo = min(a, b), hi = max(a, b);
                    c[m] = asc ? lo : hi;
                    c[o] = asc ? hi : lo;
                }
            }
}

// best[] ascending, c[] any order: best <- the K smallest of the union, ascending
template <int K>
__device__ __forceinline__ void merge_chunk(unsigned (&best)[K], unsigned (&c)[K]) {
    bitonic_sort_asc<K>(c);
#pragma unroll
    for (int m = 0; m < K; ++m) best[m] = min(best[m], c[K - 1 - m]);        // bitonic: the K smallest of the union
#pragma unroll
    for (int st = K / 2; st >= 1; st >>= 1)
#pragma unroll
        for (int m = 0; m < K; ++m)
            if ((m & st) == 0) {
                const unsigned a = best[m], b = best[m + st];
                best[m] = min(a, b);
                best[m + st] = max(a, b);
            }
}

__device__ __forceinline__ unsigned make_key(float d, int jl) { return (__float_as_uint(d) & ~0x7fu) | (unsigned)jl; }

// group descriptor in shared memory, filled by every kernel the same way
struct GroupInfo {
    int ls[KG_MAX_JETS];          // first row of jet t inside the tile
    int rows[KG_MAX_JETS];        // its rows (0 for empty / offending jets)
    int r0, R, j0, nj;            // first packed row, rows in the tile, first jet, jets
    int special;                  // offending ragged jet (owns more rows than max_particles): no neighbours
};

// returns false if the CTA has nothing to compute (also handles the offending-jet group: idx = -1, pjid)
__device__ __forceinline__ bool load_group(GroupInfo* gi, const int2* __restrict__ groups, const int32_t* __restrict__ jet_start,
                                           const int32_t* __restrict__ jet_n, const int32_t* __restrict__ meta,
                                           int32_t* __restrict__ idx_out, int32_t* __restrict__ pjid, int k) {
    if ((int)blockIdx.x >= meta[2]) return false;               // meta[2] = 0 for a poisoned batch
    const int tid = threadIdx.x;
    // one round trip: every thread of the first warp reads the group, lane t then reads jet t (all loads independent)
    if (tid < 32) {
        const int2 g = __ldg(groups + blockIdx.x);
        int n = 0, st = 0;
        if (tid < g.y) { n = __ldg(jet_n + g.x + tid); st = __ldg(jet_start + g.x + tid); }
        const int r0 = __shfl_sync(0xffffffffu, st, 0), n0 = __shfl_sync(0xffffffffu, n, 0);
        const int end = n > 0 ? st - r0 + n : 0;
        const int R = __reduce_max_sync(0xffffffffu, end);
        if (tid < KG_MAX_JETS) { gi->ls[tid] = st - r0; gi->rows[tid] = n > 0 ? n : 0; }
        if (tid == 0) { gi->j0 = g.x; gi->nj = g.y; gi->r0 = r0; gi->R = R; gi->special = (n0 < -1) ? -n0 : 0; }
    }
    __syncthreads();
    if (gi->special) {                                          // its packed rows exist and the point-tiled EdgeConv walks them
        const int rows = gi->special;
        for (int e = tid; e < rows * k; e += blockDim.x) idx_out[(size_t)gi->r0 * k + e] = -1;
        if (pjid) for (int r = tid; r < rows; r += blockDim.x) pjid[gi->r0 + r] = gi->j0;
        return false;
    }
    return gi->R > 0;
}

// row -> (jet slot, c0, c1) by a scan over the <= 16 jets of the group
__device__ __forceinline__ void row_range(const GroupInfo* gi, int i, int& t_out, int& c0, int& c1) {
    t_out = 0; c0 = 0; c1 = 0;
    for (int t = 0; t < gi->nj; ++t) {
        const int a = gi->ls[t], b = a + gi->rows[t];
        if (i >= a && i < b) { t_out = t; c0 = a; c1 = b; }
    }
}

template <int K>
__device__ __forceinline__ void write_neighbours(const unsigned (&best)[K], int32_t* __restrict__ out, int k, int base) {
    if (k == K && K >= 4) {
#pragma unroll
        for (int m = 0; m < K; m += 4) {
            int4 v;
            v.x = best[m] == KEY_NONE ? -1 : (int)(best[m] & 0x7fu) + base;
            v.y = best[m + 1] == KEY_NONE ? -1 : (int)(best[m + 1] & 0x7fu) + base;
            v.z = best[m + 2] == KEY_NONE ? -1 : (int)(best[m + 2] & 0x7fu) + base;
            v.w = best[m + 3] == KEY_NONE ? -1 : (int)(best[m + 3] & 0x7fu) + base;
            *reinterpret_cast<int4*>(out + m) = v;
        }
    } else {
#pragma unroll
        for (int m = 0; m < K; ++m)
            if (m < k) out[m] = best[m] == KEY_NONE ? -1 : (int)(best[m] & 0x7fu) + base;
    }
}

// ---- coordinates (D <= 4): exact direct differences ----------------------------------------------------------------------
constexpr int KC_THREADS = 128;

template <int K>
__global__ void __launch_bounds__(KC_THREADS)
knn_group_coords_kernel(const float* __restrict__ space, int D, const int32_t* __restrict__ jet_start,
                        const int32_t* __restrict__ jet_n, const int32_t* __restrict__ meta, const int2* __restrict__ groups,
                        int32_t* __restrict__ idx_out, int32_t* __restrict__ pjid, int k, int local_out) {
    __shared__ GroupInfo gi;
    __shared__ float4 xs[KG_ROWS];
    if (!load_group(&gi, groups, jet_start, jet_n, meta, idx_out, pjid, k)) return;
    const int i = threadIdx.x, R = gi.R;
    float4 xi = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    if (i < R) {
        const float* src = space + (size_t)(gi.r0 + i) * D;
        xi.x = __ldg(src);
        if (D > 1) xi.y = __ldg(src + 1);
        if (D > 2) xi.z = __ldg(src + 2);
        if (D > 3) xi.w = __ldg(src + 3);
    }
    xs[i] = xi;
    int t, c0, c1;
    row_range(&gi, i, t, c0, c1);
    if (i >= R) { c0 = 0; c1 = 0; }
    if (i < R && pjid) pjid[gi.r0 + i] = gi.j0 + t;
    __syncthreads();
    unsigned best[K];
#pragma unroll
    for (int m = 0; m < K; ++m) best[m] = KEY_NONE;
    // every lane walks ITS jet's candidates from c0 in chunks of K; the trip count is the warp's largest
    const int trips = (c1 - c0 + K - 1) / K;
    const int wtrips = __reduce_max_sync(0xffffffffu, trips);
    for (int tr = 0; tr < wtrips; ++tr) {
        unsigned c[K];
#pragma unroll
        for (int u = 0; u < K; ++u) {
            const int j = c0 + tr * K + u;
            const float4 xj = xs[min(j, KG_ROWS - 1)];
            // t = s_i - s_j, d = fma(t, t, d) in index order: the arithmetic of the exact path (knn.cu); padded dimensions add 0
            float tt = xi.x - xj.x, d = tt * tt;
            tt = xi.y - xj.y; d = fmaf(tt, tt, d);
            tt = xi.z - xj.z; d = fmaf(tt, tt, d);
            tt = xi.w - xj.w; d = fmaf(tt, tt, d);
            c[u] = (j < c1 && j != i) ? make_key(d, j - c0) : KEY_NONE;      // R4: self excluded by index
        }
        merge_chunk<K>(best, c);
    }
    if (i < R) write_neighbours<K>(best, idx_out + (size_t)(gi.r0 + i) * k, k, local_out ? 0 : gi.r0 + c0);
}

// ---- feature spaces: Gram matrix on the tensor cores -------------------------------------------------------------------------
// warps 0-3: thread = row = TMEM lane (selection); warps 4-7 help with the load, the means and the centring pass; warp 4 owns
// the TMEM allocation and its lane 0 issues the MMAs
constexpr int KG_THREADS = 256;
constexpr int KG_MMA_WARP = 4;

template <int D>
struct KnnGroupCfg {
    static constexpr int KBD = D / 32;                         // K blocks of 32 tf32 (128 bytes per row)
    static constexpr int XK_BYTES = KG_ROWS * 128;
    static constexpr int X_BYTES = KBD * XK_BYTES;
    static constexpr int MEAN_BYTES = KG_MAX_JETS * D * 4;
    static constexpr int SMEM_BYTES = X_BYTES + MEAN_BYTES + KG_ROWS * 4 + KG_ROWS + (int)sizeof(GroupInfo) + 2 * 8 + 16 + 64;
};

template <int D, int K>
__global__ void __launch_bounds__(KG_THREADS)
knn_group_gram_kernel(const float* __restrict__ space, const int32_t* __restrict__ jet_start, const int32_t* __restrict__ jet_n,
                      const int32_t* __restrict__ meta, const int2* __restrict__ groups, int32_t* __restrict__ idx_out,
                      int32_t* __restrict__ pjid, int k, int local_out) {
    using Cfg = KnnGroupCfg<D>;
    constexpr int KBD = Cfg::KBD;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* X = smem_raw;                    // [KBD][128 rows][32 tf32], 128B-swizzled after the centring pass
    float* mean_s = reinterpret_cast<float*>(X + Cfg::X_BYTES);                 // [KG_MAX_JETS][D]
    float* diag_s = mean_s + KG_MAX_JETS * D;                                   // [128]
    uint8_t* rowjet_s = reinterpret_cast<uint8_t*>(diag_s + KG_ROWS);           // [128] jet slot of a row
    GroupInfo* gi = reinterpret_cast<GroupInfo*>(rowjet_s + KG_ROWS);
    uint64_t* d_full = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(gi) + ((sizeof(GroupInfo) + 7) & ~7));
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(d_full + 1);
#ifdef KNN_TRACE
    unsigned long long tr[10]; int trn = 0;
#define KTR() do { if (threadIdx.x == 0) tr[trn++] = global_timer_ns(); } while (0)
#else
#define KTR() do { } while (0)
#endif
    KTR();
    if (!load_group(gi, groups, jet_start, jet_n, meta, idx_out, pjid, k)) return;
    KTR();
    if ((smem_u32(X) & 1023u) != 0u) __trap();
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int R = gi->R, r0 = gi->r0;
    if (tid == 0) { mbar_init(d_full, 1); fence_mbar_init(); }
    if (warp == KG_MMA_WARP) tmem_alloc(tmem_ptr, 128);
    // (1) the tile's rows, raw fp32, with ONE round trip to memory: 16-byte cp.async per (row, chunk), all in flight
    const float* src = space + (size_t)r0 * D;
    constexpr int CPR = D / 4;                                  // 16-byte chunks per row
    for (int e = tid; e < R * CPR; e += KG_THREADS) {
        const int r = e / CPR, c = e - r * CPR;                  // chunk c of row r: K block c / 8, chunk c % 8 of its line
        const unsigned sa = smem_u32(X + (c >> 3) * Cfg::XK_BYTES + r * 128 + ((c & 7) << 4));
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(src + (size_t)r * D + 4 * c) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    int jt = 0, c0 = 0, c1 = 0;
    if (tid < KG_ROWS) {
        row_range(gi, tid, jt, c0, c1);
        if (tid >= R) { c0 = 0; c1 = 0; }
        rowjet_s[tid] = (uint8_t)jt;
        if (tid < R && pjid) pjid[r0 + tid] = gi->j0 + jt;
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    KTR();
    const uint32_t tmem = *tmem_ptr;
    // (2) per-jet column means (lanes = consecutive columns: conflict-free); a jet's sum has a fixed order (four chains by the
    //     row's index inside the jet modulo 4, combined as (s0 + s2) + (s1 + s3)), so it does not depend on the group
    for (int e = tid; e < D * gi->nj; e += KG_THREADS) {
        const int t = e / D, c = e - t * D;
        const int a = gi->ls[t], n = gi->rows[t];
        const float* colp = reinterpret_cast<const float*>(X + (c >> 5) * Cfg::XK_BYTES) + a * 32 + (c & 31);
        float s0 = 0.0f, s1 = 0.0f, s2 = 0.0f, s3 = 0.0f;
        int r = 0;
        for (; r + 3 < n; r += 4) { s0 += colp[r * 32]; s1 += colp[(r + 1) * 32]; s2 += colp[(r + 2) * 32]; s3 += colp[(r + 3) * 32]; }
        if (r < n) s0 += colp[r * 32];
        if (r + 1 < n) s1 += colp[(r + 1) * 32];
        if (r + 2 < n) s2 += colp[(r + 2) * 32];
        mean_s[t * D + c] = n > 0 ? ((s0 + s2) + (s1 + s3)) / (float)n : 0.0f;
    }
    __syncthreads();
    KTR();
    // (3) in place: centre on the jet's mean, round to tf32 (RNA), apply the 128-byte swizzle.  One thread per 16-byte chunk,
    //     the eight lanes of a quarter-warp on one 128-byte line (row, K block): they read it whole (eight bank groups) and
    //     write it back permuted among themselves (chunk c -> c ^ (row & 7): again eight bank groups); the line's loads have
    //     all landed before its first store issues (same warp, same instruction).  Rows >= R keep whatever the buffer
    //     held: row i of A and row j of B only reach G_ij, and no entry with i >= R or j >= R is ever used.
    for (int e = tid; e < R * KBD * 8; e += KG_THREADS) {
        const int c = e & 7, l = e >> 3;
        const int kb = l / R, r = l - kb * R;
        uint8_t* line = X + kb * Cfg::XK_BYTES + r * 128;
        const float4 v = *reinterpret_cast<const float4*>(line + (c << 4));
        const float4 mu = *reinterpret_cast<const float4*>(mean_s + (int)rowjet_s[r] * D + kb * 32 + 4 * c);
        uint4 o;
        asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(o.x) : "f"(v.x - mu.x));
        asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(o.y) : "f"(v.y - mu.y));
        asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(o.z) : "f"(v.z - mu.z));
        asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(o.w) : "f"(v.w - mu.w));
        *reinterpret_cast<uint4*>(line + ((c ^ (r & 7)) << 4)) = o;
    }
    fence_proxy_async();
    __syncthreads();
    KTR();
    const int n16 = (R + 15) & ~15;
    if (warp == KG_MMA_WARP && lane == 0) {
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
        // thread = row i = TMEM lane; diagonal first (G_ii sits in this thread's own row), then the row of G 16 columns at a time
        mbar_wait(d_full, 0);
        tc_fence_after();
        KTR();
        const int i = tid;
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
        // columns any lane of this warp needs (warp-uniform: tcgen05.ld is warp-collective), aligned to the chunk width
        constexpr int CW = K < 16 ? 16 : K;
        const int lo = __reduce_min_sync(0xffffffffu, c1 > c0 ? c0 : KG_ROWS) & ~(CW - 1);
        const int hi = __reduce_max_sync(0xffffffffu, c1);
        unsigned best[K];
#pragma unroll
        for (int m = 0; m < K; ++m) best[m] = KEY_NONE;
        for (int cs = lo; cs < hi; cs += CW) {
            unsigned key[CW];
#pragma unroll
            for (int h = 0; h < CW / 16; ++h) {
                float v[16];
                tmem_ld16(tbase + cs + 16 * h, v);
                tmem_ld_wait();
#pragma unroll
                for (int u = 0; u < 16; u += 4) {
                    const int j = cs + 16 * h + u;
                    const float4 gj = *reinterpret_cast<const float4*>(diag_s + j);
                    const float gjv[4] = {gj.x, gj.y, gj.z, gj.w};
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const float d = fmaxf(fmaf(-2.0f, v[u + q], gii + gjv[q]), 0.0f);
                        const int jj = j + q;
                        key[16 * h + u + q] = (jj >= c0 && jj < c1 && jj != i) ? make_key(d, jj - c0) : KEY_NONE;   // R4
                    }
                }
            }
#pragma unroll
            for (int sub = 0; sub < CW / K; ++sub) {
                unsigned c[K];
#pragma unroll
                for (int u = 0; u < K; ++u) c[u] = key[sub * K + u];
                merge_chunk<K>(best, c);
            }
        }
        KTR();
        if (i < R) write_neighbours<K>(best, idx_out + (size_t)(r0 + i) * k, k, local_out ? 0 : r0 + c0);
    }
    tc_fence_before();
    __syncthreads();
    KTR();
#ifdef KNN_TRACE
    if (threadIdx.x == 0 && (blockIdx.x % 97) == 5)
        printf("knn<%d> cta %d R %d: group %llu load %llu mean %llu centre %llu mma %llu select %llu store %llu (ns)\n", D, blockIdx.x, R,
               tr[1] - tr[0], tr[2] - tr[1], tr[3] - tr[2], tr[4] - tr[3], tr[5] - tr[4], tr[6] - tr[5], tr[7] - tr[6]);
#endif
    if (warp == KG_MMA_WARP) tmem_dealloc(tmem, 128);
}

template <int K>
int launch_group_t(const float* space, int D, int k, int B, const Workspace& w, int32_t* idx_out, int local_out, cudaStream_t s) {
    // one CTA per possible group (at most one per jet); CTAs beyond meta[2] leave at once
    if (D <= 4) {
        knn_group_coords_kernel<K><<<B, KC_THREADS, 0, s>>>(space, D, w.jet_start, w.jet_n, w.meta, w.groups, idx_out, w.pjid, k, local_out);
        return 1;
    }
    switch (D) {
        case 64: knn_group_gram_kernel<64, K><<<B, KG_THREADS, KnnGroupCfg<64>::SMEM_BYTES, s>>>(space, w.jet_start, w.jet_n, w.meta, w.groups, idx_out, w.pjid, k, local_out); return 1;
        case 128: knn_group_gram_kernel<128, K><<<B, KG_THREADS, KnnGroupCfg<128>::SMEM_BYTES, s>>>(space, w.jet_start, w.jet_n, w.meta, w.groups, idx_out, w.pjid, k, local_out); return 1;
        case 256: knn_group_gram_kernel<256, K><<<B, KG_THREADS, KnnGroupCfg<256>::SMEM_BYTES, s>>>(space, w.jet_start, w.jet_n, w.meta, w.groups, idx_out, w.pjid, k, local_out); return 1;
        default: return 0;
    }
}

template <int D, int K>
bool configure_one() {
    return cudaFuncSetAttribute(knn_group_gram_kernel<D, K>, cudaFuncAttributeMaxDynamicSharedMemorySize, KnnGroupCfg<D>::SMEM_BYTES) == cudaSuccess &&
           cudaFuncSetAttribute(knn_group_gram_kernel<D, K>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared) == cudaSuccess;
}
template <int K>
bool configure_k() { return configure_one<64, K>() && configure_one<128, K>() && configure_one<256, K>(); }

}  // namespace

// kNN of every jet in `space` [N, D] through the grouped kernels; returns the number of kernels enqueued, or 0 if this
// (D, max_particles) has no grouped form (the caller then takes the exact path of knn.cu)
int launch_knn_group(const float* space, int D, int k, int B, int max_particles, const Workspace& w, int32_t* idx_out,
                     int local_out, cudaStream_t s) {
    if (max_particles > KG_ROWS || !(D <= 4 || D == 64 || D == 128 || D == 256)) return 0;
    if (B == 0) return 0;
    if (k <= 4) return launch_group_t<4>(space, D, k, B, w, idx_out, local_out, s);
    if (k <= 8) return launch_group_t<8>(space, D, k, B, w, idx_out, local_out, s);
    if (k <= 16) return launch_group_t<16>(space, D, k, B, w, idx_out, local_out, s);
    return launch_group_t<32>(space, D, k, B, w, idx_out, local_out, s);
}

int knn_group_configure() {
    return (configure_k<4>() && configure_k<8>() && configure_k<16>() && configure_k<32>()) ? GNN_OK : GNN_ERR_CUDA;
}

// knn_group.cu -- steps a1/a3/a5 in GNN_BF16 mode: per-jet k nearest neighbours, distances and selection in ONE kernel,
// several jets per CTA ("k=16 nearest neighbors", L97 "dynamic graph"; BASELINE.json north_star (1):
// pairwise distances on chip, top-k with ties broken by the lower index; on (eta, phi) for block 1 and on the features
// for later blocks).
//
// Work unit = a GROUP of consecutive whole jets whose rows fit one 128-row tile (schedule built by ingest_kernel:
// ~3 jets of the configs' <n> = 40 per group, so ~110 of the 128 rows are busy instead of 40 with one jet per CTA).
// thread = row = one particle; its candidates are the columns [c0, c1) of its own jet inside the tile.
//   knn_group_gram_kernel<D, K>   feature spaces, D = 64 / 128 / 256 (R28): the tile's pairwise inner products as
//       ONE tcgen05.mma chain (kind::f16 on fp16 operands, M = 128, N = rows rounded up to 16, K = D, A = B = the tile) into
//       TMEM; d(i, j) = G_ii + G_jj - 2 G_ij on rows centred on the FIRST ROW OF THEIR JET (a reference inside the jet keeps
//       the cancellation error of the Gram form below the neighbour gaps, costs no pass over the tile, and depends on
//       nothing but the jet, so batch-composition invariance stays bitwise).  The distance matrix never leaves the SM: each
//       thread reads its row of G from TMEM 16 columns at a time and selects in registers.
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
#include <algorithm>

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

// group `grp` (< meta[2]) -> *gi; returns false if there is nothing to compute (also handles the offending-jet group: idx = -1, pjid)
__device__ __forceinline__ bool load_group(GroupInfo* gi, const int2* __restrict__ groups, const int32_t* __restrict__ jet_start,
                                           const int32_t* __restrict__ jet_n, const int32_t* __restrict__ meta,
                                           int32_t* __restrict__ idx_out, int32_t* __restrict__ pjid, int k, int grp) {
    const int tid = threadIdx.x;
    // one round trip: every thread of the first warp reads the group, lane t then reads jet t (all loads independent)
    if (tid < 32) {
        const int2 g = __ldg(groups + grp);
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
                        int32_t* __restrict__ idx_out, int32_t* __restrict__ pjid, int k, int local_out, int dep) {
    __shared__ GroupInfo gi;
    __shared__ float4 xs[KG_ROWS];
    if (dep == DEP_PRIMARY) { grid_dep_wait(); grid_dep_launch(); }
    const int n_groups = meta[2];                               // 0 for a poisoned batch
    for (int grp = blockIdx.x; grp < n_groups; grp += gridDim.x) {
        if (load_group(&gi, groups, jet_start, jet_n, meta, idx_out, pjid, k, grp)) {
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
        __syncthreads();                                        // gi and xs are rewritten by the next group
    }
    if (dep == DEP_SECONDARY && blockIdx.x == 0) grid_dep_wait();
}

// ---- feature spaces: Gram matrix on the tensor cores -------------------------------------------------------------------------
// four warps: thread = row = TMEM lane; warp 0 owns
// the TMEM allocation and its lane 0 issues the MMAs
constexpr int KG_THREADS = 128;
constexpr int KG_MMA_WARP = 0;
constexpr int KG_BATCH = 4;                // items a thread has in flight (one or two round trips per tile)

template <int D>
struct KnnGroupCfg {
    static constexpr int KBD = D / 64;                         // K blocks of 64 fp16 (128 bytes per row)
    static constexpr int XK_BYTES = KG_ROWS * 128;
    static constexpr int X_BYTES = KBD * XK_BYTES;
    static constexpr int SMEM_BYTES = X_BYTES + KG_ROWS * 4 + KG_ROWS * 4 + (int)sizeof(GroupInfo) + 2 * 8 + 16 + 64;
};

// 128 threads (thread = row): a CTA is small enough in registers for several to sit on an SM BESIDE the pre kernel's CTA, so the
// groups of a batch run in one or two waves while the two kernels of a block run side by side
template <int D, int K>
__global__ void __launch_bounds__(KG_THREADS)
knn_group_gram_kernel(const float* __restrict__ space, const int32_t* __restrict__ jet_start, const int32_t* __restrict__ jet_n,
                      const int32_t* __restrict__ meta, const int2* __restrict__ groups, int32_t* __restrict__ idx_out,
                      int32_t* __restrict__ pjid, int k, int local_out, int dep) {
    using Cfg = KnnGroupCfg<D>;
    constexpr int KBD = Cfg::KBD;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* X = smem_raw;                    // [KBD][128 rows][64 fp16], 128B-swizzled: the centred rows
    float* diag_s = reinterpret_cast<float*>(X + Cfg::X_BYTES);                 // [128]
    int* ref_s = reinterpret_cast<int*>(diag_s + KG_ROWS);                      // [128] first row (inside the tile) of a row's jet
    GroupInfo* gi = reinterpret_cast<GroupInfo*>(ref_s + KG_ROWS);
    uint64_t* d_full = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(gi) + ((sizeof(GroupInfo) + 7) & ~7));
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(d_full + 1);
#ifdef KNN_TRACE
    unsigned long long tr[10]; int trn = 0;
#define KTR() do { if (threadIdx.x == 0) tr[trn++] = global_timer_ns(); } while (0)
#else
#define KTR() do { } while (0)
#endif
    if ((smem_u32(X) & 1023u) != 0u) __trap();
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) { mbar_init(d_full, 1); fence_mbar_init(); }
    if (warp == KG_MMA_WARP) tmem_alloc(tmem_ptr, 128);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_ptr;
    if (dep == DEP_PRIMARY) { grid_dep_wait(); grid_dep_launch(); }   // (DEP_SECONDARY: see gnn_internal.h)
    const int n_groups = meta[2];                               // 0 for a poisoned batch
    int iter = 0;
    for (int grp = blockIdx.x; grp < n_groups; grp += gridDim.x, ++iter) {
    KTR();
    const bool work = load_group(gi, groups, jet_start, jet_n, meta, idx_out, pjid, k, grp);
    KTR();
    if (work) {
    const int R = gi->R, r0 = gi->r0;
    int jt = 0, c0 = 0, c1 = 0;
    if (tid < KG_ROWS) {
        row_range(gi, tid, jt, c0, c1);
        if (tid >= R) { c0 = 0; c1 = 0; }
        ref_s[tid] = c0;
        if (tid < R && pjid) pjid[r0 + tid] = gi->j0 + jt;
    }
    __syncthreads();
    KTR();
    // (1) the tile's rows CENTRED ON THE FIRST ROW OF THEIR JET, rounded to fp16 (RNE; 10 mantissa bits as tf32) and stored with
    //     the 128-byte swizzle.  d(i, j) is translation invariant, so any per-jet reference point is legitimate; moving the
    //     origin into the jet keeps the cancellation error of the Gram form (G_ii + G_jj - 2 G_ij) below the neighbour gaps,
    //     and a reference that is a row of the jet itself needs no pass over the tile (no column sums, no staging of the
    //     raw rows) and depends on nothing but the jet: batch-composition invariance stays bitwise.  One item = 8 columns
    //     of a row: its own 32 bytes and the reference row's, all loads of a thread in flight together (one round trip).
    //     Rows >= R keep whatever the buffer held: row i of A and row j of B only reach G_ij, and no entry with i >= R or
    //     j >= R is ever used.
    const float* src = space + (size_t)r0 * D;
    constexpr int IPR = D / 8;                                  // items per row
    constexpr int ITEMS = (KG_ROWS * IPR + KG_THREADS - 1) / KG_THREADS;
    const int n_items = R * IPR;
#pragma unroll
    for (int i0 = 0; i0 < ITEMS; i0 += KG_BATCH) {
        float4 xa[KG_BATCH], xb[KG_BATCH], ra[KG_BATCH], rb[KG_BATCH];
#pragma unroll
        for (int u = 0; u < KG_BATCH; ++u) {
            const int e = tid + (i0 + u) * KG_THREADS;
            if (i0 + u < ITEMS && e < n_items) {
                const int r = e / IPR, c = e - r * IPR;
                const float4* xp = reinterpret_cast<const float4*>(src + (size_t)r * D + 8 * c);
                const float4* rp = reinterpret_cast<const float4*>(src + (size_t)ref_s[r] * D + 8 * c);
                xa[u] = __ldg(xp); xb[u] = __ldg(xp + 1); ra[u] = __ldg(rp); rb[u] = __ldg(rp + 1);
            }
        }
#pragma unroll
        for (int u = 0; u < KG_BATCH; ++u) {
            const int e = tid + (i0 + u) * KG_THREADS;
            if (i0 + u < ITEMS && e < n_items) {
                const int r = e / IPR, c = e - r * IPR;
                uint4 o;
                o.x = pack_f16x2(xa[u].x - ra[u].x, xa[u].y - ra[u].y);
                o.y = pack_f16x2(xa[u].z - ra[u].z, xa[u].w - ra[u].w);
                o.z = pack_f16x2(xb[u].x - rb[u].x, xb[u].y - rb[u].y);
                o.w = pack_f16x2(xb[u].z - rb[u].z, xb[u].w - rb[u].w);
                *reinterpret_cast<uint4*>(X + (c >> 3) * Cfg::XK_BYTES + r * 128 + (((c & 7) ^ (r & 7)) << 4)) = o;
            }
        }
    }
    fence_proxy_async();
    __syncthreads();
    KTR();
    const int n16 = (R + 15) & ~15;
    if (warp == KG_MMA_WARP && lane == 0) {
        tc_fence_after();
        const uint32_t idesc = idesc_f16_f32(128, n16);
        const uint32_t x_addr = smem_u32(X);
#pragma unroll
        for (int kb = 0; kb < KBD; ++kb)
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {                     // K = 16 fp16 = 32 bytes per step
                const uint64_t ad = desc_sw128(x_addr + kb * Cfg::XK_BYTES + ks * 32);
                mma_bf16_ss(tmem, ad, ad, idesc, (kb | ks) != 0);    // kind::f16; the descriptor says fp16 operands
            }
        mma_commit(d_full);
    }
    if (warp < 4) {
        // thread = row i = TMEM lane; diagonal first (G_ii sits in this thread's own row), then the row of G 16 columns at a time
        mbar_wait(d_full, iter & 1);
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
        tc_fence_before();
    }
    }   // work
    __syncthreads();                                            // the tile, gi, ref_s, diag_s and the accumulator are reused
    tc_fence_after();
    KTR();
#ifdef KNN_TRACE
    if (threadIdx.x == 0 && (blockIdx.x % 97) == 5 && work)
        printf("knn<%d> cta %d R %d: group %llu rows %llu centre %llu mma %llu select %llu store %llu (ns)\n", D, blockIdx.x, gi->R,
               tr[1] - tr[0], tr[2] - tr[1], tr[3] - tr[2], tr[4] - tr[3], tr[5] - tr[4], tr[6] - tr[5]);
    trn = 0;
#endif
    }   // groups
    tc_fence_before();
    __syncthreads();
    if (warp == KG_MMA_WARP) tmem_dealloc(tmem, 128);
    if (dep == DEP_SECONDARY && blockIdx.x == 0) grid_dep_wait();
}

template <int K>
int launch_group_t(const float* space, int D, int k, int B, const Workspace& w, int32_t* idx_out, int local_out, int dep, cudaStream_t s) {
    // one CTA per possible group (at most one per jet); CTAs beyond meta[2] leave at once
    const bool pdl = dep != DEP_NONE;
    cudaError_t e;
    if (D <= 4) {
        e = launch_k(knn_group_coords_kernel<K>, dim3(B), dim3(KC_THREADS), 0, s, pdl, space, D, w.jet_start, w.jet_n, w.meta, w.groups, idx_out, w.pjid, k, local_out, dep);
    } else if (D == 64) {
        e = launch_k(knn_group_gram_kernel<64, K>, dim3(B), dim3(KG_THREADS), KnnGroupCfg<64>::SMEM_BYTES, s, pdl, space, w.jet_start, w.jet_n, w.meta, w.groups, idx_out, w.pjid, k, local_out, dep);
    } else if (D == 128) {
        e = launch_k(knn_group_gram_kernel<128, K>, dim3(B), dim3(KG_THREADS), KnnGroupCfg<128>::SMEM_BYTES, s, pdl, space, w.jet_start, w.jet_n, w.meta, w.groups, idx_out, w.pjid, k, local_out, dep);
    } else if (D == 256) {
        e = launch_k(knn_group_gram_kernel<256, K>, dim3(B), dim3(KG_THREADS), KnnGroupCfg<256>::SMEM_BYTES, s, pdl, space, w.jet_start, w.jet_n, w.meta, w.groups, idx_out, w.pjid, k, local_out, dep);
    } else {
        return 0;
    }
    return e == cudaSuccess ? 1 : GNN_ERR_CUDA;
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
bool knn_group_supported(int D, int max_particles) {
    return max_particles <= KG_ROWS && (D <= 4 || D == 64 || D == 128 || D == 256);
}

// dep: DEP_* of gnn_internal.h (forward() only; DEP_NONE = an ordinary launch)
int launch_knn_group(const float* space, int D, int k, int B, int max_particles, const Workspace& w, int32_t* idx_out,
                     int local_out, int dep, cudaStream_t s) {
    if (!knn_group_supported(D, max_particles)) return 0;
    if (B == 0) return 0;
    if (k <= 4) return launch_group_t<4>(space, D, k, B, w, idx_out, local_out, dep, s);
    if (k <= 8) return launch_group_t<8>(space, D, k, B, w, idx_out, local_out, dep, s);
    if (k <= 16) return launch_group_t<16>(space, D, k, B, w, idx_out, local_out, dep, s);
    return launch_group_t<32>(space, D, k, B, w, idx_out, local_out, dep, s);
}

int knn_group_configure() {
    return (configure_k<4>() && configure_k<8>() && configure_k<16>() && configure_k<32>()) ? GNN_OK : GNN_ERR_CUDA;
}

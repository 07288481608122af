// knn.cu -- steps a1/a3/a5: exact per-jet k nearest neighbours ("k=16 nearest neighbors", L97
// "dynamic graph"; BASELINE.json north_star (1): pairwise distances in shared memory, top-k with ties broken by the
// lower index; on (eta, phi) for block 1 and on the features for later blocks).
//
// Exact path (GNN_FP32_VALIDATION, and gnn_debug_knn on spaces the grouped kernels of knn_group.cu do not take).
// Readings: R3 squared Euclidean, direct differences (R18: no Gram form -- its cancellation error
// exceeds the 1e-5 near-tie band); R4 self excluded by index; R5 strict order on (d, j); R6 k_eff = min(k, n-1).
// fp32 arithmetic, d = fma(t, t, d) with t = s_i - s_j, dimensions summed in index order.
//
// knn_dist_kernel (spaces of more than 4 dimensions): one CTA per (jet, group of query rows), groups sized so that a
//   typical jet is one CTA with ~100 busy threads; the jet's rows are staged 32 dimensions at a time ([n4][36] floats,
//   double-buffered with cp.async); each thread owns up to two 4x4 (query x candidate) register tiles; distances go to the
//   global (L2-resident) matrix dm [N][pld] and the particle -> jet map pjet is written on the way.
// knn_select_kernel: TWO threads per particle of the packed batch (even / odd candidates).  Each orders its first K
//   candidates with a bitonic network in registers and inserts the rest into the sorted list of 64-bit keys
//   (float bits of d << 32 | j: d >= 0, so unsigned order on the bits is numeric order and equal distances fall back to the
//   lower index); the halves are merged through one shuffle per slot.  Spaces of <= 4 dimensions (the coordinates of
//   block 1) skip the matrix: the selection computes d(i, j) on the fly with the same arithmetic.
#include "gnn_internal.h"
#include <cfloat>
#include <mutex>

namespace {

constexpr int KNN_THREADS = 128;
constexpr int KNN_QT = 32;      // queries per CTA
constexpr int KNN_DC = 32;      // dimensions staged per chunk
constexpr int KNN_LD = KNN_DC + 4;

// Selection keys: (float bits of d) << 32 | j -- exact lexicographic (d, j) order (d >= 0, so unsigned order on the bits is
// numeric order).
struct Key64 {
    typedef unsigned long long T;
    static __device__ __forceinline__ T none() { return ~0ull; }
    static __device__ __forceinline__ T make(float d, int j) { return ((T)__float_as_uint(d) << 32) | (unsigned)j; }
    static __device__ __forceinline__ int index(T k) { return (int)(k & 0xffffffffull); }
};

template <int K, typename KT>
__device__ __forceinline__ void topk_insert(KT (&best)[K], KT key) {
    // best[] ascending; key < best[K-1] is known
#pragma unroll
    for (int m = K - 1; m >= 0; --m) {
        KT lo = (m > 0) ? best[m - 1] : (KT)0;
        bool shift = (m > 0) && (key < lo);
        bool place = (key < best[m]) && !shift;
        if (shift) best[m] = lo;
        else if (place) best[m] = key;
    }
}

__global__ void __launch_bounds__(KNN_THREADS)
knn_dist_kernel(const float* __restrict__ space, int D, const int32_t* __restrict__ jet_start,
                const int32_t* __restrict__ jet_n, const int32_t* __restrict__ meta, float* __restrict__ dm, int pld,
                int2* __restrict__ pjet, int tiles_per_jet) {
    extern __shared__ __align__(16) float smem[];
    if (meta[0]) return;
    const int b = blockIdx.x / tiles_per_jet, qt = blockIdx.x - b * tiles_per_jet;
    const int n = jet_n[b];
    const int start = jet_start[b];
    if (n < -1) {                             // offending ragged jet: owns -n rows; only the particle -> jet map is needed
        for (int r = qt * KNN_THREADS + threadIdx.x; r < -n; r += tiles_per_jet * KNN_THREADS) pjet[start + r] = make_int2(start, n);
        return;
    }
    if (n <= 0) return;                       // empty jet (or offending padded jet, which owns no rows)
    const int n4 = (n + 3) & ~3;
    const int nG = n4 >> 2;                   // groups of four candidates (and of four queries)
    // query groups per CTA: as many as fill 256 thread-tiles, so that a typical jet (n ~ 40) is ONE CTA with ~100 busy
    // threads and no padded queries; ceil(nG / gpc) <= ceil(P / 32) CTAs of a jet have work
    const int gpc = min(nG, 256 / nG);
    const int q0 = qt * 4 * gpc;
    if (q0 >= n) return;
    if ((int)threadIdx.x < 4 * gpc && q0 + (int)threadIdx.x < n) pjet[start + q0 + threadIdx.x] = make_int2(start, n);
    float* S0 = smem;                         // [2][n4][KNN_LD] double-buffered chunk of dimensions of every row of the jet
    float* Dm = dm + (size_t)(start + q0) * pld;  // rows of this tile's queries in the global distance matrix
    const float* src = space + (size_t)start * D;

    // staging of dimensions [c0, c0 + 32): 16-byte cp.async when the rows are 16-byte aligned (D % 4 == 0), so a whole
    // chunk is in flight without register staging; rows >= n and the tail of the last chunk are zero
    auto stage = [&](int c0, float* Sb) {
        const int dc = min(KNN_DC, D - c0), dc4 = (dc + 3) & ~3;
        if ((D & 3) == 0) {
            const int nq = dc4 >> 2;
            for (int e = threadIdx.x; e < n4 * nq; e += KNN_THREADS) {
                const int r = (nq == 8) ? (e >> 3) : e / nq, c = e - r * nq;
                float* dst = Sb + r * KNN_LD + 4 * c;
                if (r < n) {
                    const unsigned sa = (unsigned)__cvta_generic_to_shared(dst);
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(src + (size_t)r * D + c0 + 4 * c) : "memory");
                } else {
                    *reinterpret_cast<float4*>(dst) = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                }
            }
        } else {
            for (int e = threadIdx.x; e < n4 * dc4; e += KNN_THREADS) {
                const int r = e / dc4, c = e - r * dc4;
                Sb[r * KNN_LD + c] = (r < n && c < dc) ? __ldg(src + (size_t)r * D + c0 + c) : 0.0f;
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    // phase 1: thread-tile (ig, jg) covers queries q0 + ig + gpc*a and candidates jg + nG*c (a, c = 0..3)
    const int n_tt = gpc * nG;                // <= 256: at most two tiles per thread
    float acc[2][4][4];
#pragma unroll
    for (int u = 0; u < 2; ++u)
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[u][a][c] = 0.0f;
    stage(0, S0);
    for (int c0 = 0, ci = 0; c0 < D; c0 += KNN_DC, ++ci) {
        const int dc = min(KNN_DC, D - c0), dc4 = (dc + 3) & ~3;
        const float* S = S0 + (size_t)(ci & 1) * n4 * KNN_LD;
        if (c0 + KNN_DC < D) {
            stage(c0 + KNN_DC, S0 + (size_t)((ci + 1) & 1) * n4 * KNN_LD);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncthreads();
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int tt = threadIdx.x + u * KNN_THREADS;
            if (tt < n_tt) {
                const int ig = tt / nG, jg = tt - ig * nG;
                const float* pi = S + (q0 + ig) * KNN_LD;
                const float* pj = S + jg * KNN_LD;
                for (int cc = 0; cc < dc4; cc += 4) {
                    float4 qi[4], qj[4];
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        const int qr = min(q0 + ig + gpc * r, n4 - 1) - (q0 + ig);   // tail tile: clamp (result unused)
                        qi[r] = *reinterpret_cast<const float4*>(pi + qr * KNN_LD + cc);
                        qj[r] = *reinterpret_cast<const float4*>(pj + r * nG * KNN_LD + cc);
                    }
#pragma unroll
                    for (int a = 0; a < 4; ++a)
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            float t0 = qi[a].x - qj[c].x; acc[u][a][c] = fmaf(t0, t0, acc[u][a][c]);
                            float t1 = qi[a].y - qj[c].y; acc[u][a][c] = fmaf(t1, t1, acc[u][a][c]);
                            float t2 = qi[a].z - qj[c].z; acc[u][a][c] = fmaf(t2, t2, acc[u][a][c]);
                            float t3 = qi[a].w - qj[c].w; acc[u][a][c] = fmaf(t3, t3, acc[u][a][c]);
                        }
                }
            }
        }
        __syncthreads();                      // this buffer is restaged two chunks from now
    }
#pragma unroll
    for (int u = 0; u < 2; ++u) {
        const int tt = threadIdx.x + u * KNN_THREADS;
        if (tt < n_tt) {
            const int ig = tt / nG, jg = tt - ig * nG;
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                const int qi = ig + gpc * a;                      // query within the tile
                if (q0 + qi >= n) continue;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const int j = jg + nG * c;
                    if (j < n) Dm[(size_t)qi * pld + j] = acc[u][a][c];
                }
            }
        }
    }
}

// Phase 2, its own kernel so that every lane of every warp has work: TWO threads per particle of the packed batch
// (even / odd candidates), each keeping the k smallest of its half as a sorted register list; the k smallest of the
// union are then { min(A[m], B[K-1-m]) }, a bitonic sequence that log2(K) half-cleaner stages sort in registers.  d(i, j) is read as d(j, i) (the matrix is exactly
// symmetric: (a-b)^2 and (b-a)^2 round identically), so a warp's consecutive queries read consecutive addresses.
constexpr int KSEL_THREADS = 128;
// FLY (spaces of at most 4 dimensions: the coordinates of block 1): no distance matrix, d(i, j) is computed from the rows of
// `space` with the arithmetic of knn_dist_kernel (t = s_i - s_j, d = fma(t, t, d) in index order), so both give the same bits.
template <int K, typename KEY, bool FLY>
__global__ void __launch_bounds__(KSEL_THREADS)
knn_select_kernel(const float* __restrict__ dm, int pld, const float* __restrict__ space, int D, int k, const int2* __restrict__ pjet, const int32_t* __restrict__ jet_start,
                  const int32_t* __restrict__ jet_n, const int32_t* __restrict__ meta, int32_t* __restrict__ idx_out,
                  int local_out) {
    if (meta[0]) return;
    const int t = blockIdx.x * KSEL_THREADS + threadIdx.x;
    const int q = t >> 1, half = t & 1;
    const bool live = q < meta[1];
    int2 pi = make_int2(0, -1);
    if (live) pi = __ldg(pjet + q);                             // (start, n) of the jet that owns row q, written with the distances
    // lanes that reach the pair merge below, decided while the warp is still converged (the per-lane loops over n diverge,
    // and independent thread scheduling does not promise reconvergence before the shuffle)
    const unsigned pm = __ballot_sync(0xffffffffu, live && pi.y >= 0);
    if (!live) return;                                          // both lanes of a pair leave together
    const int n = pi.y, start = pi.x;
    int32_t* out = idx_out + (size_t)q * k;
    if (n < 0) {                              // offending ragged jet (jet_n = -multiplicity): its packed rows exist and the
        for (int m = half; m < k; m += 2) out[m] = -1;            // point-tiled EdgeConv walks them: no neighbours
        return;
    }
    const int i = q - start;
    const float* col = dm + (size_t)start * pld + i;
    float qx[4] = {0.0f, 0.0f, 0.0f, 0.0f};
    if (FLY) {
        for (int c = 0; c < D; ++c) qx[c] = __ldg(space + (size_t)q * D + c);
    }
    auto dist = [&](int j) -> float {
        if (!FLY) return __ldg(col + (size_t)j * pld);
        const float* sj = space + (size_t)(start + j) * D;
        float d = 0.0f;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const float t = qx[c] - (c < D ? __ldg(sj + c) : 0.0f);
            d = fmaf(t, t, d);
        }
        return d;
    };
    // the first K candidates of this half (j = half, half + 2, ...) are loaded together and ordered by a bitonic network
    // in registers (a sorted insert costs ~100 instructions, the whole K = 16 network ~500); later ones are inserted
    typedef typename KEY::T KT;
    KT best[K];
    float dn[8];                              // the eight candidates after the first K ride the same round trip to memory
    {
        float d[K];
#pragma unroll
        for (int u = 0; u < K; ++u) {
            const int j = half + 2 * u;
            d[u] = (j < n) ? dist(j) : 0.0f;
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int j = half + 2 * (K + u);
            dn[u] = (j < n) ? dist(j) : 0.0f;
        }
#pragma unroll
        for (int u = 0; u < K; ++u) {
            const int j = half + 2 * u;
            best[u] = (j < n && j != i) ? KEY::make(d[u], j) : KEY::none();   // R4
        }
    }
#pragma unroll
    for (int size = 2; size <= K; size <<= 1)
#pragma unroll
        for (int st = size >> 1; st > 0; st >>= 1)
#pragma unroll
            for (int m = 0; m < K; ++m) {
                const int o = m ^ st;
                if (o > m) {
                    const bool asc = (m & size) == 0 || size == K;
                    const KT a = best[m], c = best[o];
                    const bool sw = asc ? (c < a) : (a < c);
                    best[m] = sw ? c : a;
                    best[o] = sw ? a : c;
                }
            }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        const int j = half + 2 * (K + u);
        if (j >= n || j == i) continue;
        const KT key = KEY::make(dn[u], j);
        if (key < best[K - 1]) topk_insert<K, KT>(best, key);
    }
    int j = half + 2 * (K + 8);
    for (; j + 14 < n; j += 16) {             // eight loads in flight per thread
        float d[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) d[u] = dist(j + 2 * u);
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (j + 2 * u == i) continue;                               // R4: by index
            const KT key = KEY::make(d[u], j + 2 * u);
            if (key < best[K - 1]) topk_insert<K, KT>(best, key);
        }
    }
    if (j < n) {                              // tail: up to eight more, predicated
        float d[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) d[u] = (j + 2 * u < n) ? dist(j + 2 * u) : 0.0f;
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (j + 2 * u >= n || j + 2 * u == i) continue;
            const KT key = KEY::make(d[u], j + 2 * u);
            if (key < best[K - 1]) topk_insert<K, KT>(best, key);
        }
    }
    // merge with the partner lane: slot m of the merge is min(A[m], B[K-1-m]); both lanes end up with the same set
    __syncwarp(pm);
    const int base = local_out ? 0 : start;
    KT r[K];
#pragma unroll
    for (int m = 0; m < K; ++m) {
        const KT mine = half ? best[K - 1 - m] : best[m];
        const KT other = __shfl_xor_sync(pm, mine, 1);
        r[m] = mine < other ? mine : other;
    }
    // r[] is bitonic: log2(K) half-cleaner stages sort it ascending (same order as a single sorted list would give)
#pragma unroll
    for (int st = K / 2; st >= 1; st >>= 1)
#pragma unroll
        for (int m = 0; m < K; ++m)
            if ((m & st) == 0) {
                const KT a = r[m], c = r[m + st];
                const bool sw = c < a;
                r[m] = sw ? c : a;
                r[m + st] = sw ? a : c;
            }
#pragma unroll
    for (int m = 0; m < K; ++m)
        if (m < k && (m & 1) == half) out[m] = (r[m] == KEY::none()) ? -1 : KEY::index(r[m]) + base;
}

// particle -> jet map for the on-the-fly selection: one thread per jet writes its rows (offending ragged jets own rows too)
__global__ void pjet_kernel(int B, const int32_t* __restrict__ jet_start, const int32_t* __restrict__ jet_n,
                            const int32_t* __restrict__ meta, int2* __restrict__ pjet) {
    if (meta[0]) return;
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const int n = jet_n[b], start = jet_start[b];
    const int rows = n < -1 ? -n : (n > 0 ? n : 0);
    for (int r = 0; r < rows; ++r) pjet[start + r] = make_int2(start, n);
}

size_t knn_smem_bytes(int P) {
    const int n4 = (P + 3) & ~3;
    return (size_t)2 * n4 * KNN_LD * sizeof(float);
}

template <int K>
int launch_knn_t(const float* space, int D, int k, int B, int P, const Workspace& w, int32_t* idx_out, int local_out,
                 cudaStream_t s) {
    const int tiles = (P + KNN_QT - 1) / KNN_QT;
    const int pld = (P + 3) & ~3;
    const long long n_upper = 2ll * B * P;                     // two threads per particle slot
    const unsigned grid = (unsigned)((n_upper + KSEL_THREADS - 1) / KSEL_THREADS);
    if (D <= 4) {
        // coordinates (block 1): distances on the fly inside the selection; the particle -> jet map comes from its own kernel
        pjet_kernel<<<(B + 127) / 128, 128, 0, s>>>(B, w.jet_start, w.jet_n, w.meta, w.pjet);
        knn_select_kernel<K, Key64, true><<<grid, KSEL_THREADS, 0, s>>>(w.dm, pld, space, D, k, w.pjet, w.jet_start, w.jet_n, w.meta, idx_out, local_out);
        return 2;
    }
    knn_dist_kernel<<<B * tiles, KNN_THREADS, knn_smem_bytes(P), s>>>(space, D, w.jet_start, w.jet_n, w.meta, w.dm, pld, w.pjet, tiles);
    knn_select_kernel<K, Key64, false><<<grid, KSEL_THREADS, 0, s>>>(w.dm, pld, space, D, k, w.pjet, w.jet_start, w.jet_n, w.meta, idx_out, local_out);
    return 2;
}

}  // namespace

int launch_knn(const float* space, int D, int k, int B, int max_particles, const Workspace& w, int32_t* idx_out,
               int local_out, int gram, cudaStream_t s, int dep) {
    if (B == 0) return 0;
    if (gram) {                               // bf16 mode: grouped kernels where they have a form for this space
        const int n = launch_knn_group(space, D, k, B, max_particles, w, idx_out, local_out, dep, s);
        if (n != 0) return n;
    }
    if (knn_smem_bytes(max_particles) > 227 * 1024) return GNN_ERR_BAD_ARG;
    if (k <= 4) return launch_knn_t<4>(space, D, k, B, max_particles, w, idx_out, local_out, s);
    if (k <= 8) return launch_knn_t<8>(space, D, k, B, max_particles, w, idx_out, local_out, s);
    if (k <= 16) return launch_knn_t<16>(space, D, k, B, max_particles, w, idx_out, local_out, s);
    return launch_knn_t<32>(space, D, k, B, max_particles, w, idx_out, local_out, s);
}

// debug entry: jet-local neighbour indices -> the global ones the EdgeConv kernels read (out-of-jet values -> -1), and the
// particle -> jet map the pooling epilogue reads (the forward gets both from the kNN kernels)
__global__ void globalize_idx_kernel(const int32_t* __restrict__ idx_local, int k, const int32_t* __restrict__ jet_start,
                                     const int32_t* __restrict__ jet_n, const int32_t* __restrict__ meta,
                                     int32_t* __restrict__ idx_global, int32_t* __restrict__ pjid) {
    if (meta[0]) return;
    const int b = blockIdx.x;
    int n = jet_n[b];
    const int start = jet_start[b];
    const int rows = n < -1 ? -n : n;
    for (int e = threadIdx.x; e < rows * k; e += blockDim.x) {
        int j = idx_local[(size_t)start * k + e];
        idx_global[(size_t)start * k + e] = (n > 0 && j >= 0 && j < n) ? j + start : -1;
    }
    for (int r = threadIdx.x; r < rows; r += blockDim.x) pjid[start + r] = b;
}

int launch_globalize_idx(const int32_t* idx_local, int k, int B, const Workspace& w, int32_t* idx_global, cudaStream_t s) {
    if (B == 0) return 0;
    globalize_idx_kernel<<<B, 128, 0, s>>>(idx_local, k, w.jet_start, w.jet_n, w.meta, idx_global, w.pjid);
    return 1;
}

int knn_configure() {
    return cudaFuncSetAttribute(knn_dist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024) == cudaSuccess
               ? GNN_OK : GNN_ERR_CUDA;
}

// ---- gnn_knn_noalloc: the exact kNN above for callers that may not allocate device memory ----------------------------------
// Who this is for: code that runs where a cudaMalloc is forbidden or fails by construction -- a plugin inside a host
// application that hands the plugin fixed buffers and owns the device heap itself, a latency-critical loop that has promised
// its scheduler never to take the allocator's device-wide lock, a process whose memory budget was carved up before this
// library was loaded.  Such a caller cannot even call gnn_create (which allocates weights and a workspace), so this entry
// takes no gnn_model.  Everything the two kernels need besides the caller's input and output -- the sanitised ragged
// descriptors, the particle -> jet map and the per-jet distance matrix -- lives in ONE array that is part of the library's
// image: the driver sets it aside on every GPU that loads libgnn.so and keeps it until the process exits (about 4.1 MiB).
//
// `knn_noalloc_scratch` below is that array.  In host code its name is only a handle the runtime knows the array by, NOT a
// device address (a kernel given `knn_noalloc_scratch` from the host would fault, or scribble on host memory on systems where
// the GPU can reach it).  The address a kernel may use comes from cudaGetSymbolAddress, asked for once per device with that
// device current, in knn_noalloc_base().
constexpr int NOALLOC_MAX_JETS = 1024;          // largest B of one call
constexpr int NOALLOC_MAX_ROWS = 8192;          // largest N of one call (particles of the whole batch)
constexpr int NOALLOC_MAX_DEVICES = 64;
// layout (byte offsets, every part 256-byte aligned):  [0, 256) status word + meta[4]  |  jet_start [MAX_JETS] int32  |
// jet_n [MAX_JETS] int32  |  pjet [MAX_ROWS] int2  |  dm [MAX_ROWS][GNN_MAX_PARTICLES] fp32
constexpr size_t NOALLOC_OFF_START = 256;
constexpr size_t NOALLOC_OFF_N = NOALLOC_OFF_START + sizeof(int32_t) * NOALLOC_MAX_JETS;
constexpr size_t NOALLOC_OFF_PJET = NOALLOC_OFF_N + sizeof(int32_t) * NOALLOC_MAX_JETS;
constexpr size_t NOALLOC_OFF_DM = NOALLOC_OFF_PJET + sizeof(int2) * NOALLOC_MAX_ROWS;
constexpr size_t NOALLOC_BYTES = NOALLOC_OFF_DM + sizeof(float) * NOALLOC_MAX_ROWS * GNN_MAX_PARTICLES;
static_assert(NOALLOC_OFF_N % 256 == 0 && NOALLOC_OFF_PJET % 256 == 0 && NOALLOC_OFF_DM % 256 == 0, "scratch parts stay 256-byte aligned");
static __device__ __align__(256) unsigned char knn_noalloc_scratch[NOALLOC_BYTES];

// device address of the scratch array on the CURRENT device (looked up on the first call per device, then remembered)
static int knn_noalloc_base(unsigned char** out) {
    static std::mutex mu;
    static unsigned char* base[NOALLOC_MAX_DEVICES] = {};
    int device = -1;
    GNN_CUDA_TRY(cudaGetDevice(&device));
    if (device < 0 || device >= NOALLOC_MAX_DEVICES) return GNN_ERR_BAD_ARG;
    std::lock_guard<std::mutex> lock(mu);
    if (base[device] == nullptr) {
        unsigned char* p = nullptr;
        GNN_CUDA_TRY(cudaGetSymbolAddress((void**)&p, knn_noalloc_scratch));
        if (p == nullptr) return GNN_ERR_CUDA;
        base[device] = p;
    }
    *out = base[device];
    return GNN_OK;
}

extern "C" int gnn_knn_noalloc(const float* space_dev, int32_t D, const int32_t* offsets_dev, int32_t B, int32_t N,
                               int32_t max_particles, int32_t k, int32_t* idx_dev, void* cuda_stream) {
    if (B < 0 || N < 0 || D < 1 || D > 1024 || k < 1 || k > GNN_MAX_K || max_particles < 1 || max_particles > GNN_MAX_PARTICLES)
        return GNN_ERR_BAD_ARG;
    if (B > NOALLOC_MAX_JETS || N > NOALLOC_MAX_ROWS) {
        std::fprintf(stderr, "libgnn: gnn_knn_noalloc: B = %d, N = %d exceed the built-in scratch (at most %d jets and %d particles "
                     "per call); split the batch or use gnn_debug_knn on a gnn_model\n", B, N, NOALLOC_MAX_JETS, NOALLOC_MAX_ROWS);
        return GNN_ERR_BATCH_TOO_LARGE;
    }
    if (B == 0) return GNN_OK;
    if (!offsets_dev || !idx_dev || (N > 0 && !space_dev)) return GNN_ERR_NULL;
    unsigned char* base = nullptr;
    int rc = knn_noalloc_base(&base);
    if (rc != GNN_OK) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    Workspace w;                                // a view of the static array: nothing here is allocated or freed
    w.status = reinterpret_cast<unsigned*>(base);
    w.meta = reinterpret_cast<int32_t*>(base + 16);
    w.jet_start = reinterpret_cast<int32_t*>(base + NOALLOC_OFF_START);
    w.jet_n = reinterpret_cast<int32_t*>(base + NOALLOC_OFF_N);
    w.pjet = reinterpret_cast<int2*>(base + NOALLOC_OFF_PJET);
    w.dm = reinterpret_cast<float*>(base + NOALLOC_OFF_DM);
    w.groups = nullptr;                         // no group schedule: the exact path does not use one
    // The array still holds whatever the previous call left.  Only the status word and meta[] are read before they are
    // written (the status word is OR-ed into), so those 256 bytes are cleared on the stream; the descriptors, the map and the
    // distances are written for every row of this batch before the selection reads them.
    GNN_CUDA_TRY(cudaMemsetAsync(base, 0, 256, s));
    if ((rc = launch_ingest(offsets_dev, nullptr, B, N, N, max_particles, w, s)) < 0) return rc;
    if ((rc = launch_knn(space_dev, D, k, B, max_particles, w, idx_dev, /*local_out=*/1, /*gram=*/0, s, DEP_NONE)) < 0) return rc;
    return cudaGetLastError() == cudaSuccess ? GNN_OK : GNN_ERR_CUDA;
}

// pool_head.cu -- steps a7/a8: masked global average pool over the particles of a jet and the FC head
// ("two fully connected layers with 256 nodes and 0.1 dropout rate to two nodes"; L270 inference mode
// => dropout is the identity; BASELINE.json north_star (3)).  fp32 in every precision mode (R19).
// Ragged input makes the "mask" implicit: only the n_b real particles of jet b are ever stored (R7, R12).
//
// One CTA per PH_JETS consecutive jets: (1) pooling, float4 loads, the CTA's threads split into row groups x channel
// quads and the group partials are reduced through shared memory in a fixed order (deterministic); (2) the FC layers as
// mat-vecs on the transposed weights Wt[in][out] with PH_JETS accumulators per thread, so a weight is read once per
// CTA instead of once per jet (the 256 KB of FC-1 weights were 268 MB of L2 traffic per forward at one jet per CTA).
#include "gnn_internal.h"

namespace {

// thread-block cluster helpers of head_split_kernel
__device__ __forceinline__ unsigned tc_cluster_rank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void tc_cluster_sync() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// generic address of `p` (a shared-memory object of this CTA) in CTA `rank` of the cluster
template <typename T>
__device__ __forceinline__ T* tc_map_shared_rank(T* p, unsigned rank) {
    unsigned long long out;
    asm volatile("mapa.u64 %0, %1, %2;" : "=l"(out) : "l"((unsigned long long)p), "r"(rank));
    return reinterpret_cast<T*>(out);
}

constexpr int PH_THREADS = 256;
constexpr int PH_JETS = 4;

struct HeadParams {
    LinF32 fc[GNN_MAX_FC + 1];
    int n_fc;
    int C;
    int n_classes;
    int wmax;        // widest activation vector (row stride of the staging arrays)
};

__global__ void __launch_bounds__(PH_THREADS)
pool_head_kernel(const float* __restrict__ x, const int32_t* __restrict__ jet_start, const int32_t* __restrict__ jet_n,
                 const int32_t* __restrict__ meta, HeadParams hp, int B, float* __restrict__ logits) {
    extern __shared__ __align__(16) float zs[];      // z0 [PH_JETS][wmax] | z1 [PH_JETS][wmax] | partials
    __shared__ int s_n[PH_JETS];                     // multiplicities (0 for offending / absent jets)
    const int b0 = blockIdx.x * PH_JETS;
    const int nj = min(PH_JETS, B - b0);
    const int C = hp.C, W = hp.wmax;
    float* z0 = zs;
    float* z1 = zs + PH_JETS * W;
    float* part = z1 + PH_JETS * W;                  // pooling: [G][PH_JETS][C]; FC: [KS][PH_JETS][ld]
    const bool poisoned = meta[0] != 0;
    // ---- pooling: the jets of this CTA are one contiguous span of rows; thread (row group rg, channel quad cq) walks rows
    // rg, rg + G, ... with eight loads in flight and flushes its partial sum when a row crosses into the next jet ---------
    if (threadIdx.x < PH_JETS) {
        const int jb = threadIdx.x;
        int n = (jb < nj && !poisoned) ? jet_n[b0 + jb] : 0;
        if (n < 0) n = 0;                            // offending jet: pools nothing (its logits become NaN below)
        s_n[jb] = n;
    }
    __syncthreads();
    const int CQ = C >> 2;                           // channel quads
    const int TQ = min(CQ, PH_THREADS);
    const int G = max(1, PH_THREADS / CQ);           // row groups
    // rows of jets are contiguous only for well-formed batches; offending jets own rows too, so walk jet by jet ranges
    for (int cq0 = 0; cq0 < CQ; cq0 += PH_THREADS) {
        const int cq = cq0 + (int)threadIdx.x % TQ, rg = (int)threadIdx.x / TQ;
        if (cq < CQ && rg < G) {
            for (int jb = 0; jb < PH_JETS; ++jb) {
                const int n = s_n[jb];
                const float4* xb = reinterpret_cast<const float4*>(x + (size_t)(jb < nj ? jet_start[b0 + jb] : 0) * C) + cq;
                float4 s = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                int i = rg;
                for (; i + 7 * G < n; i += 8 * G) {
                    float4 a[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u) a[u] = __ldg(xb + (size_t)(i + u * G) * CQ);
#pragma unroll
                    for (int u = 0; u < 8; ++u) { s.x += a[u].x; s.y += a[u].y; s.z += a[u].z; s.w += a[u].w; }
                }
                float4 a[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    a[u] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                    if (i + u * G < n) a[u] = __ldg(xb + (size_t)(i + u * G) * CQ);
                }
#pragma unroll
                for (int u = 0; u < 8; ++u) { s.x += a[u].x; s.y += a[u].y; s.z += a[u].z; s.w += a[u].w; }
                *reinterpret_cast<float4*>(part + ((size_t)rg * PH_JETS + jb) * C + 4 * cq) = s;
            }
        }
        __syncthreads();
        for (int it = threadIdx.x; it < PH_JETS * TQ; it += PH_THREADS) {
            const int jb = it / TQ, c4 = cq0 + it % TQ;
            if (c4 >= CQ) continue;
            float4 s = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            for (int g2 = 0; g2 < G; ++g2) {
                const float4 o = *reinterpret_cast<const float4*>(part + ((size_t)g2 * PH_JETS + jb) * C + 4 * c4);
                s.x += o.x; s.y += o.y; s.z += o.z; s.w += o.w;
            }
            const int n = s_n[jb];
            const float inv = n > 0 ? 1.0f / (float)n : 0.0f;           // R12: empty jet pools to 0
            *reinterpret_cast<float4*>(z0 + jb * W + 4 * c4) = make_float4(s.x * inv, s.y * inv, s.z * inv, s.w * inv);
        }
        __syncthreads();
    }
    // ---- FC head: wide layers split K over thread groups (float4 of outputs x K slice, eight weight loads in flight),
    // narrow layers (the final one) run one thread per (jet, output) ---------------------------------------------------------
    float* zin = z0; float* zout = z1;
    for (int l = 0; l < hp.n_fc; ++l) {
        const LinF32 L = hp.fc[l];
        const bool last = (l == hp.n_fc - 1);
        const int OQ = L.ld >> 2;
        if (OQ >= 16 && OQ <= PH_THREADS) {
            const int KS = PH_THREADS / OQ;                      // K slices
            const int oq = (int)threadIdx.x % OQ, ks = (int)threadIdx.x / OQ;
            if (ks < KS) {
                const int kper = (L.K + KS - 1) / KS, k0 = ks * kper, k1 = min(L.K, k0 + kper);
                float4 acc[PH_JETS];
#pragma unroll
                for (int jb = 0; jb < PH_JETS; ++jb) acc[jb] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                const float4* wp = reinterpret_cast<const float4*>(L.Wt) + oq;
                for (int c = k0; c < k1; c += 8) {
                    float4 wv[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        wv[u] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                        if (c + u < k1) wv[u] = __ldg(wp + (size_t)(c + u) * OQ);
                    }
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        if (c + u < k1) {
#pragma unroll
                            for (int jb = 0; jb < PH_JETS; ++jb) {
                                const float zv = zin[jb * W + c + u];
                                acc[jb].x = fmaf(zv, wv[u].x, acc[jb].x); acc[jb].y = fmaf(zv, wv[u].y, acc[jb].y);
                                acc[jb].z = fmaf(zv, wv[u].z, acc[jb].z); acc[jb].w = fmaf(zv, wv[u].w, acc[jb].w);
                            }
                        }
                    }
                }
#pragma unroll
                for (int jb = 0; jb < PH_JETS; ++jb)
                    *reinterpret_cast<float4*>(part + ((size_t)ks * PH_JETS + jb) * L.ld + 4 * oq) = acc[jb];
            }
            __syncthreads();
            for (int it = threadIdx.x; it < PH_JETS * L.N; it += PH_THREADS) {
                const int jb = it / L.N, o = it - jb * L.N;
                float v = __ldg(L.shift + o);
                for (int k2 = 0; k2 < KS; ++k2) v += part[((size_t)k2 * PH_JETS + jb) * L.ld + o];
                if (jb < nj) {
                    if (last) {
                        const bool bad = poisoned || jet_n[b0 + jb] < 0;
                        logits[(size_t)(b0 + jb) * hp.n_classes + o] = bad ? __int_as_float(0x7fc00000) : v;
                    } else {
                        zout[jb * W + o] = fmaxf(v, 0.0f);
                    }
                }
            }
        } else {
            // narrow layer (the final one): one WARP per (jet, output), lanes split K, fixed-order shuffle reduction
            const int wid = threadIdx.x >> 5, ln = threadIdx.x & 31;
            for (int it = wid; it < PH_JETS * L.N; it += PH_THREADS / 32) {
                const int jb = it / L.N, o = it - jb * L.N;
                float a0 = 0.0f;
                for (int c = ln; c < L.K; c += 32) a0 = fmaf(zin[jb * W + c], __ldg(L.Wt + (size_t)c * L.ld + o), a0);
#pragma unroll
                for (int sh = 16; sh > 0; sh >>= 1) a0 += __shfl_xor_sync(0xffffffffu, a0, sh);
                const float v = a0 + __ldg(L.shift + o);
                if (ln == 0 && jb < nj) {
                    if (last) {
                        const bool bad = poisoned || jet_n[b0 + jb] < 0;
                        logits[(size_t)(b0 + jb) * hp.n_classes + o] = bad ? __int_as_float(0x7fc00000) : v;
                    } else {
                        zout[jb * W + o] = fmaxf(v, 0.0f);
                    }
                }
            }
        }
        __syncthreads();
        float* t = zin; zin = zout; zout = t;
    }
}

// ---- GNN_BF16 with the pooling EdgeConv epilogue: the head alone, on the per-jet channel sums -----------------------------
// The sums arrive as exact 2^-32 fixed-point integers (edge_kernel<.., POOL>).  One CTA per HD_JETS jets; activations are kept
// TRANSPOSED in shared memory (zT[k][jet]) so that one 16-byte load feeds four jets; a thread owns four outputs x HD_JETS
// jets of one K slice of a wide layer (weights Wt[in][out] read once per CTA, eight 16-byte loads in flight), slices are
// summed through shared memory in a fixed order; the narrow final layer runs one warp per (jet, output).
// sum (unsigned 32.32 fixed point) / n in fp32: integer and fraction parts convert separately (no 64-bit or fp64 conversions,
// which are slow); the result is within 1.5 ulp of the exact mean and depends on nothing but (sum, n)
__device__ __forceinline__ float fixed_value(unsigned long long v) {
    return fmaf((float)(unsigned)(v & 0xffffffffull), 1.0f / 4294967296.0f, (float)(unsigned)(v >> 32));
}
__device__ __forceinline__ float fixed_mean(unsigned long long v, int n) { return fixed_value(v) / (float)n; }

constexpr int HD_THREADS = 256;
constexpr int HD_JETS = 8;

__global__ void __launch_bounds__(HD_THREADS)
head_kernel(const unsigned long long* __restrict__ pooled, const int32_t* __restrict__ jet_n, const int32_t* __restrict__ meta,
            HeadParams hp, int B, float* __restrict__ logits) {
    extern __shared__ __align__(16) float hs[];      // zT0 [wmax][HD_JETS] | zT1 [wmax][HD_JETS] | partials [KS][HD_JETS][ld]
    __shared__ int s_n[HD_JETS];
    const int b0 = blockIdx.x * HD_JETS;
    const int nj = min(HD_JETS, B - b0);
    const int C = hp.C, W = hp.wmax;
    float* z0 = hs;
    float* z1 = hs + W * HD_JETS;
    float* part = z1 + W * HD_JETS;
    const bool poisoned = meta[0] != 0;
    if (threadIdx.x < HD_JETS) {
        const int jb = threadIdx.x;
        int n = (jb < nj && !poisoned) ? jet_n[b0 + jb] : 0;
        s_n[jb] = n < 0 ? 0 : n;                     // offending jet: pools nothing (its logits become NaN below)
    }
    __syncthreads();
    for (int it = threadIdx.x; it < HD_JETS * C; it += HD_THREADS) {
        const int jb = it / C, c = it - jb * C;
        const int n = s_n[jb];
        float g = 0.0f;                              // R12: empty jet pools to 0
        if (n > 0) g = fixed_mean(__ldg(pooled + (size_t)(b0 + jb) * C + c), n);
        z0[c * HD_JETS + jb] = g;
    }
    __syncthreads();
    float* zin = z0; float* zout = z1;
    for (int l = 0; l < hp.n_fc; ++l) {
        const LinF32 L = hp.fc[l];
        const bool last = (l == hp.n_fc - 1);
        const int OQ = L.ld >> 2;
        if (OQ >= 16 && OQ <= HD_THREADS) {
            const int KS = HD_THREADS / OQ;                      // K slices
            const int oq = (int)threadIdx.x % OQ, ks = (int)threadIdx.x / OQ;
            if (ks < KS) {
                const int kper = (L.K + KS - 1) / KS, k0 = ks * kper, k1 = min(L.K, k0 + kper);
                float4 acc[HD_JETS];
#pragma unroll
                for (int jb = 0; jb < HD_JETS; ++jb) acc[jb] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                const float4* wp = reinterpret_cast<const float4*>(L.Wt) + oq;
                auto load8 = [&](float4 (&wv)[8], int c) {
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        wv[u] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                        if (c + u < k1) wv[u] = __ldg(wp + (size_t)(c + u) * OQ);
                    }
                };
                auto fma8 = [&](const float4 (&wv)[8], int c) {
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        if (c + u < k1) {
                            const float4 za = *reinterpret_cast<const float4*>(zin + (c + u) * HD_JETS);
                            const float4 zb = *reinterpret_cast<const float4*>(zin + (c + u) * HD_JETS + 4);
                            const float zv[HD_JETS] = {za.x, za.y, za.z, za.w, zb.x, zb.y, zb.z, zb.w};
#pragma unroll
                            for (int jb = 0; jb < HD_JETS; ++jb) {
                                acc[jb].x = fmaf(zv[jb], wv[u].x, acc[jb].x); acc[jb].y = fmaf(zv[jb], wv[u].y, acc[jb].y);
                                acc[jb].z = fmaf(zv[jb], wv[u].z, acc[jb].z); acc[jb].w = fmaf(zv[jb], wv[u].w, acc[jb].w);
                            }
                        }
                    }
                };
                // two batches of eight weight rows alternate: the loads of one are in flight while the other is multiplied
                float4 wa[8], wb[8];
                load8(wa, k0);
                for (int c = k0; c < k1; c += 16) {
                    load8(wb, c + 8);
                    fma8(wa, c);
                    load8(wa, c + 16);
                    fma8(wb, c + 8);
                }
#pragma unroll
                for (int jb = 0; jb < HD_JETS; ++jb)
                    *reinterpret_cast<float4*>(part + ((size_t)ks * HD_JETS + jb) * L.ld + 4 * oq) = acc[jb];
            }
            __syncthreads();
            for (int it = threadIdx.x; it < HD_JETS * L.N; it += HD_THREADS) {
                const int jb = it / L.N, o = it - jb * L.N;
                float v = __ldg(L.shift + o);
                for (int k2 = 0; k2 < KS; ++k2) v += part[((size_t)k2 * HD_JETS + jb) * L.ld + o];
                if (last) {
                    if (jb < nj) {
                        const bool bad = poisoned || jet_n[b0 + jb] < 0;
                        logits[(size_t)(b0 + jb) * hp.n_classes + o] = bad ? __int_as_float(0x7fc00000) : v;
                    }
                } else {
                    zout[o * HD_JETS + jb] = fmaxf(v, 0.0f);
                }
            }
        } else {
            // narrow layer (the final one): one WARP per (jet, output), lanes split K, fixed-order shuffle reduction
            const int wid = threadIdx.x >> 5, ln = threadIdx.x & 31;
            for (int it = wid; it < HD_JETS * L.N; it += HD_THREADS / 32) {
                const int jb = it / L.N, o = it - jb * L.N;
                float a0 = 0.0f;
                for (int c = ln; c < L.K; c += 32) a0 = fmaf(zin[c * HD_JETS + jb], __ldg(L.Wt + (size_t)c * L.ld + o), a0);
#pragma unroll
                for (int sh = 16; sh > 0; sh >>= 1) a0 += __shfl_xor_sync(0xffffffffu, a0, sh);
                const float v = a0 + __ldg(L.shift + o);
                if (ln == 0) {
                    if (last) {
                        if (jb < nj) {
                            const bool bad = poisoned || jet_n[b0 + jb] < 0;
                            logits[(size_t)(b0 + jb) * hp.n_classes + o] = bad ? __int_as_float(0x7fc00000) : v;
                        }
                    } else {
                        zout[o * HD_JETS + jb] = fmaxf(v, 0.0f);
                    }
                }
            }
        }
        __syncthreads();
        float* t = zin; zin = zout; zout = t;
    }
}


// ---- the head with ONE hidden layer (every BASELINE config), outputs of the hidden layer split over a CLUSTER of CTAs -------
// head_kernel above gives one CTA all of FC-1 for its jets: at B = 1024 that is 128 CTAs of 8 warps, one per SM, each walking
// a 256 KB weight matrix through dependent batches of loads (ncu: 12 % warps active, 24 us).  Here a CTA owns HS_JETS jets x
// HS_OUT hidden units and the H / HS_OUT CTAs of a jet group form a thread-block cluster: grid (jet groups, H / HS_OUT), one
// wave at B = 1024.  Thread (oq, ks) holds 4 hidden units of K slice ks (C / 16 rows of Wt, all its loads in flight at once:
// one round trip, kept in registers for both passes of 8 jets), slices are summed through shared memory in a fixed order,
// bias + ReLU, then this CTA's share of the final layer (HS_OUT terms per logit, one warp per (jet, class), fixed shuffle
// tree).  The shares go to the cluster's first CTA through distributed shared memory and are added there in rank order, so a
// logit depends neither on CTA timing nor on the batch mates: batch-composition invariance stays bitwise.
constexpr int HS_THREADS = 256;
constexpr int HS_PASS = 8;                            // jets per pass (accumulators in registers)
constexpr int HS_PASSES = 2;
constexpr int HS_JETS = HS_PASS * HS_PASSES;
constexpr int HS_OUT = 64;
constexpr int HS_KS = HS_THREADS / (HS_OUT / 4);     // 16 K slices
constexpr int HS_MAX_SPLIT = 8;                       // portable cluster size
constexpr int HS_MAX_CLASSES = 4;

template <int KPER>                                   // rows of Wt per K slice = C / HS_KS
__global__ void __launch_bounds__(HS_THREADS)
head_split_kernel(const unsigned long long* pooled, const int32_t* __restrict__ jet_n, const int32_t* __restrict__ meta,
                  LinF32 L1, LinF32 L2, int B, int n_classes, float* __restrict__ logits) {
    constexpr int C = KPER * HS_KS;
    unsigned long long* pooled_rw = const_cast<unsigned long long*>(pooled);
    __shared__ __align__(16) float zT[C * HS_PASS];                  // pooled means of one pass, [channel][jet]
    __shared__ __align__(16) float part[HS_KS * HS_PASS * HS_OUT];   // [ks][jet][out]
    __shared__ float hT[HS_JETS * HS_OUT];                           // hidden activations of this CTA, [jet][out]
    __shared__ float s_inv[HS_JETS];                                 // 1 / n (0 for empty, offending or absent jets)
    __shared__ float cl_share[HS_MAX_SPLIT * HS_JETS * HS_MAX_CLASSES];   // rank 0: [rank][jet][class]
    const unsigned rank = tc_cluster_rank(), n_rank = gridDim.y;
    // Distributed shared memory may only be touched once every CTA of the cluster has started.  Arrive now, wait just before
    // the remote stores below: by then the other CTAs have long arrived, so the wait costs nothing.
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    const int b0 = blockIdx.x * HS_JETS, o0 = blockIdx.y * HS_OUT;
    const int nj = min(HS_JETS, B - b0);
    const int tid = threadIdx.x, oq = tid % (HS_OUT / 4), ks = tid / (HS_OUT / 4);
    const int wid = tid >> 5, ln = tid & 31;
    // this thread's weights first: they depend on nothing
    float4 wv[KPER];
    const float4* wp = reinterpret_cast<const float4*>(L1.Wt + (size_t)(ks * KPER) * L1.ld + o0) + oq;
#pragma unroll
    for (int u = 0; u < KPER; ++u) wv[u] = __ldg(wp + (size_t)u * (L1.ld >> 2));
    // the jets' channel sums of a pass: every load of a thread in flight before the first conversion (one round trip)
    constexpr int CPT = (C + HS_THREADS - 1) / HS_THREADS;
    unsigned long long pv[CPT][HS_PASS];
    auto load_pooled = [&](int pass) {
#pragma unroll
        for (int i = 0; i < CPT; ++i)
#pragma unroll
            for (int jb = 0; jb < HS_PASS; ++jb) {
                const int c = tid + i * HS_THREADS, j = pass * HS_PASS + jb;
                pv[i][jb] = (c < C && j < nj) ? __ldcg(pooled + (size_t)(b0 + j) * C + c) : 0ull;
            }
    };
    // this warp's weights of the final layer (warp = (jet, class) items, lanes = hidden units ln and 32 + ln)
    float w2a[HS_MAX_CLASSES], w2b[HS_MAX_CLASSES];
#pragma unroll
    for (int o = 0; o < HS_MAX_CLASSES; ++o) {
        w2a[o] = o < n_classes ? __ldg(L2.Wt + (size_t)(o0 + ln) * L2.ld + o) : 0.0f;
        w2b[o] = o < n_classes ? __ldg(L2.Wt + (size_t)(o0 + 32 + ln) * L2.ld + o) : 0.0f;
    }
    const float shift1 = __ldg(L1.shift + o0 + (tid % HS_OUT));
    grid_dep_wait();                                 // the weight loads above run under the tail of the last EdgeConv kernel
    load_pooled(0);
    const bool poisoned = meta[0] != 0;
    if (tid < HS_JETS) {
        int n = (tid < nj && !poisoned) ? jet_n[b0 + tid] : 0;
        s_inv[tid] = n > 0 ? 1.0f / (float)n : 0.0f;   // offending jet: pools nothing (its logits become NaN below); R12: empty jet pools to 0
    }
    __syncthreads();
#pragma unroll 1
    for (int pass = 0; pass < HS_PASSES; ++pass) {
#pragma unroll
        for (int i = 0; i < CPT; ++i) {
            const int c = tid + i * HS_THREADS;
            if (c < C) {
                float z[HS_PASS];
#pragma unroll
                for (int jb = 0; jb < HS_PASS; ++jb) z[jb] = fixed_value(pv[i][jb]) * s_inv[pass * HS_PASS + jb];
                *reinterpret_cast<float4*>(zT + c * HS_PASS) = make_float4(z[0], z[1], z[2], z[3]);
                *reinterpret_cast<float4*>(zT + c * HS_PASS + 4) = make_float4(z[4], z[5], z[6], z[7]);
            }
        }
        if (pass + 1 < HS_PASSES) load_pooled(pass + 1);          // in flight during this pass's products
        __syncthreads();
        float4 acc[HS_PASS];
#pragma unroll
        for (int jb = 0; jb < HS_PASS; ++jb) acc[jb] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
#pragma unroll
        for (int u = 0; u < KPER; ++u) {
            const float4 za = *reinterpret_cast<const float4*>(zT + (ks * KPER + u) * HS_PASS);
            const float4 zb = *reinterpret_cast<const float4*>(zT + (ks * KPER + u) * HS_PASS + 4);
            const float zv[HS_PASS] = {za.x, za.y, za.z, za.w, zb.x, zb.y, zb.z, zb.w};
#pragma unroll
            for (int jb = 0; jb < HS_PASS; ++jb) {
                acc[jb].x = fmaf(zv[jb], wv[u].x, acc[jb].x); acc[jb].y = fmaf(zv[jb], wv[u].y, acc[jb].y);
                acc[jb].z = fmaf(zv[jb], wv[u].z, acc[jb].z); acc[jb].w = fmaf(zv[jb], wv[u].w, acc[jb].w);
            }
        }
#pragma unroll
        for (int jb = 0; jb < HS_PASS; ++jb)
            *reinterpret_cast<float4*>(part + (ks * HS_PASS + jb) * HS_OUT + 4 * oq) = acc[jb];
        __syncthreads();
        for (int it = tid; it < HS_PASS * HS_OUT; it += HS_THREADS) {      // it = jb * HS_OUT + o, o = tid % HS_OUT
            float v = shift1;
#pragma unroll
            for (int k2 = 0; k2 < HS_KS; ++k2) v += part[k2 * HS_PASS * HS_OUT + it];
            hT[pass * HS_PASS * HS_OUT + it] = fmaxf(v, 0.0f);
        }
        __syncthreads();                                            // zT and part are rewritten by the next pass
    }
    // final layer, this CTA's HS_OUT terms: one warp per jet (all classes), then into the first CTA's shared memory
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");   // pairs with the arrive at kernel entry: rank 0 exists
    float* dst = tc_map_shared_rank(cl_share, 0) + rank * (HS_JETS * HS_MAX_CLASSES);
    for (int jb = wid; jb < HS_JETS; jb += HS_THREADS / 32) {
        const float ha = hT[jb * HS_OUT + ln], hb = hT[jb * HS_OUT + 32 + ln];
#pragma unroll
        for (int o = 0; o < HS_MAX_CLASSES; ++o) {
            float a0 = fmaf(hb, w2b[o], ha * w2a[o]);
#pragma unroll
            for (int sh = 16; sh > 0; sh >>= 1) a0 += __shfl_xor_sync(0xffffffffu, a0, sh);
            if (ln == 0) dst[jb * HS_MAX_CLASSES + o] = a0;
        }
    }
    tc_cluster_sync();                                              // release / acquire: the shares are visible to rank 0
    if (rank != 0) return;
    // every CTA of the cluster has read the jets' channel sums: clear them for the next forward (Workspace::pool_self_cleaning)
    for (int it = tid; it < nj * C; it += HS_THREADS) pooled_rw[(size_t)b0 * C + it] = 0ull;
    for (int it = tid; it < nj * n_classes; it += HS_THREADS) {
        const int jb = it / n_classes, o = it - jb * n_classes;
        float v = __ldg(L2.shift + o);
        for (unsigned y = 0; y < n_rank; ++y) v += cl_share[(y * HS_JETS + jb) * HS_MAX_CLASSES + o];
        const bool bad = poisoned || jet_n[b0 + jb] < 0;
        logits[(size_t)(b0 + jb) * n_classes + o] = bad ? __int_as_float(0x7fc00000) : v;
    }
}

template <int KPER>
int launch_head_split(const HeadParams& hp, int B, const Workspace& w, float* logits, cudaStream_t s, bool pdl) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((B + HS_JETS - 1) / HS_JETS, hp.fc[0].N / HS_OUT);
    cfg.blockDim = dim3(HS_THREADS);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = s;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 1; at[0].val.clusterDim.y = cfg.gridDim.y; at[0].val.clusterDim.z = 1;
    at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = (pdl && gnn_pdl_enabled()) ? 2 : 1;
    GNN_CUDA_TRY(cudaLaunchKernelEx(&cfg, head_split_kernel<KPER>, (const unsigned long long*)w.pool, (const int32_t*)w.jet_n,
                                    (const int32_t*)w.meta, hp.fc[0], hp.fc[1], B, hp.n_classes, logits));
    return 1;
}

}  // namespace

// x != null: pool the stored block output [N, C]; x == null: the channel sums are in w.pool (pooling EdgeConv epilogue)
// whether launch_pool_head(x == null) takes head_split_kernel, which clears the channel sums after reading them
bool head_clears_pool(const gnn_model& m) {
    const int C = m.arch.channels[m.arch.n_blocks - 1][2];
    return m.n_fc == 2 && m.fc[0].N % HS_OUT == 0 && m.fc[0].N / HS_OUT <= HS_MAX_SPLIT && m.arch.n_classes <= HS_MAX_CLASSES &&
           (C == 256 || C == 128 || C == 64);          // (C = 512: beyond 48 KB of static shared memory)
}

int launch_pool_head(const gnn_model& m, const float* x, int B, const Workspace& w, float* logits, cudaStream_t s, bool pdl) {
    if (B == 0) return 0;
    HeadParams hp;
    hp.n_fc = m.n_fc;
    for (int i = 0; i < m.n_fc; ++i) hp.fc[i] = m.fc[i];
    hp.C = m.arch.channels[m.arch.n_blocks - 1][2];
    hp.n_classes = m.arch.n_classes;
    hp.wmax = hp.C;
    for (int i = 0; i < m.n_fc; ++i) hp.wmax = std::max(hp.wmax, (m.fc[i].N + 3) & ~3);
    if (x == nullptr && head_clears_pool(m)) {
        switch (hp.C) {
            case 64: return launch_head_split<64 / HS_KS>(hp, B, w, logits, s, pdl);
            case 128: return launch_head_split<128 / HS_KS>(hp, B, w, logits, s, pdl);
            default: return launch_head_split<256 / HS_KS>(hp, B, w, logits, s, pdl);
        }
    }
    if (x == nullptr) {
        size_t part = 4;
        for (int i = 0; i < m.n_fc; ++i) {
            const int OQ = m.fc[i].ld / 4;
            if (OQ >= 16 && OQ <= HD_THREADS) part = std::max(part, (size_t)(HD_THREADS / OQ) * HD_JETS * m.fc[i].ld);
        }
        const size_t smem = ((size_t)2 * HD_JETS * hp.wmax + part) * sizeof(float);
        head_kernel<<<(B + HD_JETS - 1) / HD_JETS, HD_THREADS, smem, s>>>(w.pool, w.jet_n, w.meta, hp, B, logits);
        return 1;
    }
    const int G = std::max(1, PH_THREADS / (hp.C / 4));
    size_t part = (size_t)G * PH_JETS * hp.C;                    // pooling partials, reused as the split-K partials
    for (int i = 0; i < m.n_fc; ++i) {
        const int OQ = m.fc[i].ld / 4;
        if (OQ >= 16 && OQ <= PH_THREADS) part = std::max(part, (size_t)(PH_THREADS / OQ) * PH_JETS * m.fc[i].ld);
    }
    const size_t smem = ((size_t)2 * PH_JETS * hp.wmax + part) * sizeof(float);
    pool_head_kernel<<<(B + PH_JETS - 1) / PH_JETS, PH_THREADS, smem, s>>>(x, w.jet_start, w.jet_n, w.meta, hp, B, logits);
    return 1;
}

// debug entry of the pooling EdgeConv epilogue: fixed-point channel sums -> g [B, C] = mean over the jet's particles
__global__ void pooled_mean_kernel(const unsigned long long* __restrict__ pooled, const int32_t* __restrict__ jet_n,
                                   const int32_t* __restrict__ meta, int B, int C, float* __restrict__ g) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= B * C) return;
    const int n = meta[0] ? 0 : jet_n[e / C];
    g[e] = n > 0 ? fixed_mean(pooled[e], n) : 0.0f;
}

int launch_pooled_mean(const gnn_model& m, int B, const Workspace& w, float* g, cudaStream_t s) {
    if (B == 0) return 0;
    const int C = m.arch.channels[m.arch.n_blocks - 1][2];
    pooled_mean_kernel<<<(B * C + 255) / 256, 256, 0, s>>>(w.pool, w.jet_n, w.meta, B, C, g);
    return 1;
}

int pool_head_configure() {
    return cudaFuncSetAttribute(pool_head_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024) == cudaSuccess &&
                   cudaFuncSetAttribute(head_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024) == cudaSuccess
               ? GNN_OK : GNN_ERR_CUDA;
}

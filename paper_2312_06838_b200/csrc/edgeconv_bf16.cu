// edgeconv_bf16.cu -- steps a2/a4/a6 in GNN_BF16 mode: the fused EdgeConv block on the 5th-generation tensor cores
// (PAPER.md L262 three EdgeConv blocks; BASELINE.json north_star (2): gather neighbours, edge feature [x_i, x_j - x_i],
// 3-layer shared MLP with BN folded in and ReLU as bf16 tcgen05/TMEM tile GEMMs, mean over k, 1x1 shortcut, with the
// [N*k, C] edge tensor never touching HBM).
//
// Factorisation: layer 1 is linear in e_ij = [x_i ; x_j - x_i], so
//     s1 * (W1 e_ij) + t1 = u_i + v_j,   u_i = s1*(W1a - W1b) x_i + t1,   v_j = s1*W1b x_j
// needs two per-PARTICLE products instead of one per edge.  Two kernels per block:
//   pre_kernel   per particle: u_i, v_i (stored bf16) and the shortcut r_i = ss*(Ws x_i) + ts (fp32), fp32 FMA.
//   edge_kernel  per tile of 128 edge rows (128/k particles x k neighbours), all on chip:
//     build   H1[r] = bf16(relu(u_i + v_j))  written straight into the 128B-swizzled K-major operand tile in smem
//     MMA     D  = H1 * W2'^T   (tcgen05.mma kind::f16, M = 128, N = C, bf16 x bf16 -> fp32 in TMEM; W2' = s2*W2)
//     E2      H2 = bf16(relu(D + t2))  TMEM -> registers -> the same operand tile (H1 is dead by then)
//     MMA     D  = H2 * W3'^T
//     E3      relu(D + t3), mean over the k_eff valid neighbour rows of each particle by a halving butterfly of
//             warp shuffles (rows = TMEM lanes = threads), + r_i, ReLU, coalesced fp32 store.
// Weights reach shared memory as pre-swizzled [rows][64] chunk images by 1-D bulk (TMA) copies into a ring of
// slots guarded by full/empty mbarriers; when both layers fit (C <= 128) every chunk is loaded once per CTA and stays
// resident, otherwise (C = 256) the ring streams them per tile from L2.
// Warp roles: warps 0-7 build / epilogue (two warpgroups = two column halves of the TMEM lanes quadrants), warp 8
// allocates TMEM and its lane 0 issues every tcgen05.mma, warp 9 lane 0 is the weight-chunk producer.
#include "gnn_internal.h"
#include "tc05.cuh"
#include <cuda_bf16.h>
#include <cstring>

namespace {

using namespace tc05;

constexpr int EDGE_ALU_THREADS = 256;
constexpr int EDGE_THREADS = 320;
constexpr int TILE_ROWS = 128;

template <int C>
struct EdgeCfg {
    static constexpr int NR = C > 256 ? 256 : C;              // weight rows (= MMA N) per chunk
    static constexpr int NH = C / NR;                         // N halves per layer
    static constexpr int KB = (C + 63) / 64;                  // 64-wide K blocks per layer
    static constexpr int KSTEPS_LAST = ((C - (KB - 1) * 64) + 15) / 16;
    static constexpr int CHUNK_BYTES = NR * 128;              // [NR][64] bf16, 128B-swizzled
    static constexpr int NCHUNK = 2 * NH * KB;                // both layers
    static constexpr bool RESIDENT = (size_t)NCHUNK * CHUNK_BYTES <= 96 * 1024;
    static constexpr int NSLOT = RESIDENT ? NCHUNK : (CHUNK_BYTES <= 32 * 1024 ? 4 : 2);
    static constexpr int H_BYTES = KB * TILE_ROWS * 128;      // KB K-blocks of [128][64] bf16
    static constexpr int TMEM_COLS = C < 32 ? 32 : C;
    static constexpr int RING_BYTES = NSLOT * CHUNK_BYTES;
    // dynamic shared memory: [ring][H][t2,t3 fp32][idx int32 x128][barriers][tmem ptr] (+1024 alignment slack)
    static constexpr int SMALL_BYTES = 2 * C * 4 + TILE_ROWS * 4 + (2 * NSLOT + 2) * 8 + 16;
    static constexpr int SMEM_BYTES = RING_BYTES + H_BYTES + SMALL_BYTES + 1024;
};

struct EdgeParams {
    const __nv_bfloat16* U;      // [N, C]
    const __nv_bfloat16* V;      // [N, C]
    const float* R;              // [N, C] shortcut
    const int32_t* idx;          // [N, k] global neighbour rows, -1 = none
    float* y;                    // [N, C]
    const int32_t* meta;         // meta[0] poisoned batch, meta[1] = N
    const uint8_t* wimg;         // NCHUNK chunk images in consumption order
    const float* shifts;         // [t2 | t3]
    int k, logk, TP, n_tiles;
};

template <int C>
__global__ void __launch_bounds__(EDGE_THREADS, (C <= 128 ? 2 : 1)) edge_kernel(EdgeParams p) {
    using Cfg = EdgeCfg<C>;
    extern __shared__ uint8_t smem_raw[];
    if (p.meta[0]) return;
    const int N = p.meta[1];
    const int n_tiles = min(p.n_tiles, (N + p.TP - 1) / p.TP);
    if ((int)blockIdx.x >= n_tiles) return;
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint8_t* ring = smem;
    uint8_t* H = ring + Cfg::RING_BYTES;
    float* shifts_s = reinterpret_cast<float*>(H + Cfg::H_BYTES);
    int32_t* idx_s = reinterpret_cast<int32_t*>(shifts_s + 2 * C);
    uint64_t* bars = reinterpret_cast<uint64_t*>(idx_s + TILE_ROWS);
    uint64_t* full = bars;                        // [NSLOT] weight chunk landed
    uint64_t* empty = bars + Cfg::NSLOT;          // [NSLOT] weight chunk consumed (streaming only)
    uint64_t* h_ready = bars + 2 * Cfg::NSLOT;    // operand tile written by the 256 ALU threads
    uint64_t* d_full = h_ready + 1;               // accumulator complete
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(d_full + 1);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int i = 0; i < Cfg::NSLOT; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
        mbar_init(h_ready, EDGE_ALU_THREADS);
        mbar_init(d_full, 1);
        fence_mbar_init();
    }
    for (int i = tid; i < 2 * C; i += EDGE_THREADS) shifts_s[i] = p.shifts[i];
    if (warp == 8) tmem_alloc(tmem_ptr, Cfg::TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_ptr;
    const int my_tiles = (n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;

    if (warp == 9) {
        // ===== weight-chunk producer ======================================================================
        if (lane == 0) {
            const int total = Cfg::RESIDENT ? Cfg::NCHUNK : Cfg::NCHUNK * my_tiles;
            for (int n = 0; n < total; ++n) {
                const int slot = n % Cfg::NSLOT;
                if (n >= Cfg::NSLOT) mbar_wait(&empty[slot], ((n / Cfg::NSLOT) - 1) & 1);
                mbar_arrive_expect_tx(&full[slot], Cfg::CHUNK_BYTES);
                bulk_g2s(ring + (size_t)slot * Cfg::CHUNK_BYTES, p.wimg + (size_t)(n % Cfg::NCHUNK) * Cfg::CHUNK_BYTES,
                         Cfg::CHUNK_BYTES, &full[slot]);
            }
        }
    } else if (warp == 8) {
        // ===== MMA issuer =================================================================================
        if (lane == 0) {
            constexpr uint32_t idesc = idesc_bf16_f32(128, Cfg::NR);
            const uint32_t h_addr = smem_u32(H), ring_addr = smem_u32(ring);
            uint32_t ph_h = 0;
            int n = 0;                                           // chunks consumed so far
            for (int t = 0; t < my_tiles; ++t) {
                for (int layer = 0; layer < 2; ++layer) {
                    mbar_wait(h_ready, ph_h); ph_h ^= 1;
                    tc_fence_after();
                    for (int nh = 0; nh < Cfg::NH; ++nh) {
                        for (int kb = 0; kb < Cfg::KB; ++kb, ++n) {
                            const int slot = Cfg::RESIDENT ? (n % Cfg::NCHUNK) : (n % Cfg::NSLOT);
                            if (!Cfg::RESIDENT || t == 0) mbar_wait(&full[slot], Cfg::RESIDENT ? 0 : ((n / Cfg::NSLOT) & 1));
                            tc_fence_after();
                            const int ksteps = (kb == Cfg::KB - 1) ? Cfg::KSTEPS_LAST : 4;
                            for (int ks = 0; ks < ksteps; ++ks) {
                                const uint64_t ad = desc_sw128(h_addr + kb * (TILE_ROWS * 128) + ks * 32);
                                const uint64_t bd = desc_sw128(ring_addr + slot * Cfg::CHUNK_BYTES + ks * 32);
                                mma_bf16_ss(tmem + nh * 256, ad, bd, idesc, (kb | ks) != 0);
                            }
                            if (!Cfg::RESIDENT) mma_commit(&empty[slot]);
                        }
                    }
                    mma_commit(d_full);
                }
            }
        }
    } else {
        // ===== build / epilogue warps ======================================================================
        const int q = warp & 3, half = warp >> 2;
        const int row = 32 * q + lane;                           // TMEM lane = edge row of the tile
        const int k = p.k, logk = p.logk;
        constexpr int CH = C / 8;                                // 16-byte chunks per operand row
        constexpr int ITEMS = TILE_ROWS * CH / EDGE_ALU_THREADS; // (row, chunk) items per thread
        constexpr int SLABS = (C >= 64) ? C / 64 : 1;            // 32-column slabs per warp (C = 32: warps 4-7 idle)
        const bool epi_active = (C >= 64) || half == 0;
        uint32_t ph_d = 0;
        for (int t = 0; t < my_tiles; ++t) {
            const int tile = blockIdx.x + t * gridDim.x;
            const int p0 = tile * p.TP;
            asm volatile("bar.sync 1, 256;" ::: "memory");       // previous tile's readers of idx_s are done
            if (tid < TILE_ROWS) {
                const int pt = p0 + (tid >> logk);
                idx_s[tid] = (pt < N) ? p.idx[(size_t)pt * k + (tid & (k - 1))] : -1;
            }
            asm volatile("bar.sync 1, 256;" ::: "memory");
            // ---- build H1 = bf16(relu(u_i + v_j)) ------------------------------------------------------
#pragma unroll
            for (int i0 = 0; i0 < ITEMS; i0 += 8) {
                uint4 vv[8], uu[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    if (i0 + i < ITEMS) {
                        const int it = tid + (i0 + i) * EDGE_ALU_THREADS;
                        const int r = it / CH, ch = it % CH;
                        const int j = idx_s[r];
                        if (j >= 0) {
                            vv[i] = __ldg(reinterpret_cast<const uint4*>(p.V + (size_t)j * C) + ch);
                            uu[i] = __ldg(reinterpret_cast<const uint4*>(p.U + (size_t)(p0 + (r >> logk)) * C) + ch);
                        } else {
                            vv[i] = make_uint4(0, 0, 0, 0); uu[i] = make_uint4(0, 0, 0, 0);
                        }
                    }
                }
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    if (i0 + i < ITEMS) {
                        const int it = tid + (i0 + i) * EDGE_ALU_THREADS;
                        const int r = it / CH, ch = it % CH;
                        uint4 h;
                        h.x = add_relu_bf16x2(vv[i].x, uu[i].x); h.y = add_relu_bf16x2(vv[i].y, uu[i].y);
                        h.z = add_relu_bf16x2(vv[i].z, uu[i].z); h.w = add_relu_bf16x2(vv[i].w, uu[i].w);
                        *reinterpret_cast<uint4*>(H + (ch >> 3) * (TILE_ROWS * 128) + r * 128 + (((ch & 7) ^ (r & 7)) << 4)) = h;
                    }
                }
            }
            fence_proxy_async();
            mbar_arrive(h_ready);
            // ---- E2: H2 = bf16(relu(D + t2)) -----------------------------------------------------------
            mbar_wait(d_full, ph_d); ph_d ^= 1;
            tc_fence_after();
            if (epi_active) {
#pragma unroll 1
                for (int s = 0; s < SLABS; ++s) {
                    const int col = (C >= 64) ? half * (C / 2) + s * 32 : 0;
                    float v[32];
                    tmem_ld32(tmem + ((uint32_t)(32 * q) << 16) + (col >> 8) * 256 + (col & 255), v);
                    tmem_ld_wait();
                    uint32_t pk[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i)
                        pk[i] = pack_relu_bf16x2(v[2 * i] + shifts_s[col + 2 * i], v[2 * i + 1] + shifts_s[col + 2 * i + 1]);
                    uint8_t* dst = H + (col >> 6) * (TILE_ROWS * 128) + row * 128;
                    const int c8 = (col & 63) >> 3;
#pragma unroll
                    for (int c = 0; c < 4; ++c)
                        *reinterpret_cast<uint4*>(dst + (((c8 + c) ^ (row & 7)) << 4)) =
                            make_uint4(pk[4 * c], pk[4 * c + 1], pk[4 * c + 2], pk[4 * c + 3]);
                }
            }
            tc_fence_before();
            fence_proxy_async();
            mbar_arrive(h_ready);
            // ---- E3: mean over the valid neighbours of relu(D + t3), + shortcut, ReLU ----------------------
            mbar_wait(d_full, ph_d); ph_d ^= 1;
            tc_fence_after();
            if (epi_active) {
                const bool valid = idx_s[row] >= 0;
                const unsigned gmask = (k >= 32) ? 0xffffffffu : (((1u << k) - 1u) << (lane & ~(k - 1)));
                const int cnt = __popc(__ballot_sync(0xffffffffu, valid) & gmask);
                const float inv = cnt > 0 ? 1.0f / (float)cnt : 0.0f;
                const int pt = p0 + (row >> logk);
                int cb = 0;                                      // first of the 32 >> logk columns this lane ends up with
                for (int s = 0; s < logk; ++s) cb += ((lane >> s) & 1) * (16 >> s);
                const int nout = 32 >> logk;
                const float* t3 = shifts_s + C;
#pragma unroll 1
                for (int s = 0; s < SLABS; ++s) {
                    const int col = (C >= 64) ? half * (C / 2) + s * 32 : 0;
                    float v[32];
                    tmem_ld32(tmem + ((uint32_t)(32 * q) << 16) + (col >> 8) * 256 + (col & 255), v);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 32; ++i) v[i] = valid ? fmaxf(v[i] + t3[col + i], 0.0f) : 0.0f;
                    // halving butterfly: after step s a lane keeps 16 >> s partial sums over 2^(s+1) rows
#pragma unroll
                    for (int s2 = 0; s2 < 5; ++s2) {
                        if (s2 < logk) {
                            const bool up = (lane >> s2) & 1;
                            const int cntv = 16 >> s2;
#pragma unroll
                            for (int i = 0; i < 16; ++i) {
                                if (i < cntv) {
                                    const float keep = up ? v[i + cntv] : v[i];
                                    const float send = up ? v[i] : v[i + cntv];
                                    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 1 << s2);
                                }
                            }
                        }
                    }
                    if (pt < N) {
                        const size_t o = (size_t)pt * C + col + cb;
#pragma unroll
                        for (int i = 0; i < 32; ++i)
                            if (i < nout) p.y[o + i] = fmaxf(fmaf(v[i], inv, __ldg(p.R + o + i)), 0.0f);
                    }
                }
            }
            tc_fence_before();
        }
    }
    __syncthreads();
    if (warp == 8) tmem_dealloc(tmem, Cfg::TMEM_COLS);
}

// ---- pre kernel: per-particle u (bf16), v (bf16), shortcut r (fp32) in fp32 FMA ------------------------------------------
// One CTA per tile of PRE_ROWS particles; x rows staged in shared memory; a thread owns 8 rows x 4 output columns of
// [u | v | r] = x * Wpre^T + bpre, Wpre^T stored [Kp][NC] (K padded to a multiple of 4 with zero rows).
constexpr int PRE_THREADS = 256;
constexpr int PRE_ROWS = 64;

struct PreParams {
    const float* x;          // [N, cin]
    const float* Wt;         // [Kp][NC]
    const float* bias;       // [NC] = [t1 | 0 | ts]
    __nv_bfloat16* U;        // [N, C1]
    __nv_bfloat16* V;        // [N, C1]
    float* R;                // [N, C3]
    const int32_t* meta;
    int cin, Kp, C1, C3, NC;
};

__global__ void __launch_bounds__(PRE_THREADS) pre_kernel(PreParams p) {
    extern __shared__ __align__(16) float xs[];      // [PRE_ROWS][Kp + 4]
    if (p.meta[0]) return;
    const int N = p.meta[1];
    const int r0 = blockIdx.x * PRE_ROWS;
    if (r0 >= N) return;
    const int ld = p.Kp + 4;
    for (int e = threadIdx.x; e < PRE_ROWS * p.Kp; e += PRE_THREADS) {
        const int r = e / p.Kp, c = e - r * p.Kp;
        xs[r * ld + c] = (r0 + r < N && c < p.cin) ? p.x[(size_t)(r0 + r) * p.cin + c] : 0.0f;
    }
    __syncthreads();
    const int ncg = p.NC >> 2;
    const int items = (PRE_ROWS / 8) * ncg;
    for (int it = threadIdx.x; it < items; it += PRE_THREADS) {
        const int rg = it / ncg, cg = it - rg * ncg;
        float acc[8][4];
#pragma unroll
        for (int r = 0; r < 8; ++r) acc[r][0] = acc[r][1] = acc[r][2] = acc[r][3] = 0.0f;
        const float* a0 = xs + (rg * 8) * ld;
        const float* w0 = p.Wt + cg * 4;
        for (int kk = 0; kk < p.Kp; kk += 4) {
            float4 w[4];
#pragma unroll
            for (int qq = 0; qq < 4; ++qq) w[qq] = __ldg(reinterpret_cast<const float4*>(w0 + (size_t)(kk + qq) * p.NC));
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const float4 a = *reinterpret_cast<const float4*>(a0 + r * ld + kk);
                acc[r][0] = fmaf(a.x, w[0].x, acc[r][0]); acc[r][1] = fmaf(a.x, w[0].y, acc[r][1]);
                acc[r][2] = fmaf(a.x, w[0].z, acc[r][2]); acc[r][3] = fmaf(a.x, w[0].w, acc[r][3]);
                acc[r][0] = fmaf(a.y, w[1].x, acc[r][0]); acc[r][1] = fmaf(a.y, w[1].y, acc[r][1]);
                acc[r][2] = fmaf(a.y, w[1].z, acc[r][2]); acc[r][3] = fmaf(a.y, w[1].w, acc[r][3]);
                acc[r][0] = fmaf(a.z, w[2].x, acc[r][0]); acc[r][1] = fmaf(a.z, w[2].y, acc[r][1]);
                acc[r][2] = fmaf(a.z, w[2].z, acc[r][2]); acc[r][3] = fmaf(a.z, w[2].w, acc[r][3]);
                acc[r][0] = fmaf(a.w, w[3].x, acc[r][0]); acc[r][1] = fmaf(a.w, w[3].y, acc[r][1]);
                acc[r][2] = fmaf(a.w, w[3].z, acc[r][2]); acc[r][3] = fmaf(a.w, w[3].w, acc[r][3]);
            }
        }
        const float4 b = __ldg(reinterpret_cast<const float4*>(p.bias + cg * 4));
        const int col = cg * 4;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int row = r0 + rg * 8 + r;
            if (row >= N) continue;
            const float o0 = acc[r][0] + b.x, o1 = acc[r][1] + b.y, o2 = acc[r][2] + b.z, o3 = acc[r][3] + b.w;
            if (col < 2 * p.C1) {
                __nv_bfloat16* dst = (col < p.C1) ? p.U + (size_t)row * p.C1 + col : p.V + (size_t)row * p.C1 + (col - p.C1);
                *reinterpret_cast<uint2*>(dst) = make_uint2(pack_bf16x2(o0, o1), pack_bf16x2(o2, o3));
            } else {
                *reinterpret_cast<float4*>(p.R + (size_t)row * p.C3 + (col - 2 * p.C1)) = make_float4(o0, o1, o2, o3);
            }
        }
    }
}

// ---- host side: weight packing and launch -----------------------------------------------------------------------------
struct Bf16BlockDev {
    const uint8_t* wimg = nullptr;
    const float* shifts = nullptr;
    const float* pre_Wt = nullptr;
    const float* pre_bias = nullptr;
    int cin = 0, Kp = 0, C = 0, NC = 0;
    int grid_cap = 148;
};
struct Bf16Scratch {
    __nv_bfloat16* U = nullptr;
    __nv_bfloat16* V = nullptr;
    float* R = nullptr;
};

uint16_t f32_to_bf16_rne(float f) {
    uint32_t u;
    std::memcpy(&u, &f, 4);
    if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x40);   // NaN
    u += 0x7fffu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

template <typename T>
int upload(gnn_model& m, const std::vector<T>& h, const T** out) {
    void* d = nullptr;
    GNN_CUDA_TRY(cudaMalloc(&d, std::max<size_t>(h.size(), 1) * sizeof(T)));
    m.allocs.push_back(d);
    GNN_CUDA_TRY(cudaMemcpy(d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
    *out = static_cast<const T*>(d);
    return GNN_OK;
}

// [C][C] folded fp32 weights of one layer -> chunk images (nh, kb), appended to img
void pack_layer(const std::vector<float>& W, int C, std::vector<uint8_t>& img) {
    const int NR = C > 256 ? 256 : C, NH = C / NR, KB = (C + 63) / 64;
    for (int nh = 0; nh < NH; ++nh)
        for (int kb = 0; kb < KB; ++kb) {
            const size_t base = img.size();
            img.resize(base + (size_t)NR * 128, 0);
            for (int nl = 0; nl < NR; ++nl)
                for (int kk = 0; kk < 64; ++kk) {
                    const int kcol = kb * 64 + kk, n = nh * NR + nl;
                    const uint16_t v = kcol < C ? f32_to_bf16_rne(W[(size_t)n * C + kcol]) : 0;
                    const size_t off = base + (size_t)nl * 128 + (size_t)(((kk >> 3) ^ (nl & 7)) << 4) + (kk & 7) * 2;
                    std::memcpy(&img[off], &v, 2);
                }
        }
}

template <int C>
int configure_edge(Bf16BlockDev& b, int n_sms) {
    GNN_CUDA_TRY(cudaFuncSetAttribute(edge_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, EdgeCfg<C>::SMEM_BYTES));
    int occ = 0;
    GNN_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, edge_kernel<C>, EDGE_THREADS, EdgeCfg<C>::SMEM_BYTES));
    if (occ < 1) return GNN_ERR_BAD_ARCH;
    const int tmem_cap = 512 / EdgeCfg<C>::TMEM_COLS;           // co-resident CTAs must all fit their TMEM columns
    b.grid_cap = n_sms * std::min(occ, tmem_cap);
    return GNN_OK;
}

template <int C>
void launch_edge_t(const EdgeParams& p, int grid, cudaStream_t s) {
    edge_kernel<C><<<grid, EDGE_THREADS, EdgeCfg<C>::SMEM_BYTES, s>>>(p);
}

}  // namespace

int edgeconv_bf16_prepare(gnn_model& m, const float* blob) {
    const gnn_arch& a = m.arch;
    const float* p = blob;
    auto* blocks = new Bf16BlockDev[GNN_MAX_BLOCKS];
    m.bf16_blocks = blocks;
    for (int l = 0; l < a.n_blocks; ++l) {
        const int cin = block_in(a, l), C = a.channels[l][0];
        const float* W1 = p; p += (size_t)C * 2 * cin;
        const float* s1 = p; p += C;
        const float* t1 = p; p += C;
        const float* W2 = p; p += (size_t)C * C;
        const float* s2 = p; p += C;
        const float* t2 = p; p += C;
        const float* W3 = p; p += (size_t)C * C;
        const float* s3 = p; p += C;
        const float* t3 = p; p += C;
        const float* Ws = p; p += (size_t)C * cin;
        const float* ss = p; p += C;
        const float* ts = p; p += C;
        Bf16BlockDev& b = blocks[l];
        b.cin = cin; b.C = C; b.Kp = (cin + 3) & ~3; b.NC = 3 * C;
        // pre weights: columns [u | v | r], rows = input channel (transposed), scale folded in fp32
        std::vector<float> Wt((size_t)b.Kp * b.NC, 0.0f), bias((size_t)b.NC, 0.0f);
        for (int o = 0; o < C; ++o) {
            for (int c = 0; c < cin; ++c) {
                const float wa = W1[(size_t)o * 2 * cin + c], wb = W1[(size_t)o * 2 * cin + cin + c];
                Wt[(size_t)c * b.NC + o] = s1[o] * (wa - wb);
                Wt[(size_t)c * b.NC + C + o] = s1[o] * wb;
                Wt[(size_t)c * b.NC + 2 * C + o] = ss[o] * Ws[(size_t)o * cin + c];
            }
            bias[o] = t1[o]; bias[2 * C + o] = ts[o];
        }
        std::vector<float> W2f((size_t)C * C), W3f((size_t)C * C), sh((size_t)2 * C);
        for (int o = 0; o < C; ++o) {
            for (int c = 0; c < C; ++c) {
                W2f[(size_t)o * C + c] = s2[o] * W2[(size_t)o * C + c];
                W3f[(size_t)o * C + c] = s3[o] * W3[(size_t)o * C + c];
            }
            sh[o] = t2[o]; sh[C + o] = t3[o];
        }
        std::vector<uint8_t> img;
        pack_layer(W2f, C, img);
        pack_layer(W3f, C, img);
        int rc;
        if ((rc = upload(m, Wt, &b.pre_Wt)) != GNN_OK || (rc = upload(m, bias, &b.pre_bias)) != GNN_OK ||
            (rc = upload(m, img, &b.wimg)) != GNN_OK || (rc = upload(m, sh, &b.shifts)) != GNN_OK)
            return rc;
        switch (C) {
            case 32: rc = configure_edge<32>(b, m.n_sms); break;
            case 64: rc = configure_edge<64>(b, m.n_sms); break;
            case 128: rc = configure_edge<128>(b, m.n_sms); break;
            case 256: rc = configure_edge<256>(b, m.n_sms); break;
            default: rc = GNN_ERR_BAD_ARCH;
        }
        if (rc != GNN_OK) return rc;
    }
    GNN_CUDA_TRY(cudaFuncSetAttribute(pre_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
    for (auto& w : m.ws) {
        auto* sc = new Bf16Scratch();
        w.bf16_scratch = sc;
        void* d = nullptr;
        GNN_CUDA_TRY(cudaMalloc(&d, (size_t)m.Nmax * m.Cmax * sizeof(__nv_bfloat16))); m.allocs.push_back(d); sc->U = (__nv_bfloat16*)d;
        GNN_CUDA_TRY(cudaMalloc(&d, (size_t)m.Nmax * m.Cmax * sizeof(__nv_bfloat16))); m.allocs.push_back(d); sc->V = (__nv_bfloat16*)d;
        GNN_CUDA_TRY(cudaMalloc(&d, (size_t)m.Nmax * m.Cmax * sizeof(float))); m.allocs.push_back(d); sc->R = (float*)d;
    }
    return GNN_OK;
}

void edgeconv_bf16_release(gnn_model& m) {
    delete[] static_cast<Bf16BlockDev*>(m.bf16_blocks);
    m.bf16_blocks = nullptr;
    for (auto& w : m.ws) { delete static_cast<Bf16Scratch*>(w.bf16_scratch); w.bf16_scratch = nullptr; }
}

int launch_edgeconv_bf16(gnn_model& m, int block, const float* x, const int32_t* idx, int N, float* y, Workspace& w,
                         cudaStream_t s) {
    if (N == 0) return 0;
    const Bf16BlockDev& b = static_cast<const Bf16BlockDev*>(m.bf16_blocks)[block];
    const Bf16Scratch& sc = *static_cast<const Bf16Scratch*>(w.bf16_scratch);
    const int k = m.arch.k;
    PreParams pp;
    pp.x = x; pp.Wt = b.pre_Wt; pp.bias = b.pre_bias; pp.U = sc.U; pp.V = sc.V; pp.R = sc.R; pp.meta = w.meta;
    pp.cin = b.cin; pp.Kp = b.Kp; pp.C1 = b.C; pp.C3 = b.C; pp.NC = b.NC;
    const size_t pre_smem = (size_t)PRE_ROWS * (b.Kp + 4) * sizeof(float);
    pre_kernel<<<(N + PRE_ROWS - 1) / PRE_ROWS, PRE_THREADS, pre_smem, s>>>(pp);
    EdgeParams ep;
    ep.U = sc.U; ep.V = sc.V; ep.R = sc.R; ep.idx = idx; ep.y = y; ep.meta = w.meta; ep.wimg = b.wimg; ep.shifts = b.shifts;
    ep.k = k; ep.logk = 0;
    while ((1 << ep.logk) < k) ++ep.logk;
    ep.TP = TILE_ROWS / k;
    ep.n_tiles = (N + ep.TP - 1) / ep.TP;
    const int grid = std::min(ep.n_tiles, b.grid_cap);
    switch (b.C) {
        case 32: launch_edge_t<32>(ep, grid, s); break;
        case 64: launch_edge_t<64>(ep, grid, s); break;
        case 128: launch_edge_t<128>(ep, grid, s); break;
        case 256: launch_edge_t<256>(ep, grid, s); break;
        default: return GNN_ERR_BAD_ARCH;
    }
    return 2;
}

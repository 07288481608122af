// edgeconv_f32.cu -- steps a2/a4/a6 in GNN_FP32_VALIDATION mode: the EdgeConv block exactly as stated
// (PAPER.md L262 three EdgeConv blocks, channels (C1,C2,C3); BASELINE.json north_star (2): gather neighbours, form
// e_ij = [x_i, x_j - x_i], 3-layer shared MLP with BN folded in and ReLU, mean over k, add the 1x1 shortcut) with
// every contraction in true fp32 FMA on CUDA cores (R18) -- no tensor cores, no factorisation.
//
// One CTA per tile of TP consecutive packed particles (padding-free: tiles ignore jet boundaries, neighbour indices
// are global).  The R = TP*k edge rows of the tile live in two shared-memory buffers that ping-pong through the three
// layers, so the [N*k, C] edge tensor never leaves the SM.  Each layer is a register-tiled SGEMM: a thread owns
// 8 rows x 4 columns, reads activations from shared memory (float4 along K, broadcast across the warp) and the
// folded, transposed weights Wt[K][Nout] from global memory / L1 (float4 along Nout, coalesced).
#include "gnn_internal.h"

namespace {

constexpr int EC_THREADS = 256;

// out[r][o] = act( sum_kk in[r][kk] * Wt[kk][o] + shift[o] ),  r < Rp (multiple of 8), o < Nout (multiple of 4)
__device__ __forceinline__ void tile_linear(const float* __restrict__ in, int ld_in, float* __restrict__ out, int ld_out,
                                            int Rp, const float* __restrict__ Wt, const float* __restrict__ shift,
                                            int Kp, int Nout, bool relu) {
    const int ncg = Nout >> 2;
    const int items = (Rp >> 3) * ncg;
    for (int it = threadIdx.x; it < items; it += EC_THREADS) {
        const int rg = it / ncg, cg = it - rg * ncg;
        float acc[8][4];
#pragma unroll
        for (int r = 0; r < 8; ++r) { acc[r][0] = acc[r][1] = acc[r][2] = acc[r][3] = 0.0f; }
        const float* a0 = in + (size_t)(rg * 8) * ld_in;
        const float* w0 = Wt + cg * 4;
        for (int kk = 0; kk < Kp; kk += 4) {
            float4 w[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) w[q] = __ldg(reinterpret_cast<const float4*>(w0 + (size_t)(kk + q) * Nout));
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                float4 a = *reinterpret_cast<const float4*>(a0 + (size_t)r * ld_in + kk);
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
        const float4 sh = __ldg(reinterpret_cast<const float4*>(shift + cg * 4));
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            float4 v = make_float4(acc[r][0] + sh.x, acc[r][1] + sh.y, acc[r][2] + sh.z, acc[r][3] + sh.w);
            if (relu) { v.x = fmaxf(v.x, 0.f); v.y = fmaxf(v.y, 0.f); v.z = fmaxf(v.z, 0.f); v.w = fmaxf(v.w, 0.f); }
            *reinterpret_cast<float4*>(out + (size_t)(rg * 8 + r) * ld_out + cg * 4) = v;
        }
    }
}

struct EcParams {
    const float* x; const int32_t* idx; float* y; const int32_t* meta;
    LinF32 l1, l2, l3, sc;
    int cin, k, TP, Rp, ldA, ldB;
};

__global__ void __launch_bounds__(EC_THREADS) edgeconv_f32_kernel(EcParams p) {
    extern __shared__ __align__(16) float smem[];
    if (p.meta[0]) return;
    const int N = p.meta[1];
    const int p0 = blockIdx.x * p.TP;
    if (p0 >= N) return;
    const int np = min(p.TP, N - p0);
    float* A = smem;                                   // [Rp][ldA]
    float* Bf = A + (size_t)p.Rp * p.ldA;              // [Rp][ldB]
    float* Xi = Bf + (size_t)p.Rp * p.ldB;             // [TP][cin4]  block inputs of the tile's particles
    int* valid = reinterpret_cast<int*>(Xi + (size_t)p.TP * ((p.cin + 3) & ~3));   // [Rp]
    const int cin = p.cin, k = p.k, cin4 = (cin + 3) & ~3;
    const int K1p = p.l1.Kp;                           // 2*cin padded to a multiple of 4

    // O2: edge features e = [x_i ; x_j - x_i] (zero rows for missing neighbours and for the row padding)
    for (int e = threadIdx.x; e < p.TP * cin4; e += EC_THREADS) {
        int pt = e / cin4, c = e - pt * cin4;
        Xi[e] = (pt < np && c < cin) ? p.x[(size_t)(p0 + pt) * cin + c] : 0.0f;
    }
    for (int r = threadIdx.x; r < p.Rp; r += EC_THREADS) {
        int pt = r / k, m = r - pt * k;
        int j = (pt < np) ? p.idx[(size_t)(p0 + pt) * k + m] : -1;
        valid[r] = j;
    }
    __syncthreads();
    for (int e = threadIdx.x; e < p.Rp * K1p; e += EC_THREADS) {
        int r = e / K1p, c = e - r * K1p;
        int j = valid[r];
        float v = 0.0f;
        if (j >= 0) {
            int pt = r / k;
            if (c < cin) v = Xi[pt * cin4 + c];
            else if (c < 2 * cin) v = p.x[(size_t)j * cin + (c - cin)] - Xi[pt * cin4 + (c - cin)];
        }
        A[(size_t)r * p.ldA + c] = v;
    }
    __syncthreads();
    // O3: three linear + folded affine + ReLU layers
    tile_linear(A, p.ldA, Bf, p.ldB, p.Rp, p.l1.Wt, p.l1.shift, p.l1.Kp, p.l1.N, true);
    __syncthreads();
    tile_linear(Bf, p.ldB, A, p.ldA, p.Rp, p.l2.Wt, p.l2.shift, p.l2.Kp, p.l2.N, true);
    __syncthreads();
    tile_linear(A, p.ldA, Bf, p.ldB, p.Rp, p.l3.Wt, p.l3.shift, p.l3.Kp, p.l3.N, true);
    __syncthreads();
    // O4-O6: mean over the valid neighbours, shortcut, ReLU
    const int c3 = p.l3.N;
    for (int e = threadIdx.x; e < np * c3; e += EC_THREADS) {
        int pt = e / c3, o = e - pt * c3;
        float s = 0.0f; int cnt = 0;
        for (int m = 0; m < k; ++m) {
            int r = pt * k + m;
            if (valid[r] >= 0) { s += Bf[(size_t)r * p.ldB + o]; ++cnt; }
        }
        float a = cnt > 0 ? s / (float)cnt : 0.0f;
        float sc = 0.0f;
        for (int c = 0; c < cin; ++c) sc = fmaf(Xi[pt * cin4 + c], __ldg(p.sc.Wt + (size_t)c * p.sc.ld + o), sc);
        sc += __ldg(p.sc.shift + o);
        p.y[(size_t)(p0 + pt) * c3 + o] = fmaxf(a + sc, 0.0f);
    }
}

struct EcGeom { int TP, Rp, ldA, ldB; size_t smem; };

EcGeom ec_geometry(const BlockDev& b, int k) {
    int wA = max(b.l1.Kp, b.c2) + 4;      // buffer A holds e (layer-1 input) and h2
    int wB = max(b.c1, b.c3) + 4;         // buffer B holds h1 and h3
    int cin4 = (b.cin + 3) & ~3;
    const size_t budget = 200 * 1024;
    int TP = 128 / k; if (TP < 1) TP = 1;
    for (;; --TP) {
        int Rp = (TP * k + 7) & ~7;
        size_t smem = ((size_t)Rp * (wA + wB) + (size_t)TP * cin4) * sizeof(float) + (size_t)Rp * sizeof(int);
        if (smem <= budget || TP == 1) return EcGeom{TP, Rp, wA, wB, smem};
    }
}

}  // namespace

int edgeconv_f32_configure() {
    if (cudaFuncSetAttribute(edgeconv_f32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess)
        return GNN_ERR_CUDA;
    return GNN_OK;
}

int launch_edgeconv_f32(const BlockDev& b, int k, const float* x, const int32_t* idx, int N, float* y,
                        const Workspace& w, cudaStream_t s) {
    if (N == 0) return 0;
    EcGeom g = ec_geometry(b, k);
    if (g.smem > 227 * 1024) return GNN_ERR_BAD_ARCH;
    EcParams p;
    p.x = x; p.idx = idx; p.y = y; p.meta = w.meta;
    p.l1 = b.l1; p.l2 = b.l2; p.l3 = b.l3; p.sc = b.sc;
    p.cin = b.cin; p.k = k; p.TP = g.TP; p.Rp = g.Rp; p.ldA = g.ldA; p.ldB = g.ldB;
    int grid = (N + g.TP - 1) / g.TP;
    edgeconv_f32_kernel<<<grid, EC_THREADS, g.smem, s>>>(p);
    return 1;
}

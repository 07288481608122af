// ingest.cu -- step a0 of the hot path: ragged descriptors (BASELINE.json north_star subsystem (4), padding-free
// handling of the ragged batch) and the stable compaction behind the padded entry point (features,
// coordinates, mask; R7: masked particles do not exist).
#include "gnn_internal.h"

// One CTA walks all jets: sanitised (start, n) so that no later kernel can index out of bounds whatever the caller's
// offsets hold.  Globally inconsistent offsets poison the whole batch (meta[0] = 1, GNN_DEV_BAD_OFFSETS); a jet
// larger than max_particles poisons only itself (jet_n < 0, GNN_DEV_JET_TOO_LARGE).  meta[1] = number of particles
// later kernels may touch.  `counts` (padded entry only) carries -1 for jets whose mask selected too many slots.
//
// Second phase: the GROUP SCHEDULE of the grouped kNN kernels (knn_group.cu).  A group is a run of consecutive whole jets
// whose rows fit one 128-row tile (at most GROUP_MAX_JETS jets; an offending ragged jet, which owns more rows than a
// tile, is a group of its own).  Greedy packing is sequential, so it is done per chunk of 32 consecutive jets by one
// warp: lane l finds next(l) = the first jet of the chunk that no longer fits a group starting at l, the group starts are
// the orbit of lane 0 under next (five pointer-doubling steps on ballots), and a block-wide scan of the chunks' group
// counts gives every group its slot.  groups[g] = (first jet, number of jets), meta[2] = number of groups.
constexpr int GROUP_ROWS = 128;
constexpr int GROUP_MAX_JETS = 16;

__global__ void __launch_bounds__(1024) ingest_kernel(const int32_t* __restrict__ offsets,
                                                      const int32_t* __restrict__ counts, int B, int N_exact, int N_cap,
                                                      int max_particles, int32_t* __restrict__ jet_start,
                                                      int32_t* __restrict__ jet_n, int32_t* __restrict__ meta,
                                                      unsigned* status, int2* __restrict__ groups) {
    __shared__ int chunk_cnt[1024];                // groups per chunk of 32 jets, then its exclusive scan
    __shared__ int warp_tot[32];
    __shared__ unsigned char rows_s[32768];        // rows a jet brings to a group (GROUP_ROWS + 1: never shares one)
    int any_bad = 0, any_big = 0;
    for (int b = threadIdx.x; b < B; b += blockDim.x) {
        int s = offsets[b], e = offsets[b + 1];
        bool bad = (s < 0) || (e < s) || (e > N_cap) || (b == 0 && s != 0) || (N_exact >= 0 && b == B - 1 && e != N_exact);
        int n = e - s;
        if (bad) { any_bad = 1; s = 0; n = -1; }
        else if (counts != nullptr && counts[b] < 0) { any_big = 1; n = -1; }       // padded: owns no packed rows
        else if (n > max_particles) { any_big = 1; n = -n; }                        // ragged: jet_n = -multiplicity
        jet_start[b] = s;
        jet_n[b] = n;
        rows_s[b] = (unsigned char)(n > 0 ? min(n, GROUP_ROWS + 1) : (n < -1 ? GROUP_ROWS + 1 : 0));   // offending ragged jet: alone
    }
    any_bad = __syncthreads_or(any_bad);
    any_big = __syncthreads_or(any_big);
    if (threadIdx.x == 0) {
        meta[0] = any_bad;
        meta[1] = any_bad ? 0 : offsets[B];
        if (any_bad) atomicOr(status, GNN_DEV_BAD_OFFSETS);
        if (any_big) atomicOr(status, GNN_DEV_JET_TOO_LARGE);
    }
    if (groups == nullptr || any_bad) { if (threadIdx.x == 0) meta[2] = 0; return; }
    // ---- group schedule (from the rows kept in shared memory: no global round trip) ------------------------------------------
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int n_chunks = (B + 31) >> 5;                         // <= 1024 for B <= 32768 (checked by the launcher)
    // pass 1: group starts per chunk -> chunk_cnt; the per-lane results are recomputed in pass 2 (cheaper than keeping them)
    auto chunk_groups = [&](int chunk, int& njets_out, unsigned& marks_out) {
        const int b = chunk * 32 + lane;
        const int rows = b < B ? (int)rows_s[b] : 0;
        int P = rows;                                           // inclusive prefix of rows inside the chunk
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, P, o); if (lane >= o) P += v; }
        const int S = P - rows;
        int next = 32;                                          // first lane that does not fit a group starting here
#pragma unroll
        for (int d = 1; d <= GROUP_MAX_JETS; ++d) {
            const int l2 = lane + d;
            const int Pv = __shfl_sync(0xffffffffu, P, l2 & 31);
            if (next == 32 && l2 < 32 && (Pv - S > GROUP_ROWS || d == GROUP_MAX_JETS)) next = l2;
        }
        if (b >= B) next = 32;
        njets_out = min(next, 32) - lane;
        if (b < B && chunk * 32 + next > B) njets_out = B - b;
        unsigned marks = 1u;                                    // lane 0 starts a group (chunk is non-empty)
        int nx = next;
#pragma unroll
        for (int it = 0; it < 5; ++it) {
            const bool mine = (marks >> lane) & 1u;
            marks |= __reduce_or_sync(0xffffffffu, (mine && nx < 32) ? (1u << nx) : 0u);
            const int n2 = __shfl_sync(0xffffffffu, nx, nx & 31);
            nx = nx < 32 ? n2 : 32;
        }
        const int nb = min(32, B - chunk * 32);                 // lanes past the batch start no group
        marks_out = nb >= 32 ? marks : (marks & ((1u << nb) - 1u));
    };
    for (int chunk = warp; chunk < n_chunks; chunk += nwarps) {
        int nj; unsigned marks;
        chunk_groups(chunk, nj, marks);
        if (lane == 0) chunk_cnt[chunk] = __popc(marks);
    }
    __syncthreads();
    // exclusive scan of chunk_cnt (n_chunks <= 1024 = blockDim): warp scans + scan of the warp totals
    {
        const int v = (int)threadIdx.x < n_chunks ? chunk_cnt[threadIdx.x] : 0;
        int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += u; }
        if (lane == 31) warp_tot[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            const int t = lane < nwarps ? warp_tot[lane] : 0;
            int ti = t;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, ti, o); if (lane >= o) ti += u; }
            warp_tot[lane] = ti - t;                            // exclusive
            if (lane == 31) meta[2] = ti;                       // total number of groups
        }
        __syncthreads();
        if ((int)threadIdx.x < n_chunks) chunk_cnt[threadIdx.x] = warp_tot[warp] + incl - v;
        __syncthreads();
    }
    for (int chunk = warp; chunk < n_chunks; chunk += nwarps) {
        int nj; unsigned marks;
        chunk_groups(chunk, nj, marks);
        if ((marks >> lane) & 1u) {
            const int slot = chunk_cnt[chunk] + __popc(marks & ((1u << lane) - 1u));
            groups[slot] = make_int2(chunk * 32 + lane, nj);
        }
    }
}

int launch_ingest(const int32_t* offsets, const int32_t* counts, int B, int N_exact, int N_cap, int max_particles,
                  Workspace& w, cudaStream_t s) {
    if (B > 32768) return GNN_ERR_BATCH_TOO_LARGE;               // group schedule: one CTA, 1024 chunks of 32 jets
    ingest_kernel<<<1, 1024, 0, s>>>(offsets, counts, B, N_exact, N_cap, max_particles, w.jet_start, w.jet_n, w.meta, w.status,
                                     w.groups);
    return 1;
}

// ---- padded entry: count -> exclusive scan -> stable scatter ----------------------------------------------------
__global__ void count_mask_kernel(const float* __restrict__ mask, int B, int P, int max_particles,
                                  int32_t* __restrict__ counts) {
    int b = blockIdx.x;
    int c = 0;
    for (int p = threadIdx.x; p < P; p += blockDim.x) c += (mask[(size_t)b * P + p] != 0.0f) ? 1 : 0;
    __shared__ int red[32];
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
        for (int i = 0; i < (int)(blockDim.x + 31) / 32; ++i) t += red[i];
        counts[b] = (t > max_particles) ? -1 : t;     // -1: offending jet, contributes no rows
    }
}

// single CTA, B <= a few 10^4: chunked Hillis-Steele scan in shared memory
__global__ void scan_counts_kernel(const int32_t* __restrict__ counts, int B, int32_t* __restrict__ offsets) {
    __shared__ int buf[1024];
    __shared__ int carry;
    if (threadIdx.x == 0) { carry = 0; offsets[0] = 0; }
    __syncthreads();
    for (int base = 0; base < B; base += 1024) {
        int i = base + threadIdx.x;
        int v = (i < B) ? max(counts[i], 0) : 0;
        buf[threadIdx.x] = v;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) {
            int t = (threadIdx.x >= (unsigned)o) ? buf[threadIdx.x - o] : 0;
            __syncthreads();
            buf[threadIdx.x] += t;
            __syncthreads();
        }
        if (i < B) offsets[i + 1] = carry + buf[threadIdx.x];
        __syncthreads();
        if (threadIdx.x == 1023) carry += buf[1023];
        __syncthreads();
    }
}

// one CTA (128 threads = 4 warps) per jet; slots are walked in order in chunks of 128 so the compaction is stable
__global__ void scatter_padded_kernel(const float* __restrict__ feats, const float* __restrict__ coords,
                                      const float* __restrict__ mask, int P, int F, int CD, int max_particles,
                                      const int32_t* __restrict__ offsets, const int32_t* __restrict__ counts,
                                      float* __restrict__ pfeats, float* __restrict__ pcoords, int channel_first) {
    int b = blockIdx.x;
    int base_out = offsets[b];
    if (counts[b] < 0) return;             // offending jet: ingest flags it, it owns no packed rows
    __shared__ int wsum[4];
    __shared__ int running;
    if (threadIdx.x == 0) running = 0;
    __syncthreads();
    for (int p0 = 0; p0 < P; p0 += 128) {
        int p = p0 + threadIdx.x;
        bool keep = (p < P) && (mask[(size_t)b * P + p] != 0.0f);
        unsigned bal = __ballot_sync(0xffffffffu, keep);
        int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
        if (lane == 0) wsum[wid] = __popc(bal);
        __syncthreads();
        int pre = running;
        for (int i = 0; i < wid; ++i) pre += wsum[i];
        pre += __popc(bal & ((1u << lane) - 1u));
        if (keep) {
            size_t src = (size_t)b * P + p, dst = (size_t)base_out + pre;
            if (channel_first) {             // [B, F, P] / [B, CD, P] (8 x 100 inputs per jet): a warp reads 32 consecutive slots
                for (int c = 0; c < F; ++c) pfeats[dst * F + c] = feats[((size_t)b * F + c) * P + p];
                for (int c = 0; c < CD; ++c) pcoords[dst * CD + c] = coords[((size_t)b * CD + c) * P + p];
            } else {
                for (int c = 0; c < F; ++c) pfeats[dst * F + c] = feats[src * F + c];
                for (int c = 0; c < CD; ++c) pcoords[dst * CD + c] = coords[src * CD + c];
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) running += wsum[0] + wsum[1] + wsum[2] + wsum[3];
        __syncthreads();
    }
}

int launch_compact_padded(const float* feats, const float* coords, const float* mask, int B, int P, int F, int CD,
                          int max_particles, Workspace& w, cudaStream_t s, bool channel_first) {
    if (B == 0) return 0;
    count_mask_kernel<<<B, 128, 0, s>>>(mask, B, P, max_particles, w.pcounts);
    scan_counts_kernel<<<1, 1024, 0, s>>>(w.pcounts, B, w.poffsets);
    scatter_padded_kernel<<<B, 128, 0, s>>>(feats, coords, mask, P, F, CD, max_particles, w.poffsets, w.pcounts, w.pfeats, w.pcoords, channel_first ? 1 : 0);
    return 3;
}


// ---- class probabilities (PAPER.md L262 ends the network in "two nodes"; the served model's FP32 output, L270, is read as
// softmax scores by the analyses): row-wise softmax of [B, n_classes] logits in fp32, max subtracted first; NaN rows stay NaN
// logits and probs may be the SAME buffer (gnn.h: "may alias"; gnn_infer_channel_first runs it in place), so neither pointer is
// __restrict__: a thread owns its row, reads z[c] before it writes probs[c], and never reads an element it has written
__global__ void softmax_kernel(const float* logits, int B, int n_classes, float* probs) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const float* z = logits + (size_t)b * n_classes;
    float mx = z[0];
    for (int c = 1; c < n_classes; ++c) mx = fmaxf(mx, z[c]);
    float sum = 0.0f;
    for (int c = 0; c < n_classes; ++c) sum += expf(z[c] - mx);
    const float inv = 1.0f / sum;
    for (int c = 0; c < n_classes; ++c) probs[(size_t)b * n_classes + c] = (z[c] != z[c]) ? z[c] : expf(z[c] - mx) * inv;
}

int launch_softmax(const float* logits, int B, int n_classes, float* probs, cudaStream_t s) {
    if (B == 0) return 0;
    softmax_kernel<<<(B + 127) / 128, 128, 0, s>>>(logits, B, n_classes, probs);
    return 1;
}

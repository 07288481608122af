// gnn_internal.h -- host runtime structures and kernel launch prototypes of libgnn.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>
#include "../../include/gnn.h"

// device status bits (sticky word per workspace slice)
enum : unsigned { GNN_DEV_BAD_OFFSETS = 1u, GNN_DEV_JET_TOO_LARGE = 2u };

// One folded linear layer as the fp32 SIMT kernels read it: Wt [Kp][Nout] (transposed, K padded to a multiple of
// 4 with zero rows), shift [Nout].  scale is already folded into Wt (include/gnn.h "Weight blob").
struct LinF32 {
    const float* Wt = nullptr;
    const float* shift = nullptr;
    int K = 0, Kp = 0, N = 0, ld = 0;   // ld = N rounded up to a multiple of 4 (row stride of Wt)
};

struct BlockDev {
    int cin = 0, c1 = 0, c2 = 0, c3 = 0;
    LinF32 l1, l2, l3, sc;   // fp32 path (and the shortcut / shifts in every mode)
};

struct Workspace {
    float* xa = nullptr;        // [Nmax, Cmax] ping
    float* xb = nullptr;        // [Nmax, Cmax] pong
    int32_t* idx = nullptr;     // [Nmax, k] global particle indices, -1 = none
    int2* pjet = nullptr;       // [Nmax] particle -> (start, n) of its jet (kNN selection: one load instead of three)
    float* dm = nullptr;        // [Nmax, max_particles rounded to 4] per-jet pairwise squared distances (kNN)
    int32_t* jet_start = nullptr;  // [Bmax] sanitised CSR
    int32_t* jet_n = nullptr;      // [Bmax] sanitised multiplicities (< 0 = offending jet; -n if it owns n packed rows)
    unsigned* status = nullptr;    // [1] sticky device status word
    int32_t* meta = nullptr;       // [4] per call: meta[0] = batch poisoned, meta[1] = particles in the batch, meta[2] = kNN groups
    int2* groups = nullptr;        // [Bmax] kNN group schedule: (first jet, jets) of runs of whole jets that fit one 128-row tile
    int32_t* pjid = nullptr;       // [Nmax] particle -> jet index (written by the grouped kNN, read by the pooling EdgeConv epilogue)
    unsigned long long* pool = nullptr;  // [Bmax, C_last] bf16 mode: per-jet channel sums of the last block's output, 2^-32 fixed point
    // padded entry
    float* pfeats = nullptr;    // [Nmax, F]
    float* pcoords = nullptr;   // [Nmax, CD]
    int32_t* poffsets = nullptr;  // [Bmax + 1]
    int32_t* pcounts = nullptr;   // [Bmax]
    void* bf16_scratch = nullptr;  // per-slice scratch of the bf16 path
    // CUDA graphs of whole forwards (gnn_infer_slice): a call whose arguments repeat an earlier call's exactly is replayed as
    // one graph launch instead of ~11 kernel launches (small batches are bound by the host's launch rate otherwise)
    struct ForwardGraph {
        const void *feats = nullptr, *coords = nullptr, *offsets = nullptr, *logits = nullptr;
        int B = 0, N = 0, n_launches = 0;
        cudaGraphExec_t exec = nullptr;      // null: seen once, not captured yet
        uint64_t last_use = 0;
    };
    std::vector<ForwardGraph> graphs;
    uint64_t graph_clock = 0;
    bool pool_self_cleaning = false;   // the head kernel of this model clears `pool` after reading it (else forward() does)
    float* hlogits = nullptr;      // [Bmax, n_classes] device staging of gnn_infer_host (inputs stage in pfeats/pcoords/poffsets)
    unsigned* h_status = nullptr;  // pinned copy of the status word (gnn_infer_host_begin / _end)
    bool host_pending = false;     // a gnn_infer_host_begin of this slice has not been collected yet
    // stage timing (gnn_profile_*): events of up to PROF_MAX_FORWARDS forwards, (n_stages + 1) per forward
    bool prof_on = false;
    int prof_stages = 0;                       // stages per forward (fixed for a model)
    int prof_forwards = 0;                     // forwards recorded since enable
    std::vector<cudaEvent_t> prof_events;
    std::vector<std::string> prof_names;
};
enum { PROF_MAX_FORWARDS = 512, GNN_MAX_FORWARD_GRAPHS = 8 };

struct gnn_model {
    gnn_arch arch{};
    int device = 0;
    int n_sms = 148;
    int64_t Nmax = 0;
    int Cmax = 0;
    std::vector<void*> allocs;          // everything cudaMalloc'ed, freed in gnn_destroy
    BlockDev blocks[GNN_MAX_BLOCKS];
    LinF32 fc[GNN_MAX_FC + 1];
    int n_fc = 0;
    std::vector<Workspace> ws;
    std::atomic<int64_t> launches{0};
    void* bf16_blocks = nullptr;        // edgeconv_bf16.cu: per-block packed weights of the tcgen05 path
};

#define GNN_CUDA_TRY(expr)                                                              \
    do {                                                                                \
        cudaError_t _e = (expr);                                                        \
        if (_e != cudaSuccess) {                                                        \
            std::fprintf(stderr, "libgnn: %s failed: %s (%s:%d)\n", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
            return GNN_ERR_CUDA;                                                        \
        }                                                                               \
    } while (0)

static inline int block_in(const gnn_arch& a, int l) { return l == 0 ? a.in_features : a.channels[l - 1][2]; }

// ---- kernel launchers (each returns the number of kernels it enqueued, or a negative gnn_status) ----------------
int launch_ingest(const int32_t* offsets, const int32_t* counts, int B, int N_exact, int N_cap, int max_particles,
                  Workspace& w, cudaStream_t s);
int launch_compact_padded(const float* feats, const float* coords, const float* mask, int B, int P, int F, int CD,
                          int max_particles, Workspace& w, cudaStream_t s, bool channel_first = false);
int launch_softmax(const float* logits, int B, int n_classes, float* probs, cudaStream_t s);
// kNN: space [N, D]; out [N, k] global indices (local_out = 0) or jet-local (local_out = 1)
// gram != 0 (bf16 mode, R28): the grouped kernels of knn_group.cu where they have a form for D (Gram distances on
// the tensor cores for feature spaces, 32-bit keys: d to 16 mantissa bits | j); 0: exact direct differences, exact (d, j) order
// dep (forward only, grouped kernels only): role of the kernel in a pair of programmatic dependent launches, see DEP_* below
int launch_knn(const float* space, int D, int k, int B, int max_particles, const Workspace& w, int32_t* idx_out,
               int local_out, int gram, cudaStream_t s, int dep = 0);
int launch_edgeconv_f32(const BlockDev& b, int k, const float* x, const int32_t* idx, int N, float* y,
                        const Workspace& w, cudaStream_t s);
int launch_globalize_idx(const int32_t* idx_local, int k, int B, const Workspace& w, int32_t* idx_global, cudaStream_t s);
int launch_pool_head(const gnn_model& m, const float* x, int B, const Workspace& w, float* logits, cudaStream_t s, bool pdl = false);
bool head_clears_pool(const gnn_model& m);
int launch_pooled_mean(const gnn_model& m, int B, const Workspace& w, float* g, cudaStream_t s);
int knn_configure();
int pool_head_configure();
int knn_group_configure();
int launch_knn_group(const float* space, int D, int k, int B, int max_particles, const Workspace& w, int32_t* idx_out,
                     int local_out, int dep, cudaStream_t s);
bool knn_group_supported(int D, int max_particles);
int edgeconv_f32_configure();


// ---- programmatic dependent launch (PDL) --------------------------------------------------------------------------------
// A kernel launched with `pdl` may start while the kernel before it in the stream is still running, once every CTA of that
// kernel has executed grid_dep_launch() (or exited).  It must execute grid_dep_wait() before it touches anything the earlier
// kernel writes (or reads and this kernel overwrites); what it does before that -- barrier and TMEM set-up, weight loads --
// overlaps the earlier kernel's tail.  Both instructions are no-ops in a kernel launched without the attribute.
// Two kernels that both depend only on the kernel before them (the per-particle pre kernel and the kNN of a block) run side
// by side as a PRIMARY / SECONDARY pair on one stream:
//   DEP_PRIMARY    launched as a dependent of the kernel before it; waits for it (after its own prologue), then at once
//                  releases its dependents.  It must be the kernel whose CTAs are all resident at once, because the
//                  secondary can only launch when every primary CTA has got that far.
//   DEP_SECONDARY  launched as a dependent of the primary; does NOT wait before reading its inputs -- a secondary CTA exists
//                  only after every primary CTA has passed its wait, i.e. the inputs of both are complete -- but its CTA 0
//                  waits for the primary before it exits, so that the pair is complete when the secondary is: the next
//                  kernel (the edge kernel, also launched with the attribute) passes its own grid_dep_wait after both.
// What a kernel may read BEFORE its grid_dep_wait: anything written two or more kernels back.  A dependent CTA exists only
// once every CTA of its predecessor has released its dependents, and the predecessors here release only after their own
// wait (primary) or exist only after the primary's wait (secondary); so everything before the pair -- the ingest kernel's
// meta[] and jet descriptors in particular -- is complete and visible to any CTA of any later kernel from its first
// instruction.  The edge kernels read meta[0..1] that early for this reason.
enum { DEP_NONE = 0, DEP_PRIMARY = 1, DEP_SECONDARY = 2 };
#ifdef __CUDACC__
__device__ __forceinline__ void grid_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_dep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

bool gnn_pdl_enabled();       // always true; -DGNN_DEV_KNOBS builds turn it off with GNN_NO_PDL in the environment (A/B of the overlap)

template <typename... KArgs, typename... Args>
cudaError_t launch_k(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, bool pdl, Args&&... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = (pdl && gnn_pdl_enabled()) ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}
#endif

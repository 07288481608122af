/* gnn.h -- C ABI of libgnn.so: batched forward inference of a dynamic-graph EdgeConv network of the ParticleNet
 * shape on one B200 (sm_100a), plus a host-side dynamic batcher.
 *
 * What is computed (citations are PAPER.md line numbers; readings R1-R27 are listed in DESIGN.md):
 *   PAPER.md L97   "ParticleNet ... applies dynamic graph convolutional neural networks and edge convolution
 *                   techniques to variable-dimensioned, unordered point cloud data"
 *   PAPER.md L262  (App. B) "five input features, two coordinates, three EdgeConv Blocks using k=16 nearest
 *                   neighbors and C=(64,64,64),(128,128,128),(256,256,256) channels, and two fully connected
 *                   layers with 256 nodes and 0.1 dropout rate to two nodes"
 *   PAPER.md L269  three FP32 inputs (features, coordinates, mask), FP32 output; L270 inference mode
 *   PAPER.md L53, L268, L271  dynamic batching (preferred batch 1024) and concurrent model instances
 * Per jet b with n particles, block l = 1..L (C_in -> C1,C2,C3), k_eff = min(k, n-1):
 *   kNN      N_i = the k_eff particles j != i of the same jet smallest under the strict order (d_ij, j),
 *            d_ij = sum_c (s_ic - s_jc)^2, s = coordinates for block 1, the previous block's output afterwards
 *   EdgeConv e_ij = [x_i ; x_j - x_i];  three times h <- ReLU(scale*(W h) + shift);  a_i = mean_j h3_ij;
 *            x'_i = ReLU(a_i + scale_s*(W_s x_i) + shift_s)
 *   pool     g = (1/n) sum_i x^L_i (g = 0 for an empty jet);  head: hidden FC + ReLU (dropout = identity), final FC.
 *
 * Conventions: every function returns GNN_OK (0) or a negative gnn_status; nothing throws across the ABI.
 * "dev" pointers are CUDA device pointers on the model's device, "host" pointers are host memory.  Only
 * gnn_create / gnn_destroy / gnn_batcher_create / gnn_batcher_destroy / gnn_status_check allocate or synchronise;
 * gnn_infer* and gnn_debug_* only enqueue kernels on the caller's stream and return.  There is no CPU fallback:
 * without a CUDA device gnn_create fails with GNN_ERR_CUDA.
 */
#ifndef GNN_H_
#define GNN_H_
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gnn_model   gnn_model;     /* opaque; owns device copies of the folded/packed weights + workspace */
typedef struct gnn_batcher gnn_batcher;   /* opaque; owns threads, pinned staging buffers and CUDA streams */

enum { GNN_MAX_BLOCKS = 4, GNN_MAX_FC = 3, GNN_MAX_PARTICLES = 128, GNN_MAX_K = 32, GNN_MAX_SLICES = 8 };

typedef enum {
    GNN_OK = 0,
    GNN_ERR_NULL = -1,            /* a required pointer is NULL */
    GNN_ERR_BAD_ARCH = -2,        /* gnn_arch field out of range (see gnn_arch) */
    GNN_ERR_BAD_BLOB_SIZE = -3,   /* bytes != gnn_weights_bytes(arch) */
    GNN_ERR_BATCH_TOO_LARGE = -4, /* B > max_batch_jets, N > max_batch_jets*max_particles, or bad slice */
    GNN_ERR_CUDA = -5,            /* a CUDA runtime call failed (including: no device) */
    GNN_ERR_BAD_OFFSETS = -6,     /* device check: offsets[0] != 0, not monotone, or offsets[B] != N (all logits NaN) */
    GNN_ERR_JET_TOO_LARGE = -7,   /* device check: some jet has more than max_particles particles (its logits NaN) */
    GNN_ERR_BAD_ARG = -8,         /* negative sizes, bad k / D in a debug call, bad batcher options */
    GNN_ERR_TIMEOUT = -9,         /* gnn_batcher_wait timed out (the ticket stays valid) */
    GNN_ERR_QUEUE_FULL = -10,     /* gnn_batcher_submit: max_pending_requests reached */
    GNN_ERR_BAD_TICKET = -11      /* unknown or already collected ticket */
} gnn_status;

typedef enum {
    GNN_FP32_VALIDATION = 0,  /* every contraction in fp32 FMA on CUDA cores (R18) */
    GNN_BF16 = 1              /* edge-MLP GEMMs as bf16 x bf16 -> fp32 tcgen05 MMAs; per-particle GEMM of blocks >= 2, kNN Gram
                                 matrices of blocks >= 2 and the stored shortcut in fp16 (10 mantissa bits; saturating at 65504:
                                 activations must stay below that); neighbour selection on 32-bit keys in every block; E3 row
                                 sum in f16x2; accumulators, block outputs, pool, head fp32 (R19, R28).
                                 Non-finite or blown-up activations are NOT propagated in this mode: each ReLU is an fmax
                                 (NaN -> 0), fp16 operands and the fixed-point pooled sums saturate, so such a jet gets finite
                                 logits and no status bit; GNN_FP32_VALIDATION propagates NaN / Inf to the logits */
} gnn_precision;

/* Architecture.  Constraints checked by gnn_create: 1 <= n_blocks <= GNN_MAX_BLOCKS;
 * coord_dims in [1,8]; 1 <= k <= GNN_MAX_K (BF16 mode: k a power of two); every channel count a multiple of 8
 * (BF16 mode: one of 32, 64, 128, 256, 512 and C1 == C2 == C3 inside a block); 0 <= n_fc_hidden <= GNN_MAX_FC;
 * 1 <= fc widths <= 1024; 1 <= n_classes <= 64; 1 <= max_particles <= GNN_MAX_PARTICLES; max_batch_jets >= 1;
 * 1 <= workspace_slices <= GNN_MAX_SLICES (0 is read as 1). */
typedef struct {
    int32_t in_features;                  /* F: per-particle input features (paper: 5; BASELINE configs: 4/7/9, R1) */
    int32_t coord_dims;                   /* 2 (L262) */
    int32_t k;                            /* neighbours, 16 (L262) */
    int32_t n_blocks;                     /* EdgeConv blocks, 3 (L262) */
    int32_t channels[GNN_MAX_BLOCKS][3];  /* (C1,C2,C3) per block */
    int32_t n_fc_hidden;                  /* hidden FC layers before the final one: 1 (FC 256 + ReLU) */
    int32_t fc_hidden[GNN_MAX_FC];
    int32_t n_classes;                    /* 2 */
    int32_t max_particles;                /* largest legal multiplicity of one jet (100 or 128 in the configs) */
    int32_t max_batch_jets;               /* sizes the workspace: largest B of one gnn_infer call */
    int32_t precision;                    /* gnn_precision */
    int32_t workspace_slices;             /* independent workspaces = max concurrent gnn_infer_slice calls */
} gnn_arch;

/* Weight blob: fp32, little-endian, in this order (weights are random in the paper's benchmark).
 * For each block l: for layer 1..3: W[out][in] row-major (layer 1: in = 2*C_in, the x_i half first, then the
 * (x_j - x_i) half), scale[out], shift[out]; then the shortcut W[C3][C_in], scale[C3], shift[C3].  Then for each FC
 * (hidden..., final): W[out][in], bias[out].  Block layers have no bias of their own: y = scale*(W x) + shift (R8).
 * gnn_create folds scale into W in fp32 and (GNN_BF16) rounds the edge-MLP weights to bf16 once (RNE). */
int gnn_weights_bytes(const gnn_arch* arch, size_t* out_bytes);

/* Copies and packs the blob (host pointer, caller keeps ownership) onto CUDA device `device`, allocates
 * `workspace_slices` workspaces sized for max_batch_jets * max_particles particles.  Synchronous. */
int gnn_create(const void* weights_host, size_t bytes, const gnn_arch* arch, int device, gnn_model** out);
void gnn_destroy(gnn_model* m);

/* Ragged forward (BASELINE.json north_star (4): padding-free).  feats_dev [N, F] and coords_dev [N, coord_dims]
 * row-major fp32, particles of one jet contiguous; offsets_dev int32 [B+1] CSR (offsets[0] = 0, offsets[B] = N);
 * logits_dev fp32 [B, n_classes] (written).  Asynchronous on `cuda_stream` (a cudaStream_t; NULL = default
 * stream).  Uses workspace slice 0 / `slice`: two calls may overlap only on different slices.  B = 0 is legal.
 * Everything is enqueued on `cuda_stream` alone (GNN_BF16: as programmatic dependent launches), so the call may be
 * captured into a CUDA graph of the caller's; gnn_infer / gnn_infer_slice also replay a graph of their own when a call's
 * arguments (pointers, B, N) repeat an earlier call's on the slice (captured on the second sighting, up to 8 per slice).
 * Host-checkable errors return at once; device-checkable ones (GNN_ERR_BAD_OFFSETS, GNN_ERR_JET_TOO_LARGE) set a
 * sticky per-slice status word read by gnn_status_check and put NaN into the offending logits.  n_b = 0 is legal
 * (logits = head(0), R12).  NaN / Inf inputs are not checked. */
int gnn_infer(gnn_model* m, const float* feats_dev, const float* coords_dev, const int32_t* offsets_dev,
              int32_t B, int32_t N, float* logits_dev, void* cuda_stream);
int gnn_infer_slice(gnn_model* m, int32_t slice, const float* feats_dev, const float* coords_dev,
                    const int32_t* offsets_dev, int32_t B, int32_t N, float* logits_dev, void* cuda_stream);

/* Padded forward (features, coordinates, mask).  feats_dev [B, P, F], coords_dev [B, P, coord_dims],
 * mask_dev [B, P] fp32, nonzero = real particle.  Masked slots are never read beyond the mask itself (they may hold
 * NaN); real particles may sit at any slots and keep their relative order (stable compaction, R7).  A jet with
 * more than max_particles real particles raises GNN_ERR_JET_TOO_LARGE.  B*P <= max_batch_jets * GNN_MAX_PARTICLES. */
int gnn_infer_padded(gnn_model* m, const float* feats_dev, const float* coords_dev, const float* mask_dev,
                     int32_t B, int32_t P, float* logits_dev, void* cuda_stream);
int gnn_infer_padded_slice(gnn_model* m, int32_t slice, const float* feats_dev, const float* coords_dev,
                           const float* mask_dev, int32_t B, int32_t P, float* logits_dev, void* cuda_stream);

/* Synchronises `cuda_stream`, returns and clears the sticky device status of `slice` (GNN_OK, GNN_ERR_BAD_OFFSETS,
 * GNN_ERR_JET_TOO_LARGE, or GNN_ERR_CUDA if the stream reports an error). */
int gnn_status_check(gnn_model* m, int32_t slice, void* cuda_stream);

/* The paper's literal I/O contract ("features", "coordinates" and "mask", all FP32; L285 Table C2: input
 * shape 8 x 100 per jet = (F + coord_dims + 1) channels x P slots, output 2): CHANNEL-FIRST padded tensors
 * points_dev [B, coord_dims, P], features_dev [B, F, P], mask_dev [B, 1, P] (slot real iff mask != 0, any slot order,
 * masked slots may hold anything).  Compacts on the device like gnn_infer_padded, runs the forward on `slice`, and
 * writes out_dev [B, n_classes]: raw logits, or with softmax != 0 the class probabilities (row-wise softmax in fp32).
 * Errors as gnn_infer_padded. */
int gnn_infer_channel_first(gnn_model* m, int32_t slice, const float* points_dev, const float* features_dev,
                            const float* mask_dev, int32_t B, int32_t P, int32_t softmax, float* out_dev, void* cuda_stream);
/* row-wise softmax of logits_dev [B, n_classes] into probs_dev (may alias), fp32, maximum subtracted first */
int gnn_softmax(const float* logits_dev, int32_t B, int32_t n_classes, float* probs_dev, void* cuda_stream);

/* The same forward from HOST buffers (layouts as gnn_infer; pinned memory makes the copies asynchronous): copies the
 * inputs to device staging owned by `slice`, runs the forward, copies logits_host [B, n_classes] back and
 * synchronises `cuda_stream` before returning.  This is the one blocking inference call.  Device-side errors are
 * returned directly (the sticky word is read and cleared). */
int gnn_infer_host(gnn_model* m, int32_t slice, const float* feats_host, const float* coords_host,
                   const int32_t* offsets_host, int32_t B, int32_t N, float* logits_host, void* cuda_stream);

/* The two halves of gnn_infer_host, for callers that keep several slices in flight: _begin enqueues the copies and the
 * forward on `cuda_stream` and returns at once (host buffers must be pinned for the copies to be asynchronous, and must stay
 * valid until _end); _end synchronises `cuda_stream`, after which logits_host is valid, and returns device-side errors.  With
 * two slices on two streams the host -> device copy of one batch runs under the forward of the other (bench.py's e2e leg).
 * One _begin per slice at a time. */
int gnn_infer_host_begin(gnn_model* m, int32_t slice, const float* feats_host, const float* coords_host,
                         const int32_t* offsets_host, int32_t B, int32_t N, float* logits_host, void* cuda_stream);
int gnn_infer_host_end(gnn_model* m, int32_t slice, void* cuda_stream);

const char* gnn_strerror(int status);
/* number of kernels the library has launched on this model since gnn_create (bench.py's gpu_launches) */
int64_t gnn_launch_count(const gnn_model* m);

/* ---- stage timing (bench.py's roofline leg) ---------------------------------------------------------------------
 * While enabled for a slice, every gnn_infer* on it records one CUDA event before the first and after each stage
 * (ingest, kNN l, EdgeConv l, ..., pool+head) on the caller's stream; up to 512 forwards are kept.  gnn_profile_read
 * synchronises on the recorded events and writes the mean milliseconds per stage over the recorded forwards;
 * *n_stages_out = stages of one forward, *n_forwards_out = forwards averaged.  Enabling clears earlier records. */
int gnn_profile_enable(gnn_model* m, int32_t slice, int32_t on);
int gnn_profile_read(gnn_model* m, int32_t slice, int32_t max_stages, float* ms_mean_out, int32_t* n_stages_out,
                     int32_t* n_forwards_out);
/* name of stage `stage` of the last recorded forward ("ingest", "knn0", "edgeconv0", ..., "pool_head"), or NULL */
const char* gnn_profile_stage_name(gnn_model* m, int32_t slice, int32_t stage);

/* ---- per-stage entry points: the same kernels the forward uses, exposed for stage-wise parity tests --------- */
/* kNN on an arbitrary space [N, D] (1 <= D <= 1024): idx_dev int32 [N, k], jet-local indices in (d, j) order,
 * -1 = none (k_eff < k). */
int gnn_debug_knn(gnn_model* m, const float* space_dev, int32_t D, const int32_t* offsets_dev, int32_t B, int32_t N,
                  int32_t k, int32_t* idx_dev, void* cuda_stream);
/* EdgeConv block `block` (0-based) given jet-local neighbour indices [N, arch.k]: x_dev [N, C_in] -> y_dev [N, C3],
 * in the model's precision mode. */
int gnn_debug_edgeconv(gnn_model* m, int32_t block, const float* x_dev, const int32_t* idx_dev,
                       const int32_t* offsets_dev, int32_t B, int32_t N, float* y_dev, void* cuda_stream);
/* GNN_BF16, k = 16, C_last <= 256 only (else GNN_ERR_BAD_ARG): the LAST EdgeConv block with the pooling epilogue the
 * forward uses in that mode (block output never stored; per-jet channel sums accumulated as exact 2^-32 fixed-point
 * integers): x_dev [N, C_in of the last block], jet-local idx_dev [N, k] -> g_dev [B, C_last] = mean over the jet's
 * particles of the block output (0 for an empty jet) = the input of the FC head. */
int gnn_debug_edgeconv_pool(gnn_model* m, const float* x_dev, const int32_t* idx_dev, const int32_t* offsets_dev,
                            int32_t B, int32_t N, float* g_dev, void* cuda_stream);
/* masked global average pool + FC head: x_dev [N, C_last] -> logits_dev [B, n_classes] */
int gnn_debug_pool_head(gnn_model* m, const float* x_dev, const int32_t* offsets_dev, int32_t B, int32_t N,
                        float* logits_dev, void* cuda_stream);

/* ---- exact kNN without a model and without any allocation --------------------------------------------------------------
 * For callers that are not allowed to allocate device memory: a plugin whose host application owns the device heap and hands
 * out fixed buffers, a real-time loop that must never wait on the allocator's device-wide lock, a process whose GPU memory
 * was fully budgeted before this library was loaded.  Those callers cannot call gnn_create either (it allocates the weights
 * and a workspace), so this entry needs no gnn_model: it is the exact kNN step alone ("k=16 nearest
 * neighbors"; same kernels, same fp32 arithmetic and (d, j) order as gnn_debug_knn on a GNN_FP32_VALIDATION model, so the
 * two return identical indices).  The kernels' intermediate data (ragged descriptors, particle -> jet map, per-jet distance
 * matrix) goes to a fixed array compiled into libgnn.so: about 4.1 MiB on every GPU that loads the library, held until the
 * process exits.  The call itself never calls cudaMalloc / cudaFree or any routine that does.
 *   space_dev [N, D] fp32 row-major (1 <= D <= 1024), offsets_dev int32 [B + 1] CSR, idx_dev int32 [N, k] (written:
 *   jet-local indices in (d, j) order, -1 behind the k_eff = min(k, n - 1) valid ones); all three are the caller's
 *   buffers on the CURRENT device (cudaSetDevice before the call on multi-GPU hosts).  Asynchronous on cuda_stream.
 * Limits: B <= 1024 jets and N <= 8192 particles per call, max_particles <= GNN_MAX_PARTICLES; anything larger is
 *   refused with GNN_ERR_BATCH_TOO_LARGE (and a line on stderr) before anything is enqueued -- split the batch.
 * First call on a device: looks up the array's device address (one cudaGetSymbolAddress, remembered per device).  Make that
 *   first call outside any stream capture.
 * Sharing: every call on a device uses the same array, and it keeps the previous call's contents (the call clears the few
 *   words that must start at zero).  Two calls whose kernels can overlap on the GPU -- different streams, or several host
 *   threads -- race on it and return garbage: keep all calls on one stream, or order them with events.
 * Offsets are checked on the device only for memory safety: with an invalid CSR (offsets[0] != 0, not monotone, offsets[B]
 *   != N) idx_dev is left untouched, and a jet with more than max_particles particles gets rows of -1; no status is
 *   reported (validate offsets on the host, where this caller has them). */
int gnn_knn_noalloc(const float* space_dev, int32_t D, const int32_t* offsets_dev, int32_t B, int32_t N,
                    int32_t max_particles, int32_t k, int32_t* idx_dev, void* cuda_stream);

/* ---- host dynamic batcher ("dynamic batching", L268 preferred batch 1024, L271 instance group) -- */
typedef struct {
    int32_t max_batch_jets;        /* coalesce up to this many jets per launch (<= arch.max_batch_jets); 1024 (L268) */
    int32_t max_queue_delay_us;    /* launch when the oldest queued request is this old; 1000 (BASELINE configs[3]) */
    int32_t n_instances;           /* concurrent launches = CUDA streams = workspace slices used (<= arch.workspace_slices) */
    int32_t max_pending_requests;  /* submit fails with GNN_ERR_QUEUE_FULL beyond this; 0 = 65536 */
} gnn_batcher_opts;
typedef struct { uint64_t id; } gnn_ticket;

int gnn_batcher_create(gnn_model* m, const gnn_batcher_opts* opts, gnn_batcher** out);
/* Thread-safe, non-blocking.  Inputs are HOST pointers laid out as in gnn_infer (offsets_host[0] = 0); they are
 * copied before the call returns.  logits_host_out [n_jets, n_classes] must stay valid until gnn_batcher_wait
 * returns for the ticket.  Offsets are validated on the host; a bad request fails alone (GNN_ERR_BAD_OFFSETS /
 * GNN_ERR_JET_TOO_LARGE) without touching its batch mates. */
int gnn_batcher_submit(gnn_batcher* b, const float* feats_host, const float* coords_host, const int32_t* offsets_host,
                       int32_t n_jets, float* logits_host_out, gnn_ticket* out);
/* Blocks until the ticket completes or timeout_us elapses (< 0: forever).  Returns the ticket's status.  queue_us =
 * submit -> launch, compute_us = launch -> logits in host memory (PAPER.md L279 splits request time this way). */
int gnn_batcher_wait(gnn_batcher* b, gnn_ticket t, int64_t timeout_us, double* queue_us, double* compute_us);
/* The same with the full split of Fig. C3: compute_us (launch -> logits in host memory, host clock) contains
 * transfer_us (host -> device and device -> host copies of the coalesced batch: the paper's "network latency", PCIe here)
 * and inference_us (the forward), both measured with CUDA events on the instance's stream. */
typedef struct { double queue_us, compute_us, transfer_us, inference_us; } gnn_request_times;
int gnn_batcher_wait_ex(gnn_batcher* b, gnn_ticket t, int64_t timeout_us, gnn_request_times* times);
int gnn_batcher_stats(gnn_batcher* b, uint64_t* n_requests, uint64_t* n_jets, uint64_t* n_launches,
                      double* mean_batch_jets);
void gnn_batcher_destroy(gnn_batcher* b);   /* drains pending tickets first */

/* ---- closed-loop load generator (App. C: perf_analyzer in synchronous mode; Table C2 sweep) ----------
 * n_clients native threads; client c cycles through requests c, c + n_clients, ... of the pool: submit -> wait -> next.
 * The pool is one ragged batch in HOST memory (layouts as gnn_infer: feats [N, F], coords [N, CD], offsets [J + 1] absolute)
 * cut into requests of consecutive jets: request r = jets [request_first_jet[r], request_first_jet[r + 1]).  After
 * warmup_ms the harness measures run_ms: jets/s, request latency (submit -> logits in client memory) mean / p50 / p90 /
 * p99, its split into queue and compute time (Fig. C3) and the mean coalesced batch size.  Blocking; returns the first
 * failing request's status, else GNN_OK. */
typedef struct {
    const float* feats_host;
    const float* coords_host;
    const int32_t* offsets_host;
    const int32_t* request_first_jet;   /* [n_requests + 1] */
    int32_t n_requests, in_features, coord_dims, n_classes;
} gnn_loadgen_pool;
typedef struct { int32_t n_clients, warmup_ms, run_ms; } gnn_loadgen_opts;
typedef struct {
    uint64_t n_requests, n_jets;
    double seconds, jets_per_s, mean_us, p50_us, p90_us, p99_us, queue_us_mean, compute_us_mean, mean_batch_jets;
    double transfer_us_mean, inference_us_mean;   /* device-side parts of compute_us (gnn_request_times) */
} gnn_loadgen_result;
int gnn_loadgen_run(gnn_batcher* b, const gnn_loadgen_pool* pool, const gnn_loadgen_opts* opts, gnn_loadgen_result* out);

/* ---- second workload: boosted-decision-tree inference (section 4.1, Fig. 6: "a small boosted decision tree
 * (BDT) with 20 input features and 100 trees"; Table C2: input shape 20, output shape 2, batches 10 K ... 2.56 M) ---
 * n_trees complete binary trees of depth `depth`.  feature_host / threshold_host [n_trees, 2^depth - 1]: internal node i
 * tests x[feature] < threshold: true -> child 2 i + 1, else (also for NaN) child 2 i + 2; leaf_host [n_trees, 2^depth]: leaf
 * j of a tree is reached at node 2^depth - 1 + j.  margin = sum over the trees, in tree order, of the reached leaves (fp32);
 * output row = (1 - p, p), p = 1 / (1 + exp(-margin)).  The arrays are copied; the forest must fit one SM's shared memory
 * (GNN_ERR_BAD_ARCH otherwise), feature indices are validated (GNN_ERR_BAD_ARG). */
typedef struct gnn_bdt gnn_bdt;
int gnn_bdt_create(const int32_t* feature_host, const float* threshold_host, const float* leaf_host, int32_t n_trees,
                   int32_t depth, int32_t n_features, int device, gnn_bdt** out);
void gnn_bdt_destroy(gnn_bdt* b);
/* x_dev [N, n_features] fp32 row-major -> out_dev [N, 2] (8-byte aligned, else GNN_ERR_BAD_ARG); asynchronous on cuda_stream */
int gnn_bdt_infer(gnn_bdt* b, const float* x_dev, int64_t N, float* out_dev, void* cuda_stream);
/* the same from / to HOST buffers (pinned memory makes the copies asynchronous); blocking; device staging owned by `b` grows
 * to the largest N seen */
int gnn_bdt_infer_host(gnn_bdt* b, const float* x_host, int64_t N, float* out_host, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* GNN_H_ */

/* trk.h -- C ABI of the B200-native Exa.TrkX inference hot path.
 *
 * One call runs the five stages of PAPER.md line 85 (section 2.2.2) on the device:
 *   S1 embedding MLP -> S2 fixed-radius graph in the latent space -> S3 filter MLP + cut ->
 *   S4 interaction-network GNN edge scores -> S5 weakly-connected components (track labels),
 * and, when asked for, S6: the track candidates as lists of hits (line 85: "Each track candidate is
 * a list of spacepoints").
 * The lifecycle mirrors the paper's backend: "loading the full
 * pipeline, performing inference, and setting the GPU device ID" == trk_create / trk_infer /
 * trk_destroy, with constants preloaded once and intermediates kept on the device (lines 77, 115).
 * Every architectural number comes from the caller (BASELINE.json configs); DESIGN.md lists the
 * readings of the paper this header relies on (C-7..C-17).
 *
 * Conventions
 *   - plain C99, no torch types; "HOST"/"DEVICE" says where a pointer must live.
 *   - all indices int32, hit features fp32 (r/1000, phi/pi, z/1000), row-major everywhere.
 *   - every function returns trk_status; no exception crosses the ABI; trk_last_error() gives text.
 *   - trk_infer and the trk_stage_* calls only enqueue work on `cuda_stream` (a cudaStream_t cast
 *     to void*, NULL = legacy default stream): they never allocate, never synchronise, and may be
 *     captured into a CUDA graph.  Host-detectable errors return before anything is enqueued.
 *   - a ctx serves one in-flight call at a time (stream-ordered); several ctxs on several streams
 *     are the analogue of several model instances.
 *   - there is no CPU fallback: trk_create fails with TRK_ERR_UNSUPPORTED_DEVICE off sm_100.
 */
#ifndef TRK_H_
#define TRK_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct trk_ctx trk_ctx; /* opaque: one "model instance" */

typedef enum {
  TRK_OK = 0,
  TRK_ERR_INVALID_ARG = 1,      /* NULL pointer, negative size, non-monotone offsets, bad enum   */
  TRK_ERR_SHAPE = 2,            /* MLP dims inconsistent with each other or with the hyperparameters */
  TRK_ERR_CAPACITY = 3,         /* a call exceeds max_hits / max_events / an output capacity      */
  TRK_ERR_CUDA = 4,             /* CUDA runtime or driver error (text in trk_last_error)          */
  TRK_ERR_OOM = 5,              /* workspace allocation failed in trk_create                      */
  TRK_ERR_UNSUPPORTED_DEVICE = 6 /* device is not compute capability 10.x                         */
} trk_status;

enum { TRK_FP32 = 0, TRK_BF16 = 1 };             /* trk_config.precision                          */
enum { TRK_FILTER_RAW = 0, TRK_FILTER_EMB = 1 }; /* trk_config.filter_input (reading C-10)        */

/* A stack of Linear layers.  weight[l] is HOST fp32 [dims[l+1]][dims[l]] (out, in) row-major,
 * bias[l] is HOST fp32 [dims[l+1]].  trk_create copies everything; the caller may free at return. */
typedef struct {
  int32_t n_layers;
  const int32_t* dims;          /* HOST, n_layers + 1 entries, e.g. {3,1024,1024,1024,12}         */
  const float* const* weight;   /* HOST array of n_layers HOST pointers                            */
  const float* const* bias;     /* HOST array of n_layers HOST pointers                            */
} trk_mlp;

typedef struct {
  uint32_t struct_size;         /* = sizeof(trk_config), for versioning                            */
  int32_t device;               /* CUDA device ordinal, fixed for the ctx lifetime */
  int32_t precision;            /* TRK_FP32: SIMT fp32 everywhere.  TRK_BF16: tcgen05 GEMMs with bf16
                                   operands (weights/activations rounded RNE) and fp32 accumulation;
                                   needs hidden widths that are multiples of 64 and H in {64,128}.  */
  /* S1: embedding MLP, ReLU between layers, none on the output. dims[0] == 3.                     */
  trk_mlp embed;
  /* S2: for every hit i the K nearest hits j of the same event with outer(i,j) and d2 <= r^2, d2 in
   * fp64 from the fp32 embedding (k ascending, no FMA); outer <=> (r,|z|,index) lexicographically
   * larger; ties in d2 -> lower index (readings C-7..C-9, C-11).  1 <= frnn_k <= 128.             */
  float frnn_radius;
  int32_t frnn_k;
  const float* grid_proj;       /* HOST fp32 [d_e][grid_dims] with orthonormal columns used only to
                                   bin hits (any such matrix gives the same graph, reading C-21);
                                   NULL = the first grid_dims latent coordinates                    */
  int32_t grid_dims;            /* 1..3                                                             */
  /* S3: score = sigmoid(MLP([u_src ; u_dst])), u = embedding row (TRK_FILTER_EMB) or raw hit row
   * (TRK_FILTER_RAW); kept iff score > filter_cut (strict); kept edges stay in (src,dst) order.    */
  trk_mlp filter;               /* dims[0] == 2*u, last dim == 1                                    */
  int32_t filter_input;
  float filter_cut;
  /* S4: interaction network of DESIGN.md "S4" (reading C-12): all five MLPs have 2 layers.        */
  int32_t gnn_hidden;           /* H                                                                */
  int32_t gnn_iters;            /* T, weights shared across iterations                              */
  int32_t gnn_layernorm;        /* 1: ReLU(LayerNorm(.)) after every GNN Linear but the last (eps 1e-5,
                                   no affine, reading C-13); 0: plain ReLU                          */
  trk_mlp node_enc;             /* 3  -> H -> H                                                     */
  trk_mlp edge_enc;             /* 4  -> H -> H   on (dr, dphi wrapped to (-1,1], dz, deta)         */
  trk_mlp edge_net;             /* 3H -> H -> H   on [h_src ; h_dst ; e], residual                  */
  trk_mlp node_net;             /* 3H -> H -> H   on [h ; sum_in e ; sum_out e], residual           */
  trk_mlp edge_dec;             /* 3H -> H -> 1   on [h_src ; h_dst ; e], then sigmoid              */
  /* S5: keep edges with gnn score > gnn_cut (strict); label = smallest hit index of the component. */
  float gnn_cut;
  /* Workspace is sized once from these; nothing is allocated later.                               */
  int64_t max_hits;             /* N summed over the events of one call                             */
  int64_t max_events;
  int64_t max_cand_edges;       /* S2 output capacity; max_hits*frnn_k can never overflow           */
  int64_t max_kept_edges;       /* S3 output capacity (data dependent)                              */
  /* S6: a track candidate is a component with at least min_track_hits hits (values < 1 mean 1;
   * the paper states no minimum, reading C-23).  Used only when track outputs are wanted. */
  int32_t min_track_hits;
  /* Workspace / search-structure sizing, 0 = default (neither changes any result):
   *   filter_chunk_rows  the layer-by-layer S3 (used when the fused S3 kernel does not apply to the filter's shape, or with
   *                      trk_set_option "filter_fused" = 0) processes the candidate edges in passes of this many rows
   *                      (rounded up to 128); its two activation buffers hold rows x widest layer bf16 each.  Default:
   *                      128 x SMs rows when the fused kernel applies (the chunked path is then only a test variant), else
   *                      128 x SMs x 64 rows (1 212 416 on a B200: 2.5 GB per buffer) -- DESIGN.md section 6.
   *   grid_max           upper bound of the S2 search grid's cells per axis and event (1..128).  Default (and upper limit):
   *                      the largest value whose cell table (max_events x grid_max^3 x 16 radius buckets) fits 2^22 entries.  */
  int64_t filter_chunk_rows;
  int32_t grid_max;
} trk_config;

typedef struct {
  int32_t n_events;
  const int32_t* event_offsets; /* HOST, n_events+1 entries, [0] == 0, non-decreasing; N = last     */
  const float* hits;            /* DEVICE fp32 [N][3]                                               */
} trk_batch;

/* Outputs: all DEVICE, caller-owned, NULL = not wanted (counts is required, labels too unless N == 0).
 * Edges are global hit indices, sorted by (src, dst).  If a capacity is too small the list is
 * truncated deterministically (lowest (src,dst) first), counts[3] is set to 1 and labels are the
 * components of the truncated graph.                                                              */
typedef struct {
  int32_t* labels;              /* [N]                                                              */
  int32_t* counts;              /* [4] = {E_c, E_k, E_t (edges passing gnn_cut), overflow flag}     */
  int32_t* edge_src;            /* [edge_capacity] kept (S3) edges                                  */
  int32_t* edge_dst;
  float* edge_score;            /* [edge_capacity] S4 sigmoid scores of the kept edges              */
  int64_t edge_capacity;
  int32_t* cand_src;            /* [cand_capacity] S2 edges                                         */
  int32_t* cand_dst;
  float* cand_score;            /* [cand_capacity] S3 sigmoid scores                                */
  int64_t cand_capacity;
  float* embedding;             /* [N][d_e] S1 output                                               */
  /* S6 (all three or none): tracks ordered by label (= their smallest hit index), the hits of a track
   * in ascending hit index.  If there are more than track_capacity tracks the first track_capacity
   * are written and counts[3] is set.                                                              */
  int32_t* track_offsets;       /* [track_capacity+1]; track t = track_hits[offsets[t] .. offsets[t+1]) */
  int32_t* track_hits;          /* [N]; entries beyond the last track are -1                         */
  int32_t* track_counts;        /* [2] = {number of tracks T, hits in tracks = track_offsets[T]}      */
  int64_t track_capacity;
} trk_result;

trk_status trk_create(const trk_config* cfg, trk_ctx** out);
trk_status trk_infer(trk_ctx* ctx, const trk_batch* batch, const trk_result* result, void* cuda_stream);
trk_status trk_destroy(trk_ctx* ctx);

/* The served request (spacepoints in, track candidates out) with HOST
 * buffers: copies hits H2D, runs trk_infer on the ctx's own stream, copies labels (and, when the
 * pointers are non-NULL, counts[4]) D2H and synchronises.  hits_host/labels_host should be pinned. */
trk_status trk_infer_host(trk_ctx* ctx, int32_t n_events, const int32_t* event_offsets,
                          const float* hits_host, int32_t* labels_host, int32_t* counts_host);

/* The same request returning the track candidates themselves: additionally copies
 * track_offsets_host[T+1] and track_hits_host[track_offsets[T]] D2H; both must hold N+1 / N entries.
 * counts_host is [6] = counts[4] followed by {T, hits in tracks}.  labels_host may be NULL.          */
trk_status trk_infer_host_tracks(trk_ctx* ctx, int32_t n_events, const int32_t* event_offsets, const float* hits_host,
                                 int32_t* labels_host, int32_t* track_offsets_host, int32_t* track_hits_host,
                                 int32_t* counts_host);

const char* trk_status_string(trk_status s);
const char* trk_last_error(const trk_ctx* ctx); /* ctx may be NULL: error of the last failed trk_create */
int64_t trk_workspace_bytes(const trk_ctx* ctx);
/* Number of kernels of this library launched by the most recent trk_infer on ctx (host-side count; reset on entry, so it
 * is 0 after a call that was refused before anything was enqueued). */
int64_t trk_last_launch_count(const trk_ctx* ctx);

/* Per-stage timing of trk_infer with CUDA events recorded on the call's stream at the stage
 * boundaries (the analogue of perf_analyzer's latency breakdown).
 * trk_profile_enable(ctx, 1) creates the CUDA events (the only allocation of the profiling mode: trk_infer itself never
 * allocates) and makes the following trk_infer calls record 6 events; trk_profile_stage_ms
 * waits for the last one and writes the HOST array ms[5] = {S1, S2, S3 (incl. compaction), S4, S5}. */
trk_status trk_profile_enable(trk_ctx* ctx, int32_t on);
trk_status trk_profile_stage_ms(trk_ctx* ctx, float* ms);
/* Per-launch device time of the dominant kernel of the path, from CUDA-event pairs recorded around each
 * such launch of the last profiled trk_infer.  With the fused S3 kernel (the default) there is ONE launch that runs every
 * layer of the filter MLP over all counts[0] candidate edges and *rows_per_launch is -1.  With the layer-by-layer S3
 * ("filter_fused" = 0) the launches are the hidden-layer GEMMs (K >= 256) in launch order: chunk 0 layer 2, chunk 0 layer 3,
 * chunk 1 layer 2, ...; chunk c covers candidate edges [c * *rows_per_launch, (c+1) * *rows_per_launch) clipped to counts[0]
 * (launches of chunks beyond the candidate count are empty) and a launch does 2 * rows * K * N flop with K = N = the hidden
 * width.  Writes HOST ms[min(capacity, *n_launches)]. */
trk_status trk_profile_kernel_ms(trk_ctx* ctx, float* ms, int32_t capacity, int32_t* n_launches, int64_t* rows_per_launch);

/* Stage hooks: run ONE stage on caller-supplied DEVICE inputs (BASELINE.json north_star: "each
 * stage fed the oracle's own inputs for that stage").  Same kernels as trk_infer.  Unless noted
 * all pointers are DEVICE; sizes are HOST scalars and must respect the ctx capacities.            */

/* S1: emb fp32 [n][d_e]. */
trk_status trk_stage_embed(trk_ctx* ctx, const float* hits, int64_t n, float* emb, void* cuda_stream);
/* S2: writes src/dst [<= capacity] sorted by (src,dst), rowptr [n+1], count[2] = {E_c, overflow}.
 * event_offsets is HOST. */
trk_status trk_stage_frnn(trk_ctx* ctx, const float* emb, const float* hits, const int32_t* event_offsets,
                          int32_t n_events, int32_t* src, int32_t* dst, int32_t* rowptr, int64_t capacity,
                          int32_t* count, void* cuda_stream);
/* S3: score fp32 [n_edges] for the given edges; feat is the embedding [n][d_e] or the hits [n][3]
 * according to filter_input.  n is the number of rows of feat. */
trk_status trk_stage_filter(trk_ctx* ctx, const float* feat, int64_t n, const int32_t* src, const int32_t* dst,
                            int64_t n_edges, float* score, void* cuda_stream);
/* S3 tail: stable compaction of the edges with score > filter_cut; count[2] = {E_k, overflow}. */
trk_status trk_stage_compact(trk_ctx* ctx, const int32_t* src, const int32_t* dst, const float* score,
                             int64_t n_edges, int32_t* out_src, int32_t* out_dst, int64_t capacity,
                             int32_t* count, void* cuda_stream);
/* S4: score fp32 [n_edges] = sigmoid(GNN logit).  Edges must be sorted by (src,dst). */
trk_status trk_stage_gnn(trk_ctx* ctx, const float* hits, int64_t n, const int32_t* src, const int32_t* dst,
                         int64_t n_edges, float* score, void* cuda_stream);
/* S4 bookkeeping only: the scatter structure of the message passing, as trk_stage_gnn builds it (same kernels).  Edges
 * sorted by (src,dst).  in_rowptr [n+1] / in_perm [n_edges]: the in-edges of node v are in_perm[in_rowptr[v] ..
 * in_rowptr[v+1]) in ASCENDING edge index -- the fixed order in which sum_in e is accumulated, so that S4 gives the same
 * bits run to run; out_rowptr [n+1]: the out-edges of v are the edge range [out_rowptr[v], out_rowptr[v+1]).  n >= 1. */
trk_status trk_stage_gnn_csr(trk_ctx* ctx, const float* hits, int64_t n, const int32_t* src, const int32_t* dst,
                             int64_t n_edges, int32_t* in_rowptr, int32_t* in_perm, int32_t* out_rowptr, void* cuda_stream);
/* S5: labels int32 [n]; edges with score > cut are kept. */
trk_status trk_stage_cc(trk_ctx* ctx, int64_t n, const int32_t* src, const int32_t* dst, const float* score,
                        int64_t n_edges, float cut, int32_t* labels, void* cuda_stream);

/* S5 without a context and without any allocation (csrc/cc_noalloc.cu).
 * For callers that may not allocate device memory: a backend that lives inside a memory budget fixed by the serving
 * framework that owns the GPU, code running where cudaMalloc is forbidden or would stall the
 * device (while a stream capture is open elsewhere in the process, inside a stream host callback), and loops that cannot
 * afford the implicit synchronisation of cudaMalloc / cudaFree.  trk_create allocates the whole workspace, so none of
 * the ctx entry points is usable there; this one computes the same labels as trk_stage_cc (label = smallest hit index of
 * the component, edges with score > cut kept) with the union-find parent array in a fixed array inside the library image.
 *   - runs on the caller's CURRENT device; src/dst/score [n_edges] and labels [n] are DEVICE memory of that device and
 *     stay caller-owned; only kernels are enqueued on cuda_stream (no cudaMalloc, cudaFree, memset, sync or library call).
 *   - limit: n <= TRK_CC_NOALLOC_MAX_HITS.  A larger n is refused with TRK_ERR_CAPACITY before anything is enqueued
 *     (text in trk_last_error(NULL)).  The array costs TRK_CC_NOALLOC_MAX_HITS x 4 bytes = 4 MiB on every GPU that
 *     loads libtrk.so, used or not, until the process exits.
 *   - the first call on a device looks up the device address of that array (cudaGetSymbolAddress, which may also make
 *     the runtime load the module): make that first call before starting any stream capture.
 *   - all calls on a device share the one array, and it keeps what the previous call left there; each call re-initialises
 *     the n entries it uses, so results never depend on earlier calls -- but two calls that overlap on the same GPU
 *     (different streams or threads) race on it.  Order them on one stream or with events.                            */
#define TRK_CC_NOALLOC_MAX_HITS 1048576
trk_status trk_cc_noalloc(int64_t n, const int32_t* src, const int32_t* dst, const float* score, int64_t n_edges,
                          float cut, int32_t* labels, void* cuda_stream);

/* S6: track lists from labels [n] (as S5 writes them: label = smallest hit index of the component).
 * track_offsets [capacity+1], track_hits [n], track_counts [3] = {T, hits in tracks, overflow}.    */
trk_status trk_stage_tracks(trk_ctx* ctx, const int32_t* labels, int64_t n, int32_t min_hits, int32_t* track_offsets,
                            int64_t capacity, int32_t* track_hits, int32_t* track_counts, void* cuda_stream);

/* Kernel hook for tests/bench: out = act(A W^T + bias) through the ctx-independent tcgen05 GEMM on the caller's current
 * device.  A DEVICE bf16 [m][k] (k % 64 == 0), W DEVICE bf16 [n][k] (n % 64 == 0), bias DEVICE fp32 [n], out DEVICE bf16
 * [m][n]; relu != 0 applies ReLU; pair = 1: CTA-pair kernel (tcgen05.mma.cta_group::2, 256-row tiles) when the shape
 * allows it (n % 128 == 0 and k >= 256), pair = 0: single-CTA 128-row tiles.  Thread safe (no shared state). */
trk_status trk_gemm_bf16(const void* a, const void* w, const float* bias, void* out, int64_t m, int32_t n,
                         int32_t k, int32_t relu, int32_t pair, void* cuda_stream);

/* TEST / TUNING hook, per context: selects between kernel variants that compute the same result (each is parity-tested,
 * tests/test_gpu_stages.py, tests/test_gpu_gemm.py).  Not part of the served path; call it only while no trk_* call on
 * this ctx is running.
 *   "gemm_pair"       1 (default): dense layers with >= 128 output columns and K >= 256 run on CTA pairs
 *                     (tcgen05.mma.cta_group::2, 256-row tiles); 0: single-CTA 128-row tiles.
 *   "gnn_fused"       1 (default): with gnn_hidden == 128 the S4 encoders, edge update, node update and decoder run as
 *                     fused two-layer CTA-pair kernels (gnn_fused.cuh); 0: layer-by-layer GEMM launches with the exact
 *                     split first layer.
 *   "filter_fused"    1 (default): when the filter MLP is 2u -> W -> W -> W -> 1 with 2u <= 32 and W a multiple of 256 (<= 1024) S3
 *                     runs as ONE persistent CTA-pair kernel with L2-resident activations (filter_fused.cuh); 0: layer by layer,
 *                     one GEMM launch per layer over passes of trk_config.filter_chunk_rows edges.
 *   "epi_split"       (layer-by-layer S3 only) 1 (default): bf16-output layers with 256-column tiles and a single 64-wide K block (the first layer
 *                     of the S3 filter MLP) run their epilogue on eight warps (two per TMEM lane quadrant); 2: in addition
 *                     that layer's input rows [e_src ; e_dst] are gathered inside the GEMM kernel instead of by a separate
 *                     launch (measured slower on the pileup-200 event, so not the default); 0: four warps.
 *   "filter_max_pairs" 0 (default): the fused S3 kernel runs one CTA pair per two SMs; v > 0: at most v pairs, which leaves SMs
 *                     free for the other stages of another model instance on another stream (bench.py --scan).  Same scores.
 *   "gemm_row_major"  16 (default): a CTA pair of the pair GEMM walks all column tiles of one row block before the next
 *                     row block when there are at least 16 row blocks per pair (A rows re-read from L2, no DRAM
 *                     re-reads); 0: tiles in pair strides, column fastest.
 * Returns TRK_ERR_INVALID_ARG for an unknown key. */
trk_status trk_set_option(trk_ctx* ctx, const char* key, int64_t value);

#ifdef __cplusplus
}
#endif
#endif /* TRK_H_ */

// Shared declarations of the trk library (CUDA path).  No code here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "trk.h"

namespace trk {

constexpr int kMaxEmbDim = 16;      // d_e is padded to a multiple of 4, at most 16
constexpr int kMaxEvents = 1024;    // event offsets travel as a kernel parameter
constexpr int kPhiBins = 1024;           // S4: nodes are visited by phi bin in the segmented sums (graph.cu)
constexpr int kRBuckets = 16;            // FRNN: radius buckets inside a spatial cell (a tracking detector has ~10 layers)
constexpr int64_t kMaxCells = 1 << 22;  // FRNN cell-table entries (spatial cells x radius buckets) summed over the events of a call
constexpr int kFilterChunkTilesPerSm = 64;  // default S3 rows per pass = 128 x sm_count x 64 (trk_config.filter_chunk_rows overrides):
                                            // 2.5 GB per activation buffer buys 5 launches per 1.2 M candidate edges

// ---- test / tuning options (trk_set_option), per context ----
enum { kKnobGemmPair = 0, kKnobGnnFused = 1, kKnobEpiSplit = 2, kKnobRowMajor = 3, kKnobFilterFused = 4, kKnobFilterPairs = 5, kKnobCount = 6 };

// One Linear layer resident on the device.
struct DevLinear {
  int in = 0, out = 0;
  float* w_f32 = nullptr;           // [out][in]
  float* b_f32 = nullptr;           // [out]
  std::vector<float> b_host;        // the same on the host, zero padded to out_pad (small layers pass it as a kernel parameter)
  __nv_bfloat16* w_bf16 = nullptr;  // [out_pad][in_pad] K-major, zero padded (bf16 mode only)
  int in_pad = 0, out_pad = 0;
};

struct DevMlp {
  std::vector<DevLinear> layers;
};

// Device-side FRNN grid parameters (written by a 1-thread kernel, read by the others).
struct GridParams {
  float origin[3];
  float inv_cell[3];
  int dims[3];
  int cells_per_event;        // spatial cells of one event (the cell table has kRBuckets entries per spatial cell)
  float proj_eps;             // rounding slack of the fp32 projection, scaled with max|e| (frnn_grid_setup_kernel)
  float r_origin, r_inv;      // radius bucket = clamp(floor((r - r_origin) * r_inv), 0, kRBuckets - 1)
};

struct EventOffsets {
  int32_t v[kMaxEvents + 1];
};

struct Workspace {
  char* base = nullptr;
  size_t bytes = 0;
};

}  // namespace trk

struct trk_ctx {
  trk_config cfg;                   // scalar hyperparameters (pointers inside are not kept)
  int device = 0;
  int sm_count = 148;
  int d_e = 0, d_e_pad = 0;         // embedding width and its padding to a multiple of 4
  int filter_u = 0;                 // width of one endpoint's filter input
  int H = 0;
  cudaStream_t own_stream = nullptr;
  std::string last_error;
  int64_t launch_count = 0;
  int64_t knobs[trk::kKnobCount] = {1, 1, 1, 16, 1, 0};   // gemm_pair, gnn_fused, epi_split, gemm_row_major, filter_fused, filter_max_pairs (trk_set_option)
  std::vector<const void*> smem_attr_set;          // kernels whose dynamic shared-memory limit has been raised on ctx->device
  bool profiling = false;
  cudaEvent_t prof_ev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  bool prof_valid = false;
  // per-launch timing of the dominant kernel (the K >= 256 hidden-layer GEMMs of S3): event pairs, in launch order
  std::vector<cudaEvent_t> kprof_ev;
  int kprof_n = 0;                  // launches recorded by the last profiled trk_infer

  trk::DevMlp embed, filter, node_enc, edge_enc, edge_net, node_net, edge_dec;
  float* grid_proj = nullptr;       // [d_e_pad][3] device
  int grid_dims = 3;
  int grid_max = 32;                // upper bound of cells per axis and event (128 .. 8 by max_events)

  // stacked bf16 weights of the split first layers (bf16 mode): [2H][H] = [W1[:, :H] ; W1[:, H:2H]]
  __nv_bfloat16* edge_net_wab = nullptr;
  __nv_bfloat16* edge_net_wc = nullptr;    // [H][H] = W1[:, 2H:3H]
  __nv_bfloat16* edge_dec_wab = nullptr;
  __nv_bfloat16* edge_dec_wc = nullptr;
  __nv_bfloat16* filter_w1_pad = nullptr;  // [1024][64] = W1 zero padded in K
  // fused S3 kernel (filter_fused.cuh): the per-pair activation scratch
  bool filter_fusable = false;             // filter = 2u -> W -> W -> W -> 1, 2u <= 32, W a multiple of 256, W <= 1024
  __nv_bfloat16* filter_s1 = nullptr;      // [sm_count/2 * 256][W]  act1
  __nv_bfloat16* filter_s2 = nullptr;      // [sm_count/2 * 256][W]  act2
  // first layers of the S4 encoders for the tensor core (gnn_fused.cuh kEncode): [H][64], columns (2k, 2k+1) = w[:, k] twice
  __nv_bfloat16* node_enc_w1p = nullptr;
  __nv_bfloat16* edge_enc_w1p = nullptr;
  float filter_b_last = 0.f;               // bias of the filter's final Linear(W -> 1)
  float edge_dec_b_last = 0.f;             // bias of the decoder's final Linear(H -> 1)

  trk::Workspace ws;
  // ---- workspace carve-up (device pointers into ws.base) ----
  int32_t* ev_of_hit = nullptr;     // [max_hits] event id per hit
  float* emb = nullptr;             // [max_hits][d_e]
  // S1 / S3 activations
  void* act0 = nullptr;             // bf16 or fp32 [rows][width]
  void* act1 = nullptr;
  void* act_in = nullptr;           // S3 gathered input rows
  float* partial = nullptr;         // [chunk][4] fused last-layer partial dots
  int64_t act_rows = 0;
  int64_t filter_chunk = 0;         // S3 rows per pass: min(kFilterChunkRows, max_cand_edges rounded up to 128)
  // S2
  float* proj = nullptr;            // [max_hits][3]
  int32_t* bbox = nullptr;          // [16]: ordered-int min/max of the three binning coordinates [0..6), of the radius feature [6..8), bits of max|e| [8]
  trk::GridParams* grid = nullptr;
  int32_t* cell_of_hit = nullptr;   // [max_hits]
  int32_t* cell_count = nullptr;    // [max_cells+1]
  int32_t* cell_start = nullptr;    // [max_cells+1]
  int32_t* cell_fill = nullptr;     // [max_cells]
  float* semb = nullptr;            // [max_hits][d_e_pad] sorted by cell
  float4* smeta = nullptr;          // [max_hits] (r, |z|, idx bits, cell bits)
  float4* sproj = nullptr;          // [max_hits] binning coordinates P^T e, sorted by cell
  float proj_gain = 1.f;            // >= largest eigenvalue of P^T P (Gershgorin), 1 without a projection
  int32_t* slots = nullptr;         // [max_hits][K]
  int32_t* deg = nullptr;           // [max_hits+1]
  int32_t* rowptr = nullptr;        // [max_hits+1]
  int32_t* scan_tmp = nullptr;      // block sums for scans
  int64_t max_cells = 0;
  // edges
  int32_t* cand_src = nullptr;      // [max_cand_edges]
  int32_t* cand_dst = nullptr;
  float* cand_score = nullptr;
  int32_t* kept_src = nullptr;      // [max_kept_edges]
  int32_t* kept_dst = nullptr;
  float* kept_score = nullptr;
  int32_t* counts = nullptr;        // [8] device: {E_c, E_k, E_t, overflow, ...}
  int32_t* flag_scan = nullptr;     // [max_cand_edges] compaction offsets
  // S4
  void* X = nullptr;                // [max_hits][3H]  (h | m_in | m_out)  bf16 or fp32
  void* E = nullptr;                // [max_kept_edges][H]
  void* T1 = nullptr;               // [max(max_hits,max_kept_edges)][H]
  float* PAB = nullptr;             // [max_hits][2H] fp32 per-node halves of the split first layer
  float* cat = nullptr;             // fp32 mode: [max(E,N)][3H]
  int32_t* in_rowptr = nullptr;     // [max_hits+1] CSR by dst
  int32_t* in_perm = nullptr;       // [max_kept_edges]
  int32_t* in_fill = nullptr;       // [max_hits]
  int32_t* out_rowptr = nullptr;    // [max_hits+1] CSR by src (edges are src-sorted)
  int32_t* node_order = nullptr;    // [max_hits] the nodes by phi bin: the order in which the segmented sums visit them (graph.cu)
  int32_t* phi_bins = nullptr;      // [2 * (kPhiBins + 1)] counts / starts of the phi bins
  int4* seg_tasks = nullptr;        // [2 max_hits] (node, first entry, end entry, direction) of the segmented sums, in visiting order
  // S5
  int32_t* parent = nullptr;        // [max_hits]
  // S6 (tracks.cu): sizes / flags / scans and the (key, value) ping-pong of the radix sort, [max_hits+2] each
  int32_t *tk_a = nullptr, *tk_b = nullptr, *tk_c = nullptr, *tk_d = nullptr, *tk_e = nullptr, *tk_f = nullptr, *tk_g = nullptr;
  int32_t* tk_hist = nullptr;       // [256 * ceil(max_hits/256) + 2] digit-major block histograms
  int32_t* tk_hist_scan = nullptr;
  // trk_infer_host staging (device side)
  float* io_hits = nullptr;         // [max_hits][3]
  int32_t* io_labels = nullptr;     // [max_hits]
  int32_t* io_counts = nullptr;     // [8]: counts[4], then {n_tracks, n_track_hits}
  int32_t* io_track_offsets = nullptr;  // [max_hits+1]
  int32_t* io_track_hits = nullptr;     // [max_hits]
};

namespace trk {

// ---- error plumbing ----
trk_status fail(trk_ctx* ctx, trk_status s, const std::string& msg);
#define TRK_CUDA(ctx, expr)                                                                   \
  do {                                                                                        \
    cudaError_t _e = (expr);                                                                  \
    if (_e != cudaSuccess)                                                                    \
      return ::trk::fail((ctx), TRK_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(_e)); \
  } while (0)
#define TRK_TRY(expr)                   \
  do {                                  \
    trk_status _s = (expr);             \
    if (_s != TRK_OK) return _s;        \
  } while (0)

// Every kernel launch of the library goes through this so that launches can be counted.
// Every kernel is launched with programmatic stream serialization and starts with griddepcontrol.wait: the launch of a kernel
// (grid set-up, block scheduling) overlaps the drain of the kernel before it in the stream, its first instruction still waits
// for that kernel's completion and memory flush.  No kernel triggers its dependents early (griddepcontrol.launch_dependents at the
// top of every kernel was measured slower: S2 0.49 -> 0.51 ms, S4 2.01 -> 2.07 ms).  Measured: S2 0.52 -> 0.49, S4 2.09 -> 2.01 ms.
#define TRK_GRID_DEP_WAIT() asm volatile("griddepcontrol.wait;" ::: "memory")
#define TRK_LAUNCH(ctx, kernel, grid_, block_, smem_, strm_, ...)                 \
  do {                                                                           \
    cudaLaunchConfig_t _cfg = {};                                                \
    _cfg.gridDim = dim3(grid_);                                                  \
    _cfg.blockDim = dim3(block_);                                                \
    _cfg.dynamicSmemBytes = (size_t)(smem_);                                     \
    _cfg.stream = (strm_);                                                      \
    cudaLaunchAttribute _attr[1];                                                \
    _attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;            \
    _attr[0].val.programmaticStreamSerializationAllowed = 1;                     \
    _cfg.attrs = _attr;                                                          \
    _cfg.numAttrs = 1;                                                           \
    cudaLaunchKernelEx(&_cfg, kernel, __VA_ARGS__);                              \
    (ctx)->launch_count++;                                                       \
    cudaError_t _e = cudaPeekAtLastError();                                      \
    if (_e != cudaSuccess)                                                       \
      return ::trk::fail((ctx), TRK_ERR_CUDA, std::string(#kernel) + ": " + cudaGetErrorString(_e)); \
  } while (0)

inline int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute of a kernel: it is raised once per context (a context
// is bound to one device; the caller's current device is ctx->device inside every entry point, see DeviceGuard in api.cu).
template <class Kernel>
inline trk_status ensure_smem(trk_ctx* ctx, Kernel kern, int bytes) {
  const void* key = reinterpret_cast<const void*>(kern);
  for (const void* k : ctx->smem_attr_set)
    if (k == key) return TRK_OK;
  TRK_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  ctx->smem_attr_set.push_back(key);
  return TRK_OK;
}

// ---- util_kernels.cu ----
trk_status exclusive_scan_i32(trk_ctx* ctx, const int32_t* in, int32_t* out, int64_t n, int32_t* tmp, cudaStream_t st);
trk_status fill_i32(trk_ctx* ctx, int32_t* p, int32_t v, int64_t n, cudaStream_t st);
trk_status compact_edges(trk_ctx* ctx, const int32_t* src, const int32_t* dst, const float* score, const int32_t* n_dev,
                         int64_t n_cap, float cut, int32_t* out_src, int32_t* out_dst, int64_t out_cap, int32_t* count_out,
                         int32_t* overflow_flag, cudaStream_t st);

// ---- frnn.cu ----
trk_status frnn_build(trk_ctx* ctx, const float* emb, const float* hits, int64_t n, int32_t n_events, int32_t* src,
                      int32_t* dst, int32_t* rowptr_out, int64_t capacity, int32_t* count_out, int32_t* overflow_flag,
                      cudaStream_t st);

trk_status set_event_ids(trk_ctx* ctx, const int32_t* offsets_host, int n_events, int64_t n, cudaStream_t st);

// ---- cc.cu ----
trk_status cc_labels(trk_ctx* ctx, int64_t n, const int32_t* src, const int32_t* dst, const float* score,
                     const int32_t* n_edges_dev, int64_t n_edges_cap, float cut, int32_t* labels, int32_t* pass_count,
                     cudaStream_t st);

// ---- tracks.cu ----
// track_offsets [capacity+1], track_hits [n] (entries beyond the last track are -1), track_counts [2] = {T, hits in tracks}
trk_status build_tracks(trk_ctx* ctx, const int32_t* labels, int64_t n, int min_hits, int32_t* track_offsets, int64_t capacity,
                        int32_t* track_hits, int32_t* track_counts, int32_t* overflow_flag, cudaStream_t st);

}  // namespace trk

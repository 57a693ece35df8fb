// C ABI of the trk library (include/trk.h): context lifecycle, workspace planning, the five-stage
// pipeline of PAPER.md line 85 and the per-stage hooks.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>

#include "common.cuh"
#include "graph.cuh"
#include "nn.cuh"

namespace trk {

static std::string g_create_error;
static std::mutex g_create_mutex;

trk_status fail(trk_ctx* ctx, trk_status s, const std::string& msg) {
  if (ctx) {
    ctx->last_error = msg;
  } else {
    std::lock_guard<std::mutex> lk(g_create_mutex);
    g_create_error = msg;
  }
  return s;
}

trk_status gemm_bf16_hook(trk_ctx* ctx, const void* a, const void* w, const float* bias, void* out, int64_t m, int n, int k, int relu,
                          cudaStream_t st);

namespace {

// Every entry point that touches the device runs with ctx->device current and restores the caller's device on return
// (a process may hold contexts on several GPUs: include/trk.h "device").
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};

int round_up(int v, int m) { return (v + m - 1) / m * m; }

bool mlp_ok(const trk_mlp& m, int n_layers_min) {
  if (m.n_layers < n_layers_min || !m.dims || !m.weight || !m.bias) return false;
  for (int l = 0; l <= m.n_layers; ++l)
    if (m.dims[l] <= 0) return false;
  for (int l = 0; l < m.n_layers; ++l)
    if (!m.weight[l] || !m.bias[l]) return false;
  return true;
}

uint16_t f32_to_bf16_rne(float f) {
  uint32_t u;
  std::memcpy(&u, &f, 4);
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x40);  // NaN
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

// Uploads fp32 weights/biases; in bf16 mode also a zero padded bf16 copy [out_pad][in_pad].
trk_status upload_mlp(trk_ctx* ctx, const trk_mlp& m, DevMlp* out, bool bf16) {
  out->layers.resize(m.n_layers);
  for (int l = 0; l < m.n_layers; ++l) {
    DevLinear& L = out->layers[l];
    L.in = m.dims[l];
    L.out = m.dims[l + 1];
    L.in_pad = round_up(L.in, 64);
    L.out_pad = L.out <= 16 ? 16 : round_up(L.out, 64);
    const size_t nw = (size_t)L.in * L.out;
    TRK_CUDA(ctx, cudaMalloc(&L.w_f32, nw * 4));
    TRK_CUDA(ctx, cudaMalloc(&L.b_f32, (size_t)L.out_pad * 4));
    TRK_CUDA(ctx, cudaMemcpy(L.w_f32, m.weight[l], nw * 4, cudaMemcpyHostToDevice));
    std::vector<float> b(L.out_pad, 0.f);
    std::memcpy(b.data(), m.bias[l], (size_t)L.out * 4);
    TRK_CUDA(ctx, cudaMemcpy(L.b_f32, b.data(), (size_t)L.out_pad * 4, cudaMemcpyHostToDevice));
    L.b_host = b;
    if (bf16) {
      std::vector<uint16_t> w((size_t)L.in_pad * L.out_pad, 0);
      for (int o = 0; o < L.out; ++o)
        for (int i = 0; i < L.in; ++i) w[(size_t)o * L.in_pad + i] = f32_to_bf16_rne(m.weight[l][(size_t)o * L.in + i]);
      TRK_CUDA(ctx, cudaMalloc(&L.w_bf16, w.size() * 2));
      TRK_CUDA(ctx, cudaMemcpy(L.w_bf16, w.data(), w.size() * 2, cudaMemcpyHostToDevice));
    }
  }
  return TRK_OK;
}

// bf16 [rows][cols] built from columns [c0, c0+cols) of a host fp32 [rows][ld] matrix, stacked pieces allowed.
trk_status upload_bf16_block(trk_ctx* ctx, const std::vector<uint16_t>& host, __nv_bfloat16** dev) {
  TRK_CUDA(ctx, cudaMalloc(dev, host.size() * 2));
  TRK_CUDA(ctx, cudaMemcpy(*dev, host.data(), host.size() * 2, cudaMemcpyHostToDevice));
  return TRK_OK;
}

void free_mlp(DevMlp& m) {
  for (auto& L : m.layers) {
    cudaFree(L.w_f32);
    cudaFree(L.b_f32);
    cudaFree(L.w_bf16);
  }
  m.layers.clear();
}

struct Carver {
  size_t off = 0;
  char* base = nullptr;
  template <typename T>
  void take(T** p, size_t count) {
    off = (off + 1023) & ~(size_t)1023;
    if (base) *p = reinterpret_cast<T*>(base + off);
    off += count * sizeof(T);
  }
};

// One pass computes the size (base == nullptr), a second assigns the pointers.
void carve(trk_ctx* c, Carver& k) {
  const trk_config& f = c->cfg;
  const bool bf = f.precision == TRK_BF16;
  const size_t N = (size_t)f.max_hits, EC = (size_t)f.max_cand_edges, EK = (size_t)f.max_kept_edges;
  const size_t es = bf ? 2 : 4;
  const int H = c->H;
  const size_t f_w1 = c->filter.layers.empty() ? 0 : (size_t)c->filter.layers[0].out_pad;
  int maxw = 64;
  for (auto& L : c->embed.layers) maxw = std::max(maxw, L.out_pad);
  for (auto& L : c->filter.layers) maxw = std::max(maxw, L.out_pad);
  {
    // layer-by-layer S3: rows per pass.  With the fused S3 kernel (the default when the shape allows it) the chunked path only
    // serves as a test variant, so its buffers stay small unless the caller sizes them.
    int64_t chunk = (int64_t)128 * c->sm_count * (c->filter_fusable ? 1 : kFilterChunkTilesPerSm);
    if (f.filter_chunk_rows > 0) chunk = (f.filter_chunk_rows + 127) / 128 * 128;
    c->filter_chunk = std::min<int64_t>(chunk, ((int64_t)EC + 127) / 128 * 128);
  }
  c->act_rows = (int64_t)std::max<size_t>(N, (size_t)c->filter_chunk);
  char* p = nullptr;
  k.take(&c->ev_of_hit, N);
  k.take(&c->emb, N * c->d_e);
  k.take(&p, (size_t)c->act_rows * maxw * es); c->act0 = p;
  k.take(&p, (size_t)c->act_rows * maxw * es); c->act1 = p;
  k.take(&p, (size_t)c->filter_chunk * (bf ? 64 * 2 : 2 * c->filter_u * 4)); c->act_in = p;
  k.take(&c->partial, (size_t)c->filter_chunk * 16);
  if (c->filter_fusable) {
    const size_t rows = (size_t)(c->sm_count / 2) * 256;
    k.take(&c->filter_s1, rows * f_w1);
    k.take(&c->filter_s2, rows * f_w1);
  }
  k.take(&c->proj, N * 3);
  k.take(&c->bbox, 16);
  k.take(&c->grid, 1);
  k.take(&c->cell_of_hit, N);
  k.take(&c->cell_count, (size_t)c->max_cells + 1);
  k.take(&c->cell_start, (size_t)c->max_cells + 1);
  k.take(&c->cell_fill, (size_t)c->max_cells + 1);
  k.take(&c->semb, N * c->d_e_pad);
  k.take(&c->smeta, N);
  k.take(&c->sproj, N);
  k.take(&c->slots, N * f.frnn_k);
  k.take(&c->deg, N + 2);
  k.take(&c->rowptr, N + 2);
  const size_t scan_n = std::max(std::max(EC, (size_t)c->max_cells + 1), std::max(N + 1024, EK));
  k.take(&c->scan_tmp, scan_n / 2048 + 4);
  k.take(&c->cand_src, EC);
  k.take(&c->cand_dst, EC);
  k.take(&c->cand_score, EC);
  k.take(&c->kept_src, EK);
  k.take(&c->kept_dst, EK);
  k.take(&c->kept_score, EK);
  k.take(&c->counts, 8);
  const size_t R = std::max(N, EK);
  k.take(&p, N * 3 * H * es); c->X = p;
  k.take(&p, EK * H * es); c->E = p;
  k.take(&p, R * H * (bf ? 2 : 8)); c->T1 = p;
  if (bf) k.take(&c->PAB, N * 2 * H);
  else k.take(&c->cat, R * 3 * H);
  k.take(&c->in_rowptr, N + 2);
  k.take(&c->in_perm, EK);
  k.take(&c->in_fill, N + 2);
  k.take(&c->out_rowptr, N + 2);
  k.take(&c->node_order, N);
  k.take(&c->phi_bins, 2 * (kPhiBins + 1));
  k.take(&c->seg_tasks, 2 * N);
  k.take(&c->parent, N);
  for (int32_t** t : {&c->tk_a, &c->tk_b, &c->tk_c, &c->tk_d, &c->tk_e, &c->tk_f, &c->tk_g}) k.take(t, N + 2);
  k.take(&c->tk_hist, (N + 255) / 256 * 256 + 2);
  k.take(&c->tk_hist_scan, (N + 255) / 256 * 256 + 2);
  k.take(&c->io_hits, N * 3);
  k.take(&c->io_labels, N);
  k.take(&c->io_counts, 8);
  k.take(&c->io_track_offsets, N + 1);
  k.take(&c->io_track_hits, N);
}

__global__ void finalize_counts_kernel(const int32_t* __restrict__ counts, int64_t edge_cap, int64_t cand_cap, int32_t* __restrict__ out) {
  TRK_GRID_DEP_WAIT();
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  int of = counts[3];
  if (edge_cap >= 0 && counts[1] > edge_cap) of = 1;
  if (cand_cap >= 0 && counts[0] > cand_cap) of = 1;
  out[0] = counts[0];
  out[1] = counts[1];
  out[2] = counts[2];
  out[3] = of;
}

__global__ void zero_counts_kernel(int32_t* counts) {
  TRK_GRID_DEP_WAIT();
  if (threadIdx.x < 8) counts[threadIdx.x] = 0;
}

trk_status check_batch(trk_ctx* ctx, int32_t n_events, const int32_t* off, int64_t* n_out) {
  if (n_events < 0 || !off) return fail(ctx, TRK_ERR_INVALID_ARG, "event_offsets is NULL or n_events < 0");
  if (n_events > ctx->cfg.max_events || n_events > kMaxEvents) return fail(ctx, TRK_ERR_CAPACITY, "n_events exceeds max_events");
  if (off[0] != 0) return fail(ctx, TRK_ERR_INVALID_ARG, "event_offsets[0] must be 0");
  for (int i = 0; i < n_events; ++i)
    if (off[i + 1] < off[i]) return fail(ctx, TRK_ERR_INVALID_ARG, "event_offsets must be non-decreasing");
  const int64_t n = n_events > 0 ? off[n_events] : 0;
  if (n > ctx->cfg.max_hits) return fail(ctx, TRK_ERR_CAPACITY, "number of hits exceeds max_hits");
  *n_out = n;
  return TRK_OK;
}

trk_status embed_dispatch(trk_ctx* ctx, const float* hits, int64_t n, float* emb, cudaStream_t st) {
  if (n <= 0) return TRK_OK;
  return ctx->cfg.precision == TRK_BF16 ? embed_forward_bf16(ctx, hits, n, emb, st) : embed_forward_fp32(ctx, hits, n, emb, st);
}
trk_status filter_dispatch(trk_ctx* ctx, const float* feat, const int32_t* src, const int32_t* dst, const int32_t* n_dev, int64_t cap,
                           float* score, cudaStream_t st) {
  if (cap <= 0) return TRK_OK;
  return ctx->cfg.precision == TRK_BF16 ? filter_forward_bf16(ctx, feat, src, dst, n_dev, cap, score, st)
                                        : filter_forward_fp32(ctx, feat, src, dst, n_dev, cap, score, st);
}
trk_status gnn_dispatch(trk_ctx* ctx, const float* hits, int64_t n, const int32_t* src, const int32_t* dst, const int32_t* n_dev,
                        int64_t cap, float* score, cudaStream_t st) {
  if (n <= 0) return TRK_OK;
  return ctx->cfg.precision == TRK_BF16 ? gnn_forward_bf16(ctx, hits, n, src, dst, n_dev, cap, score, st)
                                        : gnn_forward_fp32(ctx, hits, n, src, dst, n_dev, cap, score, st);
}

}  // namespace
}  // namespace trk

using namespace trk;

extern "C" {

const char* trk_status_string(trk_status s) {
  switch (s) {
    case TRK_OK: return "TRK_OK";
    case TRK_ERR_INVALID_ARG: return "TRK_ERR_INVALID_ARG";
    case TRK_ERR_SHAPE: return "TRK_ERR_SHAPE";
    case TRK_ERR_CAPACITY: return "TRK_ERR_CAPACITY";
    case TRK_ERR_CUDA: return "TRK_ERR_CUDA";
    case TRK_ERR_OOM: return "TRK_ERR_OOM";
    case TRK_ERR_UNSUPPORTED_DEVICE: return "TRK_ERR_UNSUPPORTED_DEVICE";
  }
  return "TRK_ERR_UNKNOWN";
}

const char* trk_last_error(const trk_ctx* ctx) {
  if (ctx) return ctx->last_error.c_str();
  // the create-time message is copied under the lock into a per-thread buffer: a concurrent failing trk_create may
  // reallocate the shared string
  static thread_local std::string copy;
  std::lock_guard<std::mutex> lk(g_create_mutex);
  copy = g_create_error;
  return copy.c_str();
}
int64_t trk_workspace_bytes(const trk_ctx* ctx) { return ctx ? (int64_t)ctx->ws.bytes : 0; }
int64_t trk_last_launch_count(const trk_ctx* ctx) { return ctx ? ctx->launch_count : 0; }

trk_status trk_destroy(trk_ctx* ctx) {
  if (!ctx) return TRK_OK;
  DeviceGuard guard(ctx->device);
  if (ctx->own_stream) {
    cudaStreamSynchronize(ctx->own_stream);
    cudaStreamDestroy(ctx->own_stream);
  }
  cudaDeviceSynchronize();
  for (auto& e : ctx->prof_ev)
    if (e) cudaEventDestroy(e);
  for (auto& e : ctx->kprof_ev) cudaEventDestroy(e);
  for (DevMlp* m : {&ctx->embed, &ctx->filter, &ctx->node_enc, &ctx->edge_enc, &ctx->edge_net, &ctx->node_net, &ctx->edge_dec}) free_mlp(*m);
  cudaFree(ctx->grid_proj);
  cudaFree(ctx->edge_net_wab);
  cudaFree(ctx->edge_net_wc);
  cudaFree(ctx->edge_dec_wab);
  cudaFree(ctx->edge_dec_wc);
  cudaFree(ctx->filter_w1_pad);
  cudaFree(ctx->node_enc_w1p);
  cudaFree(ctx->edge_enc_w1p);
  cudaFree(ctx->ws.base);
  delete ctx;
  return TRK_OK;
}

trk_status trk_create(const trk_config* cfg, trk_ctx** out) {
  if (!cfg || !out) return fail(nullptr, TRK_ERR_INVALID_ARG, "cfg or out is NULL");
  *out = nullptr;
  if (cfg->struct_size != sizeof(trk_config)) return fail(nullptr, TRK_ERR_INVALID_ARG, "trk_config.struct_size mismatch");
  if (cfg->precision != TRK_FP32 && cfg->precision != TRK_BF16) return fail(nullptr, TRK_ERR_INVALID_ARG, "bad precision");
  if (cfg->filter_input != TRK_FILTER_RAW && cfg->filter_input != TRK_FILTER_EMB) return fail(nullptr, TRK_ERR_INVALID_ARG, "bad filter_input");
  if (cfg->max_hits <= 0 || cfg->max_events <= 0 || cfg->max_cand_edges <= 0 || cfg->max_kept_edges <= 0)
    return fail(nullptr, TRK_ERR_INVALID_ARG, "capacities must be positive");
  if (cfg->max_hits > (1ll << 30) || cfg->max_cand_edges > (1ll << 31) - 4096 || cfg->max_kept_edges > (1ll << 31) - 4096)
    return fail(nullptr, TRK_ERR_CAPACITY, "capacities exceed the int32 index range");
  if (cfg->max_events > kMaxEvents) return fail(nullptr, TRK_ERR_CAPACITY, "max_events > 1024");
  if (cfg->frnn_k < 1 || cfg->frnn_k > 128) return fail(nullptr, TRK_ERR_INVALID_ARG, "frnn_k must be in 1..128");
  // S2 scans per-hit degrees (<= frnn_k each) into int32 row offsets before the capacity clamp applies
  if (cfg->max_hits * (int64_t)cfg->frnn_k > (int64_t)INT32_MAX)
    return fail(nullptr, TRK_ERR_CAPACITY, "max_hits * frnn_k exceeds the int32 index range");
  if (cfg->filter_chunk_rows < 0 || cfg->grid_max < 0 || cfg->grid_max > 128)
    return fail(nullptr, TRK_ERR_INVALID_ARG, "filter_chunk_rows must be >= 0 and grid_max in 0..128");
  if (!(cfg->frnn_radius >= 0.f)) return fail(nullptr, TRK_ERR_INVALID_ARG, "frnn_radius must be >= 0");
  if (cfg->grid_dims < 1 || cfg->grid_dims > 3) return fail(nullptr, TRK_ERR_INVALID_ARG, "grid_dims must be 1..3");
  if (cfg->gnn_iters < 0 || cfg->gnn_hidden <= 0) return fail(nullptr, TRK_ERR_INVALID_ARG, "bad GNN hyperparameters");
  if (!mlp_ok(cfg->embed, 1) || !mlp_ok(cfg->filter, 1) || !mlp_ok(cfg->node_enc, 2) || !mlp_ok(cfg->edge_enc, 2) ||
      !mlp_ok(cfg->edge_net, 2) || !mlp_ok(cfg->node_net, 2) || !mlp_ok(cfg->edge_dec, 2))
    return fail(nullptr, TRK_ERR_INVALID_ARG, "an MLP description is incomplete");
  const int H = cfg->gnn_hidden;
  const int d_e = cfg->embed.dims[cfg->embed.n_layers];
  const int u = cfg->filter_input == TRK_FILTER_EMB ? d_e : 3;
  auto two = [&](const trk_mlp& m, int in, int outw) {
    return m.n_layers == 2 && m.dims[0] == in && m.dims[1] == H && m.dims[2] == outw;
  };
  if (cfg->embed.dims[0] != 3) return fail(nullptr, TRK_ERR_SHAPE, "embed.dims[0] must be 3");
  if (d_e < 1 || d_e > kMaxEmbDim) return fail(nullptr, TRK_ERR_SHAPE, "embedding width must be 1..16");
  if (cfg->grid_dims > d_e) return fail(nullptr, TRK_ERR_SHAPE, "grid_dims exceeds the embedding width");
  if (cfg->filter.dims[0] != 2 * u) return fail(nullptr, TRK_ERR_SHAPE, "filter.dims[0] must be twice the endpoint feature width");
  if (cfg->filter.dims[cfg->filter.n_layers] != 1) return fail(nullptr, TRK_ERR_SHAPE, "filter must end in one output");
  if (!two(cfg->node_enc, 3, H) || !two(cfg->edge_enc, 4, H) || !two(cfg->edge_net, 3 * H, H) || !two(cfg->node_net, 3 * H, H) ||
      !two(cfg->edge_dec, 3 * H, 1))
    return fail(nullptr, TRK_ERR_SHAPE, "GNN MLP dims must be {3,H,H} {4,H,H} {3H,H,H} {3H,H,H} {3H,H,1}");
  if (H % 4 != 0) return fail(nullptr, TRK_ERR_SHAPE, "gnn_hidden must be a multiple of 4");
  const bool bf = cfg->precision == TRK_BF16;
  if (bf) {
    if (H != 64 && H != 128) return fail(nullptr, TRK_ERR_SHAPE, "TRK_BF16 needs gnn_hidden 64 or 128");
    if (cfg->embed.n_layers < 2 || cfg->filter.n_layers < 2) return fail(nullptr, TRK_ERR_SHAPE, "TRK_BF16 needs >= 2 layers in embed and filter");
    for (int l = 1; l < cfg->embed.n_layers; ++l)
      if (cfg->embed.dims[l] % 64) return fail(nullptr, TRK_ERR_SHAPE, "TRK_BF16 needs hidden widths that are multiples of 64");
    for (int l = 1; l < cfg->filter.n_layers; ++l)
      if (cfg->filter.dims[l] % 64 || cfg->filter.dims[l] > 1024) return fail(nullptr, TRK_ERR_SHAPE, "TRK_BF16 filter widths: multiples of 64, <= 1024");
    if (2 * u > 64) return fail(nullptr, TRK_ERR_SHAPE, "TRK_BF16 needs a filter input of at most 64 values");
  }

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev)
    return fail(nullptr, TRK_ERR_CUDA, "no such CUDA device");
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess) return fail(nullptr, TRK_ERR_CUDA, "cudaGetDeviceProperties failed");
  if (prop.major != 10) return fail(nullptr, TRK_ERR_UNSUPPORTED_DEVICE, "this library is built for sm_100a (B200) only");
  DeviceGuard guard(cfg->device);
  {
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != cfg->device) return fail(nullptr, TRK_ERR_CUDA, "cudaSetDevice failed");
  }

  trk_ctx* ctx = new trk_ctx();
  ctx->cfg = *cfg;
  ctx->cfg.grid_proj = nullptr;
  ctx->device = cfg->device;
  ctx->sm_count = prop.multiProcessorCount;
  ctx->d_e = d_e;
  ctx->d_e_pad = round_up(d_e, 4);
  ctx->filter_u = u;
  ctx->H = H;
  ctx->grid_dims = cfg->grid_dims;
  // cells per axis and event: the finest grid whose cell table fits (the cell edge never goes below r, so a finer bound only
  // helps: candidates per query fall with the cell volume until the edge reaches r)
  ctx->grid_max = 1;
  for (int g = 128; g > 1; --g)
    if (cfg->max_events * (int64_t)g * g * g * kRBuckets <= kMaxCells) { ctx->grid_max = g; break; }
  if (cfg->grid_max > 0) ctx->grid_max = std::min(ctx->grid_max, cfg->grid_max);
  ctx->max_cells = (int64_t)cfg->max_events * ctx->grid_max * ctx->grid_max * ctx->grid_max * kRBuckets;

  trk_status s = TRK_OK;
  auto bail = [&](trk_status st) {
    { std::lock_guard<std::mutex> lk(g_create_mutex); g_create_error = ctx->last_error; }
    trk_destroy(ctx);
    return st;
  };
  struct { const trk_mlp* m; DevMlp* d; } mlps[] = {{&cfg->embed, &ctx->embed}, {&cfg->filter, &ctx->filter},
      {&cfg->node_enc, &ctx->node_enc}, {&cfg->edge_enc, &ctx->edge_enc}, {&cfg->edge_net, &ctx->edge_net},
      {&cfg->node_net, &ctx->node_net}, {&cfg->edge_dec, &ctx->edge_dec}};
  for (auto& e : mlps)
    if ((s = upload_mlp(ctx, *e.m, e.d, bf)) != TRK_OK) return bail(s);
  ctx->filter_b_last = cfg->filter.bias[cfg->filter.n_layers - 1][0];
  ctx->edge_dec_b_last = cfg->edge_dec.bias[1][0];
  if (cfg->grid_proj) {
    std::vector<float> P((size_t)ctx->d_e * 3, 0.f);
    for (int k = 0; k < d_e; ++k)
      for (int a = 0; a < cfg->grid_dims; ++a) P[k * 3 + a] = cfg->grid_proj[k * cfg->grid_dims + a];
    // shrink every column to norm <= 1 so the projection can never lengthen a distance
    for (int a = 0; a < cfg->grid_dims; ++a) {
      double nn = 0;
      for (int k = 0; k < d_e; ++k) nn += (double)P[k * 3 + a] * P[k * 3 + a];
      const double sc = nn > 0 ? std::min(1.0, 1.0 / std::sqrt(nn)) * (1.0 - 1e-6) : 0.0;
      for (int k = 0; k < d_e; ++k) P[k * 3 + a] = (float)(P[k * 3 + a] * sc);
    }
    // ||P^T v||^2 <= lambda ||v||^2 with lambda = largest eigenvalue of P^T P <= max absolute row sum (Gershgorin)
    double gain = 0.0;
    for (int a = 0; a < 3; ++a) {
      double rowsum = 0.0;
      for (int b = 0; b < 3; ++b) {
        double g = 0.0;
        for (int k = 0; k < d_e; ++k) g += (double)P[k * 3 + a] * P[k * 3 + b];
        rowsum += std::fabs(g);
      }
      gain = std::max(gain, rowsum);
    }
    ctx->proj_gain = (float)std::max(gain * (1.0 + 1e-6), 1e-12);
    if (cudaMalloc(&ctx->grid_proj, P.size() * 4) != cudaSuccess ||
        cudaMemcpy(ctx->grid_proj, P.data(), P.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess)
      return bail(fail(ctx, TRK_ERR_OOM, "grid_proj upload failed"));
  }
  if (bf) {
    // split first layers of edge_net / edge_dec: [Wa ; Wb] stacked [2H][H] and Wc [H][H]
    auto split = [&](const trk_mlp& m, __nv_bfloat16** wab, __nv_bfloat16** wc) -> trk_status {
      std::vector<uint16_t> ab((size_t)2 * H * H), c((size_t)H * H);
      const float* W = m.weight[0];  // [H][3H]
      for (int o = 0; o < H; ++o)
        for (int i = 0; i < H; ++i) {
          ab[(size_t)o * H + i] = f32_to_bf16_rne(W[(size_t)o * 3 * H + i]);
          ab[(size_t)(H + o) * H + i] = f32_to_bf16_rne(W[(size_t)o * 3 * H + H + i]);
          c[(size_t)o * H + i] = f32_to_bf16_rne(W[(size_t)o * 3 * H + 2 * H + i]);
        }
      TRK_TRY(upload_bf16_block(ctx, ab, wab));
      return upload_bf16_block(ctx, c, wc);
    };
    if ((s = split(cfg->edge_net, &ctx->edge_net_wab, &ctx->edge_net_wc)) != TRK_OK) return bail(s);
    if ((s = split(cfg->edge_dec, &ctx->edge_dec_wab, &ctx->edge_dec_wc)) != TRK_OK) return bail(s);
    // filter first layer with K zero padded to 64
    const int w1 = cfg->filter.dims[1], k1 = cfg->filter.dims[0];
    std::vector<uint16_t> p((size_t)round_up(w1, 64) * 64, 0);
    for (int o = 0; o < w1; ++o)
      for (int i = 0; i < k1; ++i) p[(size_t)o * 64 + i] = f32_to_bf16_rne(cfg->filter.weight[0][(size_t)o * k1 + i]);
    if ((s = upload_bf16_block(ctx, p, &ctx->filter_w1_pad)) != TRK_OK) return bail(s);
    // fused S3 kernel (filter_fused.cuh): applicable shape
    {
      const trk_mlp& m = cfg->filter;
      const int W = m.dims[1];
      ctx->filter_fusable = m.n_layers == 4 && k1 <= 32 && W % 256 == 0 && W <= 1024 && m.dims[2] == W && m.dims[3] == W;
    }
    // encoder first layers (K = 3 / 4) as a [H][64] bf16 K block: every weight column twice, once for the hi and once for the
    // lo half of its fp32 input feature (gnn_fused.cuh kEncode)
    auto dup = [&](const trk_mlp& m, __nv_bfloat16** out) -> trk_status {
      const int k = m.dims[0];
      std::vector<uint16_t> w((size_t)H * 64, 0);
      for (int o = 0; o < H; ++o)
        for (int i = 0; i < k; ++i) w[(size_t)o * 64 + 2 * i] = w[(size_t)o * 64 + 2 * i + 1] = f32_to_bf16_rne(m.weight[0][(size_t)o * k + i]);
      return upload_bf16_block(ctx, w, out);
    };
    if ((s = dup(cfg->node_enc, &ctx->node_enc_w1p)) != TRK_OK) return bail(s);
    if ((s = dup(cfg->edge_enc, &ctx->edge_enc_w1p)) != TRK_OK) return bail(s);
  }

  Carver size_pass;
  carve(ctx, size_pass);
  ctx->ws.bytes = size_pass.off + 1024;
  if (cudaMalloc(&ctx->ws.base, ctx->ws.bytes) != cudaSuccess) {
    cudaGetLastError();
    ctx->ws.base = nullptr;
    return bail(fail(ctx, TRK_ERR_OOM, "workspace allocation of " + std::to_string(ctx->ws.bytes) + " bytes failed"));
  }
  Carver assign;
  assign.base = ctx->ws.base;
  carve(ctx, assign);
  if (cudaMemset(ctx->ws.base, 0, ctx->ws.bytes) != cudaSuccess) return bail(fail(ctx, TRK_ERR_CUDA, "workspace memset failed"));
  if (cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking) != cudaSuccess)
    return bail(fail(ctx, TRK_ERR_CUDA, "stream creation failed"));
  if (cudaDeviceSynchronize() != cudaSuccess) return bail(fail(ctx, TRK_ERR_CUDA, "device synchronisation failed in trk_create"));
  *out = ctx;
  return TRK_OK;
}

trk_status trk_infer(trk_ctx* ctx, const trk_batch* batch, const trk_result* res, void* cuda_stream) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->device);
  ctx->launch_count = 0;   // counts the launches of THIS call: a call refused below leaves it at 0 (nothing enqueued)
  ctx->prof_valid = false;
  if (!batch || !res) return fail(ctx, TRK_ERR_INVALID_ARG, "batch or result is NULL");
  if (!res->counts) return fail(ctx, TRK_ERR_INVALID_ARG, "result.counts is required");
  int64_t n = 0;
  TRK_TRY(check_batch(ctx, batch->n_events, batch->event_offsets, &n));
  if (n > 0 && !res->labels) return fail(ctx, TRK_ERR_INVALID_ARG, "result.labels is required");
  if (n > 0 && !batch->hits) return fail(ctx, TRK_ERR_INVALID_ARG, "batch.hits is NULL");
  if ((res->edge_src || res->edge_dst || res->edge_score) && res->edge_capacity <= 0)
    return fail(ctx, TRK_ERR_INVALID_ARG, "edge outputs requested with edge_capacity <= 0");
  if ((res->cand_src || res->cand_dst || res->cand_score) && res->cand_capacity <= 0)
    return fail(ctx, TRK_ERR_INVALID_ARG, "candidate outputs requested with cand_capacity <= 0");
  const bool want_t = res->track_offsets || res->track_hits || res->track_counts;
  if (want_t && (!res->track_offsets || !res->track_hits || !res->track_counts || res->track_capacity <= 0))
    return fail(ctx, TRK_ERR_INVALID_ARG, "track outputs need track_offsets, track_hits, track_counts and track_capacity > 0");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const trk_config& f = ctx->cfg;
  ctx->kprof_n = 0;
  TRK_LAUNCH(ctx, zero_counts_kernel, 1, 32, 0, st, ctx->counts);
  const bool prof = ctx->profiling && n > 0;
  ctx->prof_valid = false;
#define TRK_MARK(i) do { if (prof) TRK_CUDA(ctx, cudaEventRecord(ctx->prof_ev[i], st)); } while (0)
  if (n > 0) {
    TRK_TRY(set_event_ids(ctx, batch->event_offsets, batch->n_events, n, st));
    TRK_MARK(0);
    TRK_TRY(embed_dispatch(ctx, batch->hits, n, ctx->emb, st));
    TRK_MARK(1);
    TRK_TRY(frnn_build(ctx, ctx->emb, batch->hits, n, batch->n_events, ctx->cand_src, ctx->cand_dst, nullptr, f.max_cand_edges,
                       &ctx->counts[0], &ctx->counts[3], st));
    TRK_MARK(2);
    const float* feat = f.filter_input == TRK_FILTER_EMB ? ctx->emb : batch->hits;
    const int64_t cand_cap = std::min<int64_t>(f.max_cand_edges, n * f.frnn_k);
    TRK_TRY(filter_dispatch(ctx, feat, ctx->cand_src, ctx->cand_dst, &ctx->counts[0], cand_cap, ctx->cand_score, st));
    TRK_TRY(compact_edges(ctx, ctx->cand_src, ctx->cand_dst, ctx->cand_score, &ctx->counts[0], cand_cap, f.filter_cut, ctx->kept_src,
                          ctx->kept_dst, f.max_kept_edges, &ctx->counts[1], &ctx->counts[3], st));
    const int64_t kept_cap = std::min<int64_t>(f.max_kept_edges, cand_cap);
    TRK_MARK(3);
    TRK_TRY(gnn_dispatch(ctx, batch->hits, n, ctx->kept_src, ctx->kept_dst, &ctx->counts[1], kept_cap, ctx->kept_score, st));
    TRK_MARK(4);
    TRK_TRY(cc_labels(ctx, n, ctx->kept_src, ctx->kept_dst, ctx->kept_score, &ctx->counts[1], kept_cap, f.gnn_cut, res->labels,
                      &ctx->counts[2], st));
    TRK_MARK(5);
    ctx->prof_valid = prof;
    if (want_t)
      TRK_TRY(build_tracks(ctx, res->labels, n, f.min_track_hits, res->track_offsets, res->track_capacity, res->track_hits,
                           res->track_counts, &ctx->counts[3], st));
    if (res->embedding) TRK_CUDA(ctx, cudaMemcpyAsync(res->embedding, ctx->emb, (size_t)n * ctx->d_e * 4, cudaMemcpyDeviceToDevice, st));
    const size_t ne = (size_t)std::min<int64_t>(res->edge_capacity, kept_cap), nc = (size_t)std::min<int64_t>(res->cand_capacity, cand_cap);
    if (res->edge_src) TRK_CUDA(ctx, cudaMemcpyAsync(res->edge_src, ctx->kept_src, ne * 4, cudaMemcpyDeviceToDevice, st));
    if (res->edge_dst) TRK_CUDA(ctx, cudaMemcpyAsync(res->edge_dst, ctx->kept_dst, ne * 4, cudaMemcpyDeviceToDevice, st));
    if (res->edge_score) TRK_CUDA(ctx, cudaMemcpyAsync(res->edge_score, ctx->kept_score, ne * 4, cudaMemcpyDeviceToDevice, st));
    if (res->cand_src) TRK_CUDA(ctx, cudaMemcpyAsync(res->cand_src, ctx->cand_src, nc * 4, cudaMemcpyDeviceToDevice, st));
    if (res->cand_dst) TRK_CUDA(ctx, cudaMemcpyAsync(res->cand_dst, ctx->cand_dst, nc * 4, cudaMemcpyDeviceToDevice, st));
    if (res->cand_score) TRK_CUDA(ctx, cudaMemcpyAsync(res->cand_score, ctx->cand_score, nc * 4, cudaMemcpyDeviceToDevice, st));
  }
  if (n <= 0 && want_t) TRK_TRY(build_tracks(ctx, nullptr, 0, 1, res->track_offsets, res->track_capacity, res->track_hits, res->track_counts, nullptr, st));
  const bool want_e = res->edge_src || res->edge_dst || res->edge_score, want_c = res->cand_src || res->cand_dst || res->cand_score;
  TRK_LAUNCH(ctx, finalize_counts_kernel, 1, 32, 0, st, ctx->counts, want_e ? res->edge_capacity : (int64_t)-1,
             want_c ? res->cand_capacity : (int64_t)-1, res->counts);
  return TRK_OK;
}

trk_status trk_infer_host(trk_ctx* ctx, int32_t n_events, const int32_t* event_offsets, const float* hits_host, int32_t* labels_host,
                          int32_t* counts_host) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->device);
  int64_t n = 0;
  TRK_TRY(check_batch(ctx, n_events, event_offsets, &n));
  if (n > 0 && (!hits_host || !labels_host)) return fail(ctx, TRK_ERR_INVALID_ARG, "hits_host or labels_host is NULL");
  cudaStream_t st = ctx->own_stream;
  if (n > 0) TRK_CUDA(ctx, cudaMemcpyAsync(ctx->io_hits, hits_host, (size_t)n * 12, cudaMemcpyHostToDevice, st));
  trk_batch b{n_events, event_offsets, ctx->io_hits};
  trk_result r;
  std::memset(&r, 0, sizeof(r));
  r.labels = ctx->io_labels;
  r.counts = ctx->io_counts;
  TRK_TRY(trk_infer(ctx, &b, &r, st));
  if (n > 0) TRK_CUDA(ctx, cudaMemcpyAsync(labels_host, ctx->io_labels, (size_t)n * 4, cudaMemcpyDeviceToHost, st));
  if (counts_host) TRK_CUDA(ctx, cudaMemcpyAsync(counts_host, ctx->io_counts, 16, cudaMemcpyDeviceToHost, st));
  TRK_CUDA(ctx, cudaStreamSynchronize(st));
  return TRK_OK;
}

trk_status trk_infer_host_tracks(trk_ctx* ctx, int32_t n_events, const int32_t* event_offsets, const float* hits_host,
                                 int32_t* labels_host, int32_t* track_offsets_host, int32_t* track_hits_host, int32_t* counts_host) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->device);
  int64_t n = 0;
  TRK_TRY(check_batch(ctx, n_events, event_offsets, &n));
  if (!track_offsets_host || !counts_host || (n > 0 && (!hits_host || !track_hits_host)))
    return fail(ctx, TRK_ERR_INVALID_ARG, "infer_host_tracks: a required host pointer is NULL");
  cudaStream_t st = ctx->own_stream;
  if (n > 0) TRK_CUDA(ctx, cudaMemcpyAsync(ctx->io_hits, hits_host, (size_t)n * 12, cudaMemcpyHostToDevice, st));
  trk_batch b{n_events, event_offsets, ctx->io_hits};
  trk_result r;
  std::memset(&r, 0, sizeof(r));
  r.labels = ctx->io_labels;
  r.counts = ctx->io_counts;
  r.track_offsets = ctx->io_track_offsets;
  r.track_hits = ctx->io_track_hits;
  r.track_counts = ctx->io_counts + 4;
  r.track_capacity = std::max<int64_t>(n, 1);
  TRK_TRY(trk_infer(ctx, &b, &r, st));
  if (n > 0 && labels_host) TRK_CUDA(ctx, cudaMemcpyAsync(labels_host, ctx->io_labels, (size_t)n * 4, cudaMemcpyDeviceToHost, st));
  TRK_CUDA(ctx, cudaMemcpyAsync(counts_host, ctx->io_counts, 24, cudaMemcpyDeviceToHost, st));
  TRK_CUDA(ctx, cudaStreamSynchronize(st));
  // the sizes are known now: copy exactly the T+1 offsets and the hits of the tracks
  const int64_t T = counts_host[4], nh = counts_host[5];
  TRK_CUDA(ctx, cudaMemcpyAsync(track_offsets_host, ctx->io_track_offsets, (size_t)(T + 1) * 4, cudaMemcpyDeviceToHost, st));
  if (nh > 0) TRK_CUDA(ctx, cudaMemcpyAsync(track_hits_host, ctx->io_track_hits, (size_t)nh * 4, cudaMemcpyDeviceToHost, st));
  TRK_CUDA(ctx, cudaStreamSynchronize(st));
  return TRK_OK;
}

trk_status trk_profile_enable(trk_ctx* ctx, int32_t on) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->device);
  if (on && !ctx->prof_ev[0]) {
    for (auto& e : ctx->prof_ev) TRK_CUDA(ctx, cudaEventCreate(&e));
    // one event pair per hidden-layer GEMM launch of S3 (trk_profile_kernel_ms): created here so that trk_infer never allocates
    const size_t pairs = (size_t)ceil_div(ctx->cfg.max_cand_edges, ctx->filter_chunk) * ctx->filter.layers.size();
    while (ctx->kprof_ev.size() < 2 * pairs) {
      cudaEvent_t e;
      TRK_CUDA(ctx, cudaEventCreate(&e));
      ctx->kprof_ev.push_back(e);
    }
  }
  ctx->profiling = on != 0;
  ctx->prof_valid = false;
  return TRK_OK;
}

trk_status trk_profile_stage_ms(trk_ctx* ctx, float* ms) {
  if (!ctx || !ms) return TRK_ERR_INVALID_ARG;
  if (!ctx->prof_valid) return fail(ctx, TRK_ERR_INVALID_ARG, "no profiled trk_infer call to read");
  TRK_CUDA(ctx, cudaEventSynchronize(ctx->prof_ev[5]));
  for (int i = 0; i < 5; ++i) TRK_CUDA(ctx, cudaEventElapsedTime(&ms[i], ctx->prof_ev[i], ctx->prof_ev[i + 1]));
  return TRK_OK;
}

trk_status trk_profile_kernel_ms(trk_ctx* ctx, float* ms, int32_t capacity, int32_t* n_launches, int64_t* rows_per_launch) {
  if (!ctx || !n_launches || capacity < 0 || (capacity > 0 && !ms)) return TRK_ERR_INVALID_ARG;
  if (!ctx->prof_valid) return fail(ctx, TRK_ERR_INVALID_ARG, "no profiled trk_infer call to read");
  TRK_CUDA(ctx, cudaEventSynchronize(ctx->prof_ev[5]));
  *n_launches = ctx->kprof_n;
  // fused S3 (one launch runs every layer over all candidate edges): -1; layer by layer: the rows of one pass
  if (rows_per_launch) *rows_per_launch = ctx->filter_fusable && ctx->knobs[kKnobFilterFused] != 0 ? -1 : ctx->filter_chunk;
  for (int i = 0; i < ctx->kprof_n && i < capacity; ++i)
    TRK_CUDA(ctx, cudaEventElapsedTime(&ms[i], ctx->kprof_ev[(size_t)i * 2], ctx->kprof_ev[(size_t)i * 2 + 1]));
  return TRK_OK;
}

// ------------------------------------------------------------------ stage hooks
trk_status trk_stage_embed(trk_ctx* ctx, const float* hits, int64_t n, float* emb, void* cuda_stream) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->device);
  if (n < 0 || (n > 0 && (!hits || !emb))) return fail(ctx, TRK_ERR_INVALID_ARG, "stage_embed: bad arguments");
  if (n > ctx->cfg.max_hits) return fail(ctx, TRK_ERR_CAPACITY, "stage_embed: n exceeds max_hits");
  return embed_dispatch(ctx, hits, n, emb, (cudaStream_t)cuda_stream);
}

trk_status trk_stage_frnn(trk_ctx* ctx, const float* emb, const float* hits, const int32_t* event_offsets, int32_t n_events,
                          int32_t* src, int32_t* dst, int32_t* rowptr, int64_t capacity, int32_t* count, void* cuda_stream) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->device);
  int64_t n = 0;
  TRK_TRY(check_batch(ctx, n_events, event_offsets, &n));
  if (!count || capacity < 0 || (capacity > 0 && (!src || !dst))) return fail(ctx, TRK_ERR_INVALID_ARG, "stage_frnn: bad arguments");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  TRK_LAUNCH(ctx, zero_counts_kernel, 1, 32, 0, st, ctx->counts);
  if (n > 0) {
    if (!emb || !hits) return fail(ctx, TRK_ERR_INVALID_ARG, "stage_frnn: emb or hits is NULL");
    TRK_TRY(set_event_ids(ctx, event_offsets, n_events, n, st));
    TRK_TRY(frnn_build(ctx, emb, hits, n, n_events, src, dst, rowptr, capacity, &ctx->counts[0], &ctx->counts[3], st));
  } else if (rowptr) {
    TRK_CUDA(ctx, cudaMemsetAsync(rowptr, 0, 4, st));
  }
  TRK_CUDA(ctx, cudaMemcpyAsync(count, &ctx->counts[0], 4, cudaMemcpyDeviceToDevice, st));
  TRK_CUDA(ctx, cudaMemcpyAsync(count + 1, &ctx->counts[3], 4, cudaMemcpyDeviceToDevice, st));
  return TRK_OK;
}

trk_status trk_stage_filter(trk_ctx* ctx, const float* feat, int64_t n, const int32_t* src, const int32_t* dst, int64_t n_edges,
                            float* score, void* cuda_stream) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->device);
  if (n < 0 || n_edges < 0 || (n_edges > 0 && (!feat || !src || !dst || !score))) return fail(ctx, TRK_ERR_INVALID_ARG, "stage_filter: bad arguments");
  return filter_dispatch(ctx, feat, src, dst, nullptr, n_edges, score, (cudaStream_t)cuda_stream);
}

trk_status trk_stage_compact(trk_ctx* ctx, const int32_t* src, const int32_t* dst, const float* score, int64_t n_edges,
                             int32_t* out_src, int32_t* out_dst, int64_t capacity, int32_t* count, void* cuda_stream) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->device);
  if (n_edges < 0 || capacity < 0 || !count || (n_edges > 0 && (!src || !dst || !score || !out_src || !out_dst)))
    return fail(ctx, TRK_ERR_INVALID_ARG, "stage_compact: bad arguments");
  if (n_edges > ctx->cfg.max_cand_edges) return fail(ctx, TRK_ERR_CAPACITY, "stage_compact: n_edges exceeds max_cand_edges");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  TRK_LAUNCH(ctx, zero_counts_kernel, 1, 32, 0, st, ctx->counts);
  // n_edges is a host scalar here: store it in counts[5] and use it as the device count
  TRK_TRY(fill_i32(ctx, &ctx->counts[5], (int32_t)n_edges, 1, st));
  TRK_TRY(compact_edges(ctx, src, dst, score, &ctx->counts[5], n_edges, ctx->cfg.filter_cut, out_src, out_dst, capacity,
                        &ctx->counts[1], &ctx->counts[3], st));
  TRK_CUDA(ctx, cudaMemcpyAsync(count, &ctx->counts[1], 4, cudaMemcpyDeviceToDevice, st));
  TRK_CUDA(ctx, cudaMemcpyAsync(count + 1, &ctx->counts[3], 4, cudaMemcpyDeviceToDevice, st));
  return TRK_OK;
}

trk_status trk_stage_gnn(trk_ctx* ctx, const float* hits, int64_t n, const int32_t* src, const int32_t* dst, int64_t n_edges,
                         float* score, void* cuda_stream) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->device);
  if (n < 0 || n_edges < 0 || (n > 0 && !hits) || (n_edges > 0 && (!src || !dst || !score)))
    return fail(ctx, TRK_ERR_INVALID_ARG, "stage_gnn: bad arguments");
  if (n > ctx->cfg.max_hits || n_edges > ctx->cfg.max_kept_edges) return fail(ctx, TRK_ERR_CAPACITY, "stage_gnn: exceeds max_hits / max_kept_edges");
  return gnn_dispatch(ctx, hits, n, src, dst, nullptr, n_edges, score, (cudaStream_t)cuda_stream);
}

trk_status trk_stage_gnn_csr(trk_ctx* ctx, const float* hits, int64_t n, const int32_t* src, const int32_t* dst, int64_t n_edges,
                             int32_t* in_rowptr, int32_t* in_perm, int32_t* out_rowptr, void* cuda_stream) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->device);
  if (n <= 0 || n_edges < 0 || !hits || !in_rowptr || !out_rowptr || (n_edges > 0 && (!src || !dst || !in_perm)))
    return fail(ctx, TRK_ERR_INVALID_ARG, "stage_gnn_csr: bad arguments");
  if (n > ctx->cfg.max_hits || n_edges > ctx->cfg.max_kept_edges) return fail(ctx, TRK_ERR_CAPACITY, "stage_gnn_csr: exceeds max_hits / max_kept_edges");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  TRK_TRY(build_gnn_csr(ctx, hits, src, dst, nullptr, n_edges, n, st));
  TRK_CUDA(ctx, cudaMemcpyAsync(in_rowptr, ctx->in_rowptr, (size_t)(n + 1) * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
  TRK_CUDA(ctx, cudaMemcpyAsync(out_rowptr, ctx->out_rowptr, (size_t)(n + 1) * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
  if (n_edges > 0) TRK_CUDA(ctx, cudaMemcpyAsync(in_perm, ctx->in_perm, (size_t)n_edges * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
  return TRK_OK;
}

trk_status trk_stage_cc(trk_ctx* ctx, int64_t n, const int32_t* src, const int32_t* dst, const float* score, int64_t n_edges,
                        float cut, int32_t* labels, void* cuda_stream) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->device);
  if (n < 0 || n_edges < 0 || (n > 0 && !labels) || (n_edges > 0 && (!src || !dst || !score)))
    return fail(ctx, TRK_ERR_INVALID_ARG, "stage_cc: bad arguments");
  if (n > ctx->cfg.max_hits) return fail(ctx, TRK_ERR_CAPACITY, "stage_cc: n exceeds max_hits");
  return cc_labels(ctx, n, src, dst, score, nullptr, n_edges, cut, labels, nullptr, (cudaStream_t)cuda_stream);
}

trk_status trk_stage_tracks(trk_ctx* ctx, const int32_t* labels, int64_t n, int32_t min_hits, int32_t* track_offsets, int64_t capacity,
                            int32_t* track_hits, int32_t* track_counts, void* cuda_stream) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->device);
  if (n < 0 || capacity <= 0 || !track_offsets || !track_counts || (n > 0 && (!labels || !track_hits)))
    return fail(ctx, TRK_ERR_INVALID_ARG, "stage_tracks: bad arguments");
  if (n > ctx->cfg.max_hits) return fail(ctx, TRK_ERR_CAPACITY, "stage_tracks: n exceeds max_hits");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  TRK_TRY(fill_i32(ctx, track_counts, 0, 3, st));
  return build_tracks(ctx, labels, n, min_hits, track_offsets, capacity, track_hits, track_counts, track_counts + 2, st);
}

trk_status trk_set_option(trk_ctx* ctx, const char* key, int64_t value) {
  if (!ctx) return TRK_ERR_INVALID_ARG;
  if (!key) return fail(ctx, TRK_ERR_INVALID_ARG, "trk_set_option: key is NULL");
  static const struct { const char* name; int knob; } keys[] = {
      {"gemm_pair", kKnobGemmPair}, {"gnn_fused", kKnobGnnFused}, {"epi_split", kKnobEpiSplit}, {"gemm_row_major", kKnobRowMajor},
      {"filter_fused", kKnobFilterFused}, {"filter_max_pairs", kKnobFilterPairs}};
  for (const auto& k : keys)
    if (std::strcmp(key, k.name) == 0) {
      ctx->knobs[k.knob] = value;
      return TRK_OK;
    }
  return fail(ctx, TRK_ERR_INVALID_ARG, std::string("trk_set_option: unknown key ") + key);
}

trk_status trk_gemm_bf16(const void* a, const void* w, const float* bias, void* out, int64_t m, int32_t n, int32_t k, int32_t relu,
                         int32_t pair, void* cuda_stream) {
  if (!a || !w || !bias || !out || m <= 0 || (pair != 0 && pair != 1)) return fail(nullptr, TRK_ERR_INVALID_ARG, "gemm_bf16: bad arguments");
  if (k % 64 != 0 || n % 64 != 0) return fail(nullptr, TRK_ERR_SHAPE, "gemm_bf16: k and n must be multiples of 64");
  trk_ctx hook_ctx;  // per call (runs on the caller's current device): only sm_count, knobs, launch_count and last_error are used
  hook_ctx.knobs[kKnobGemmPair] = pair;
  int dev = 0;
  cudaGetDevice(&dev);
  hook_ctx.device = dev;
  cudaDeviceGetAttribute(&hook_ctx.sm_count, cudaDevAttrMultiProcessorCount, dev);
  trk_status s = gemm_bf16_hook(&hook_ctx, a, w, bias, out, m, n, k, relu, (cudaStream_t)cuda_stream);
  if (s != TRK_OK) fail(nullptr, s, hook_ctx.last_error);
  return s;
}

}  // extern "C"

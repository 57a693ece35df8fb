// TRK_FP32 precision: S1, S3 and S4 on the plain fp32 ALUs (SIMT).  This is the path of the toy
// config (BASELINE.json configs[0], "1e-4 relative if run in fp32") and of any layer shape the
// tcgen05 path does not take (hidden widths that are not multiples of 64).  It is not tuned: the
// measured configs run in TRK_BF16 on the tensor cores (nn_bf16.cu, gemm_tc.cuh).
#include "common.cuh"
#include "graph.cuh"
#include "nn.cuh"

namespace trk {
namespace {

constexpr int TM = 64, TN = 64, TK = 16;

__device__ __forceinline__ int64_t rows_of(const int32_t* m_dev, int64_t m_off, int64_t m_cap) {
  if (!m_dev) return m_cap;
  int64_t m = (int64_t)*m_dev - m_off;
  return m < 0 ? 0 : (m > m_cap ? m_cap : m);
}

// C[m][n] = act(sum_k A[m][k] W[n][k] + b[n]);  ACT 0 none, 1 relu, 2 sigmoid
template <int ACT>
__global__ void __launch_bounds__(256)
linear_f32_kernel(const float* __restrict__ A, int lda, const float* __restrict__ W, const float* __restrict__ bias,
                  float* __restrict__ C, int ldc, const int32_t* __restrict__ m_dev, int64_t m_off, int64_t m_cap, int N, int K) {
  TRK_GRID_DEP_WAIT();
  __shared__ float As[TK][TM + 4];
  __shared__ float Ws[TK][TN + 4];
  const int64_t M = rows_of(m_dev, m_off, m_cap);
  const int64_t m0 = (int64_t)blockIdx.x * TM;
  if (m0 >= M) return;
  const int n0 = blockIdx.y * TN;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
  for (int k0 = 0; k0 < K; k0 += TK) {
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      const int idx = threadIdx.x + t * 256;   // 0..1023
      const int r = idx >> 4, c = idx & 15;    // row in tile, k in tile (k fastest: coalesced along K)
      const int64_t gm = m0 + r;
      const int gk = k0 + c;
      As[c][r] = (gm < M && gk < K) ? A[gm * lda + gk] : 0.f;
      const int gn = n0 + r;
      Ws[c][r] = (gn < N && gk < K) ? W[(int64_t)gn * K + gk] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < TK; ++k) {
      float a[4], w[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[k][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) w[j] = Ws[k][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], w[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int64_t gm = m0 + ty * 4 + i;
    if (gm >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int gn = n0 + tx * 4 + j;
      if (gn >= N) continue;
      float v = acc[i][j] + (bias ? bias[gn] : 0.f);
      if (ACT == 1) v = fmaxf(v, 0.f);
      if (ACT == 2) v = 1.f / (1.f + expf(-v));
      C[gm * ldc + gn] = v;
    }
  }
}

// Row-wise: v = ReLU(LayerNorm(x)) (or ReLU(x)); out = (res ? res : 0) + v.  One warp per row; in-place safe.
__global__ void __launch_bounds__(256)
ln_relu_f32_kernel(const float* __restrict__ x, int ldx, const float* __restrict__ res, int ldr, float* __restrict__ out, int ldo,
                   const int32_t* __restrict__ m_dev, int64_t m_cap, int N, int use_ln) {
  TRK_GRID_DEP_WAIT();
  const int64_t M = rows_of(m_dev, 0, m_cap);
  const int lane = threadIdx.x & 31;
  const int64_t row = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (row >= M) return;
  const float* xr = x + row * ldx;
  float mean = 0.f, rstd = 1.f;
  if (use_ln) {
    float s = 0.f;
    for (int c = lane; c < N; c += 32) s += xr[c];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    mean = s / (float)N;
    float q = 0.f;
    for (int c = lane; c < N; c += 32) { float d = xr[c] - mean; q += d * d; }
    for (int o = 16; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
    rstd = rsqrtf(q / (float)N + 1e-5f);
  }
  for (int c = lane; c < N; c += 32) {
    float v = fmaxf((xr[c] - mean) * rstd, 0.f);
    if (res) v += res[row * ldr + c];
    out[row * ldo + c] = v;
  }
}

// out[k] = [feat[src[k]] ; feat[dst[k]]], u floats each.
__global__ void gather_pair_f32_kernel(const float* __restrict__ feat, int u, const int32_t* __restrict__ src,
                                       const int32_t* __restrict__ dst, const int32_t* __restrict__ m_dev, int64_t m_off,
                                       int64_t m_cap, float* __restrict__ out) {
  TRK_GRID_DEP_WAIT();
  const int64_t M = rows_of(m_dev, m_off, m_cap);
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t row = i / (2 * u);
  if (row >= M) return;
  const int c = (int)(i % (2 * u));
  const int64_t node = c < u ? src[m_off + row] : dst[m_off + row];
  out[i] = feat[node * u + (c < u ? c : c - u)];
}

// cat[k] = [h[src[k]] ; h[dst[k]] ; e[k]]   (h rows have stride ldh)
__global__ void gather_edge_cat_f32_kernel(const float* __restrict__ h, int ldh, const float* __restrict__ e, int H,
                                           const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
                                           const int32_t* __restrict__ m_dev, int64_t m_cap, float* __restrict__ cat) {
  TRK_GRID_DEP_WAIT();
  const int64_t M = rows_of(m_dev, 0, m_cap);
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t row = i / (3 * H);
  if (row >= M) return;
  const int c = (int)(i % (3 * H));
  float v;
  if (c < H) v = h[(int64_t)src[row] * ldh + c];
  else if (c < 2 * H) v = h[(int64_t)dst[row] * ldh + (c - H)];
  else v = e[row * H + (c - 2 * H)];
  cat[i] = v;
}

}  // namespace

// (dr, dphi wrapped to (-1,1], dz, deta) per edge; shared with the bf16 path (nn.cuh).
__global__ void edge_features_kernel(const float* __restrict__ hits, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
                                     const int32_t* __restrict__ m_dev, int64_t m_cap, float4* __restrict__ out) {
  TRK_GRID_DEP_WAIT();
  const int64_t M = m_dev ? min((int64_t)max(*m_dev, 0), m_cap) : m_cap;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= M) return;
  out[k] = edge_features(hits, src[k], dst[k]);
}

namespace {

trk_status linear_f32(trk_ctx* ctx, int act, const float* A, int lda, const DevLinear& L, float* C, int ldc, const int32_t* m_dev,
                      int64_t m_off, int64_t m_cap, cudaStream_t st) {
  if (m_cap <= 0) return TRK_OK;
  dim3 grid((unsigned)ceil_div(m_cap, TM), (unsigned)ceil_div(L.out, TN));
  if (act == 0) TRK_LAUNCH(ctx, linear_f32_kernel<0>, grid, 256, 0, st, A, lda, L.w_f32, L.b_f32, C, ldc, m_dev, m_off, m_cap, L.out, L.in);
  else if (act == 1) TRK_LAUNCH(ctx, linear_f32_kernel<1>, grid, 256, 0, st, A, lda, L.w_f32, L.b_f32, C, ldc, m_dev, m_off, m_cap, L.out, L.in);
  else TRK_LAUNCH(ctx, linear_f32_kernel<2>, grid, 256, 0, st, A, lda, L.w_f32, L.b_f32, C, ldc, m_dev, m_off, m_cap, L.out, L.in);
  return TRK_OK;
}

trk_status ln_relu_f32(trk_ctx* ctx, const float* x, int ldx, const float* res, int ldr, float* out, int ldo, const int32_t* m_dev,
                       int64_t m_cap, int N, cudaStream_t st) {
  if (m_cap <= 0) return TRK_OK;
  TRK_LAUNCH(ctx, ln_relu_f32_kernel, (unsigned)ceil_div(m_cap * 32, 256), 256, 0, st, x, ldx, res, ldr, out, ldo, m_dev, m_cap, N,
             ctx->cfg.gnn_layernorm);
  return TRK_OK;
}

// Two Linear layers, both followed by LNR; result (+ residual) written to out.
trk_status mlp2_lnr_f32(trk_ctx* ctx, const float* in, int ldin, const DevMlp& mlp, float* tmp, const float* res, int ldr, float* out,
                        int ldo, const int32_t* m_dev, int64_t m_cap, cudaStream_t st) {
  const int H = ctx->H;
  float* t2 = tmp + (size_t)m_cap * H;  // second half of the scratch
  TRK_TRY(linear_f32(ctx, 0, in, ldin, mlp.layers[0], tmp, H, m_dev, 0, m_cap, st));
  TRK_TRY(ln_relu_f32(ctx, tmp, H, nullptr, 0, tmp, H, m_dev, m_cap, H, st));
  TRK_TRY(linear_f32(ctx, 0, tmp, H, mlp.layers[1], t2, H, m_dev, 0, m_cap, st));
  TRK_TRY(ln_relu_f32(ctx, t2, H, res, ldr, out, ldo, m_dev, m_cap, H, st));
  return TRK_OK;
}

}  // namespace

trk_status embed_forward_fp32(trk_ctx* ctx, const float* hits, int64_t n, float* emb, cudaStream_t st) {
  const auto& L = ctx->embed.layers;
  const float* in = hits;
  int ldin = 3;
  float* bufs[2] = {(float*)ctx->act0, (float*)ctx->act1};
  for (size_t l = 0; l < L.size(); ++l) {
    const bool last = l + 1 == L.size();
    float* out = last ? emb : bufs[l & 1];
    TRK_TRY(linear_f32(ctx, last ? 0 : 1, in, ldin, L[l], out, L[l].out, nullptr, 0, n, st));
    in = out;
    ldin = L[l].out;
  }
  return TRK_OK;
}

trk_status filter_forward_fp32(trk_ctx* ctx, const float* feat, const int32_t* src, const int32_t* dst,
                               const int32_t* n_edges_dev, int64_t n_edges_cap, float* score, cudaStream_t st) {
  const auto& L = ctx->filter.layers;
  const int u = ctx->filter_u;
  float* bufs[2] = {(float*)ctx->act0, (float*)ctx->act1};
  for (int64_t off = 0; off < n_edges_cap; off += ctx->filter_chunk) {
    const int64_t cap = std::min<int64_t>(ctx->filter_chunk, n_edges_cap - off);
    float* gin = (float*)ctx->act_in;
    TRK_LAUNCH(ctx, gather_pair_f32_kernel, (unsigned)ceil_div(cap * 2 * u, 256), 256, 0, st, feat, u, src, dst, n_edges_dev, off,
               cap, gin);
    const float* in = gin;
    int ldin = 2 * u;
    for (size_t l = 0; l < L.size(); ++l) {
      const bool last = l + 1 == L.size();
      float* out = last ? score + off : bufs[l & 1];
      TRK_TRY(linear_f32(ctx, last ? 2 : 1, in, ldin, L[l], out, L[l].out, n_edges_dev, off, cap, st));
      in = out;
      ldin = L[l].out;
    }
  }
  return TRK_OK;
}

trk_status gnn_forward_fp32(trk_ctx* ctx, const float* hits, int64_t n, const int32_t* src, const int32_t* dst,
                            const int32_t* n_edges_dev, int64_t n_edges_cap, float* score, cudaStream_t st) {
  const int H = ctx->H;
  float* X = (float*)ctx->X;    // [n][3H]: h | m_in | m_out
  float* E = (float*)ctx->E;    // [E][H]
  float* T1 = (float*)ctx->T1;  // scratch, 2 * rows * H floats
  float* cat = ctx->cat;
  TRK_TRY(build_gnn_csr(ctx, hits, src, dst, n_edges_dev, n_edges_cap, n, st));
  // encoders
  TRK_TRY(mlp2_lnr_f32(ctx, hits, 3, ctx->node_enc, T1, nullptr, 0, X, 3 * H, nullptr, n, st));
  if (n_edges_cap > 0) {
    TRK_LAUNCH(ctx, edge_features_kernel, (unsigned)ceil_div(n_edges_cap, 256), 256, 0, st, hits, src, dst, n_edges_dev, n_edges_cap,
               (float4*)cat);
    TRK_TRY(mlp2_lnr_f32(ctx, cat, 4, ctx->edge_enc, T1, nullptr, 0, E, H, n_edges_dev, n_edges_cap, st));
  }
  for (int t = 0; t < ctx->cfg.gnn_iters; ++t) {
    if (n_edges_cap > 0) {
      TRK_LAUNCH(ctx, gather_edge_cat_f32_kernel, (unsigned)ceil_div(n_edges_cap * 3 * H, 256), 256, 0, st, X, 3 * H, E, H, src, dst,
                 n_edges_dev, n_edges_cap, cat);
      TRK_TRY(mlp2_lnr_f32(ctx, cat, 3 * H, ctx->edge_net, T1, E, H, E, H, n_edges_dev, n_edges_cap, st));
    }
    TRK_TRY(segment_sums(ctx, E, false, n, X, st));
    TRK_TRY(mlp2_lnr_f32(ctx, X, 3 * H, ctx->node_net, T1, X, 3 * H, X, 3 * H, nullptr, n, st));
  }
  if (n_edges_cap > 0) {
    TRK_LAUNCH(ctx, gather_edge_cat_f32_kernel, (unsigned)ceil_div(n_edges_cap * 3 * H, 256), 256, 0, st, X, 3 * H, E, H, src, dst,
               n_edges_dev, n_edges_cap, cat);
    TRK_TRY(linear_f32(ctx, 0, cat, 3 * H, ctx->edge_dec.layers[0], T1, H, n_edges_dev, 0, n_edges_cap, st));
    TRK_TRY(ln_relu_f32(ctx, T1, H, nullptr, 0, T1, H, n_edges_dev, n_edges_cap, H, st));
    TRK_TRY(linear_f32(ctx, 2, T1, H, ctx->edge_dec.layers[1], score, 1, n_edges_dev, 0, n_edges_cap, st));
  }
  return TRK_OK;
}

}  // namespace trk

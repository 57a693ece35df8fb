// TRK_BF16 precision: S1, S3 and S4 with every dense layer on the tcgen05 tensor cores
// (gemm_tc.cuh); layers whose K is 3 or 4 run on the plain ALUs in fp32 (they are <0.1% of the flops).
//
// S1   hits -> [SIMT 3->W] -> GEMM+ReLU ... -> GEMM (N padded to 16, fp32 out) = embedding
// S3   per chunk of ctx->filter_chunk edges (up to 64 row tiles per SM; the activations of a chunk stream through HBM):
//        gather [e_src ; e_dst] -> bf16 [rows][64] (K zero-padded) -> GEMM+ReLU ... -> last hidden GEMM
//        with the final Linear(W->1) folded into its epilogue as per-tile partial dots -> sigmoid
// S4   the first layer of edge_net / edge_dec is split exactly:
//        W1 [h_s ; h_d ; e] = Wa h_s + Wb h_d + Wc e
//      so one per-node GEMM (N = 2H) produces PA|PB in fp32 and the per-edge GEMM has K = H only;
//      the epilogue gathers PA[src] + PB[dst], applies LayerNorm+ReLU (+ residual) in registers.
//      This halves the per-edge flops against the dense concat.
#include <mutex>

#include "common.cuh"
#include "gemm_tc.cuh"
#include "gemm_tc2.cuh"
#include "filter_fused.cuh"
#include "gnn_fused.cuh"
#include "graph.cuh"
#include "nn.cuh"

namespace trk {
namespace {

using bf16 = __nv_bfloat16;

// ---------------------------------------------------------------- tensor maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  });
  return fn;
}

// bf16 matrix [rows][k] with row stride ld (elements); box = 64 (k) x box_rows; 128-byte swizzle.
trk_status make_tmap(trk_ctx* ctx, CUtensorMap* m, const void* base, int64_t rows, int k, int64_t ld, int box_rows) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return fail(ctx, TRK_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
  cuuint64_t dims[2] = {(cuuint64_t)k, (cuuint64_t)(rows > 0 ? rows : 1)};
  cuuint64_t strides[1] = {(cuuint64_t)ld * 2};
  cuuint32_t box[2] = {64u, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1u, 1u};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(ctx, TRK_ERR_CUDA, "cuTensorMapEncodeTiled failed with code " + std::to_string((int)r));
  return TRK_OK;
}

// Output of a TMA-store epilogue: bf16 [rows][n] with row stride ld (elements).
struct OutBf16 {
  bf16* ptr = nullptr;
  int64_t rows = 0;
  int64_t ld = 0;
};

// A [a_rows][K] bf16 (row stride lda), W [n_pad][K] bf16 K-major; rows of the product resolved on the device.
template <int BN, class Epi>
trk_status launch_gemm(trk_ctx* ctx, const bf16* A, int64_t a_rows, int64_t lda, int K, const bf16* W, int n_pad, tc::Rows rows,
                       const typename Epi::Params& ep, cudaStream_t st, OutBf16 out = OutBf16(), const tc::AGather* ag = nullptr) {
  if (rows.m_cap <= 0) return TRK_OK;
  if (K % tc::BK != 0 || n_pad % BN != 0) return fail(ctx, TRK_ERR_SHAPE, "gemm: K must be a multiple of 64 and N of the tile");
  auto kern = tc::gemm_tc_kernel<BN, Epi>;
  TRK_TRY(ensure_smem(ctx, kern, tc::smem_bytes(BN, Epi::kTmaStore)));
  // tcgen05.mma.cta_group::2 on 256 x BN tiles when the K loop is long enough to matter (measured: with one K block the
  // epilogue paces the tile and coupling two CTAs only adds waiting)
  const bool pair = BN >= 128 && K >= 4 * tc::BK && ctx->knobs[kKnobGemmPair] != 0;
  CUtensorMap ta, tb, tc_out;
  TRK_TRY(make_tmap(ctx, &ta, A, a_rows, K, lda, tc::BM));
  TRK_TRY(make_tmap(ctx, &tb, W, n_pad, K, K, pair ? BN / 2 : BN));
  if (Epi::kTmaStore) {
    if (!out.ptr || out.ld % 8 != 0) return fail(ctx, TRK_ERR_SHAPE, "gemm: the bf16 output needs a row stride that is a multiple of 8");
    TRK_TRY(make_tmap(ctx, &tc_out, out.ptr, out.rows, n_pad, out.ld, 32));
  } else {
    tc_out = ta;
  }
  const int n_tiles = n_pad / BN;
  if constexpr (BN >= 128) {
    if (pair) {
      auto kern2 = tc::gemm_tc2_kernel<BN, Epi>;
      TRK_TRY(ensure_smem(ctx, kern2, tc::smem_bytes_pair(BN, Epi::kTmaStore)));
      const int64_t ptiles = ceil_div(rows.m_cap, tc::kPairBM) * n_tiles;
      const unsigned grid2 = 2u * (unsigned)std::min<int64_t>(ptiles, ctx->sm_count / 2);
      TRK_LAUNCH(ctx, kern2, grid2, tc::kThreads, tc::smem_bytes_pair(BN, Epi::kTmaStore), st, ta, tb, tc_out, rows, n_tiles, K / tc::BK, ep,
                 (int)ctx->knobs[kKnobRowMajor]);
      return TRK_OK;
    }
  }
  const int64_t tiles = ceil_div(rows.m_cap, tc::BM) * n_tiles;
  const unsigned grid = (unsigned)std::min<int64_t>(tiles, ctx->sm_count);
  if constexpr (BN == 256 && Epi::kTmaStore) {
    // a single K block per tile: the bf16-store epilogue paces the kernel, so it gets eight warps (column split)
    if (K == tc::BK && ag && ctx->knobs[kKnobEpiSplit] >= 2) {
      // ... and its A operand is gathered in the kernel (S3 first layer: no separate gather launch, no staging buffer)
      auto kern4 = tc::gemm_tc_kernel<BN, Epi, 2, true>;
      TRK_TRY(ensure_smem(ctx, kern4, tc::smem_bytes(BN, true, 2)));
      TRK_LAUNCH(ctx, kern4, grid, tc::threads_for(2, true), tc::smem_bytes(BN, true, 2), st, ta, tb, tc_out, rows, n_tiles, K / tc::BK, ep, *ag);
      return TRK_OK;
    }
    if (K == tc::BK && ctx->knobs[kKnobEpiSplit] != 0) {
      auto kern3 = tc::gemm_tc_kernel<BN, Epi, 2>;
      TRK_TRY(ensure_smem(ctx, kern3, tc::smem_bytes(BN, true, 2)));
      TRK_LAUNCH(ctx, kern3, grid, tc::threads_for(2), tc::smem_bytes(BN, true, 2), st, ta, tb, tc_out, rows, n_tiles, K / tc::BK, ep, tc::AGather{});
      return TRK_OK;
    }
  }
  TRK_LAUNCH(ctx, kern, grid, tc::kThreads, tc::smem_bytes(BN, Epi::kTmaStore), st, ta, tb, tc_out, rows, n_tiles, K / tc::BK, ep, tc::AGather{});
  return TRK_OK;
}

int pick_bn(int n_pad) { return n_pad % 256 == 0 ? 256 : (n_pad % 128 == 0 ? 128 : 64); }

// out: bf16 [out_rows][ldo]; every 128-row tile that holds a valid row is written in full (rows beyond out_rows are clipped).
trk_status gemm_bias_act(trk_ctx* ctx, const bf16* A, int64_t a_rows, int64_t lda, const DevLinear& L, bf16* out, int64_t out_rows,
                         int ldo, int relu, tc::Rows rows, cudaStream_t st, const tc::AGather* ag = nullptr) {
  tc::EpiBiasActBf16::Params ep{L.b_f32, relu};
  const OutBf16 o{out, out_rows, ldo};
  switch (pick_bn(L.out_pad)) {
    case 256: return launch_gemm<256, tc::EpiBiasActBf16>(ctx, A, a_rows, lda, L.in_pad, L.w_bf16, L.out_pad, rows, ep, st, o, ag);
    case 128: return launch_gemm<128, tc::EpiBiasActBf16>(ctx, A, a_rows, lda, L.in_pad, L.w_bf16, L.out_pad, rows, ep, st, o);
    default: return launch_gemm<64, tc::EpiBiasActBf16>(ctx, A, a_rows, lda, L.in_pad, L.w_bf16, L.out_pad, rows, ep, st, o);
  }
}

trk_status gemm_relu_dot(trk_ctx* ctx, const bf16* A, int64_t a_rows, int64_t lda, const DevLinear& L, const float* w_last,
                         float* partial, int* n_tiles_out, tc::Rows rows, cudaStream_t st) {
  const int bn = pick_bn(L.out_pad);
  tc::EpiReluDot::Params ep{L.b_f32, w_last, partial, L.out_pad / bn};
  *n_tiles_out = L.out_pad / bn;
  switch (bn) {
    case 256: return launch_gemm<256, tc::EpiReluDot>(ctx, A, a_rows, lda, L.in_pad, L.w_bf16, L.out_pad, rows, ep, st);
    case 128: return launch_gemm<128, tc::EpiReluDot>(ctx, A, a_rows, lda, L.in_pad, L.w_bf16, L.out_pad, rows, ep, st);
    default: return launch_gemm<64, tc::EpiReluDot>(ctx, A, a_rows, lda, L.in_pad, L.w_bf16, L.out_pad, rows, ep, st);
  }
}

trk_status gemm_store_f32(trk_ctx* ctx, const bf16* A, int64_t a_rows, int64_t lda, int K, const bf16* W, int n_pad, float* out,
                          tc::Rows rows, cudaStream_t st) {
  tc::EpiStoreF32::Params ep{out, n_pad};
  if (n_pad % 256 == 0) return launch_gemm<256, tc::EpiStoreF32>(ctx, A, a_rows, lda, K, W, n_pad, rows, ep, st);
  return launch_gemm<128, tc::EpiStoreF32>(ctx, A, a_rows, lda, K, W, n_pad, rows, ep, st);
}

trk_status gemm_row_ln(trk_ctx* ctx, const bf16* A, int64_t a_rows, int64_t lda, int K, const bf16* W, tc::EpiRowLn::Params ep,
                       tc::Rows rows, cudaStream_t st) {
  if (ctx->H == 128) return launch_gemm<128, tc::EpiRowLn>(ctx, A, a_rows, lda, K, W, 128, rows, ep, st);
  return launch_gemm<64, tc::EpiRowLn>(ctx, A, a_rows, lda, K, W, 64, rows, ep, st);
}

// bias vectors of the two layers into the by-value kernel parameter block (layer 2 is absent in the decoder: zeros)
static void fill_bias(gf::FusedParams& p, const DevLinear& L1, const DevLinear& L2) {
  for (int c = 0; c < gf::kH; ++c) {
    p.b1[c] = c < (int)L1.b_host.size() ? L1.b_host[c] : 0.f;
    p.b2[c] = c < (int)L2.b_host.size() ? L2.b_host[c] : 0.f;
  }
}

// Fused edge update / decoder of S4 (gnn_fused.cuh), H = 128: E <- E + LNR(W2 LNR(W1 [h_s ; h_d ; e] + b1) + b2) in place,
// or score = sigmoid(w_out . LNR(W1 [h_s ; h_d ; e] + b1) + b_out).
template <int MODE>
trk_status launch_edge_fused(trk_ctx* ctx, const bf16* X, int64_t ldx, bf16* E, int64_t e_rows, const int32_t* src, const int32_t* dst,
                             const DevLinear& L1, const DevLinear& L2, const float* w_out, float b_out, float* score, tc::Rows rows,
                             cudaStream_t st) {
  if (rows.m_cap <= 0) return TRK_OK;
  auto kern = gf::gnn_fused_kernel<MODE>;
  TRK_TRY(ensure_smem(ctx, kern, gf::kSmemFused));
  CUtensorMap tw1, tw2, te, test;
  TRK_TRY(make_tmap(ctx, &tw1, L1.w_bf16, gf::kH, 3 * gf::kH, 3 * gf::kH, 64));
  TRK_TRY(make_tmap(ctx, &tw2, L2.w_bf16, gf::kH, gf::kH, gf::kH, 64));
  TRK_TRY(make_tmap(ctx, &te, E, e_rows, gf::kH, gf::kH, 128));
  TRK_TRY(make_tmap(ctx, &test, E, e_rows, gf::kH, gf::kH, 32));
  gf::FusedParams p{X, ldx, src, dst, {}, {}, ctx->cfg.gnn_layernorm, w_out, b_out, score, nullptr};
  fill_bias(p, L1, L2);
  const int64_t ptiles = ceil_div(rows.m_cap, 2 * gf::kTileRows);
  const unsigned grid = 2u * (unsigned)std::min<int64_t>(ptiles, ctx->sm_count / 2);
  TRK_LAUNCH(ctx, kern, grid, gf::kFusedThreads, gf::kSmemFused, st, tw1, tw2, te, test, rows, p);
  return TRK_OK;
}

// Fused node update of S4 (gnn_fused.cuh, kNode), H = 128: X[:, 0:H] <- X[:, 0:H] + LNR(W2 LNR(W1 X + b1) + b2) in place.
trk_status launch_node_fused(trk_ctx* ctx, bf16* X, int64_t x_rows, const DevLinear& L1, const DevLinear& L2, tc::Rows rows,
                             cudaStream_t st) {
  if (rows.m_cap <= 0) return TRK_OK;
  auto kern = gf::gnn_fused_kernel<gf::kNode>;
  TRK_TRY(ensure_smem(ctx, kern, gf::kSmemFused));
  CUtensorMap tw1, tw2, tx, txst;
  TRK_TRY(make_tmap(ctx, &tw1, L1.w_bf16, gf::kH, 3 * gf::kH, 3 * gf::kH, 64));
  TRK_TRY(make_tmap(ctx, &tw2, L2.w_bf16, gf::kH, gf::kH, gf::kH, 64));
  TRK_TRY(make_tmap(ctx, &tx, X, x_rows, 3 * gf::kH, 3 * gf::kH, 128));
  TRK_TRY(make_tmap(ctx, &txst, X, x_rows, gf::kH, 3 * gf::kH, 32));
  gf::FusedParams p{X, 3 * gf::kH, nullptr, nullptr, {}, {}, ctx->cfg.gnn_layernorm, nullptr, 0.f, nullptr, nullptr};
  fill_bias(p, L1, L2);
  const int64_t ptiles = ceil_div(rows.m_cap, 2 * gf::kTileRows);
  const unsigned grid = 2u * (unsigned)std::min<int64_t>(ptiles, ctx->sm_count / 2);
  TRK_LAUNCH(ctx, kern, grid, gf::kFusedThreads, gf::kSmemFused, st, tw1, tw2, tx, txst, rows, p);
  return TRK_OK;
}

// Fused encoder of S4 (gnn_fused.cuh, kEncode), H = 128: out[m] = LNR(W2 LNR(W1 f_m + b1) + b2), f_m = the 3 features of node m
// (src == nullptr) or the 4 edge features of (src[m], dst[m]); w1p is the [H][64] hi/lo copy of W1; out bf16 with row stride ldo.
trk_status launch_encoder_fused(trk_ctx* ctx, const float* hits, const int32_t* src, const int32_t* dst, const bf16* w1p, const DevLinear& L1,
                                const DevLinear& L2, bf16* out, int64_t out_rows, int64_t ldo, tc::Rows rows, cudaStream_t st) {
  if (rows.m_cap <= 0) return TRK_OK;
  auto kern = gf::gnn_fused_kernel<gf::kEncode>;
  TRK_TRY(ensure_smem(ctx, kern, gf::kSmemFused));
  CUtensorMap tw1, tw2, tout;
  TRK_TRY(make_tmap(ctx, &tw1, w1p, gf::kH, 64, 64, 64));
  TRK_TRY(make_tmap(ctx, &tw2, L2.w_bf16, gf::kH, gf::kH, gf::kH, 64));
  TRK_TRY(make_tmap(ctx, &tout, out, out_rows, gf::kH, ldo, 32));
  gf::FusedParams p{nullptr, 0, src, dst, {}, {}, ctx->cfg.gnn_layernorm, nullptr, 0.f, nullptr, hits};
  fill_bias(p, L1, L2);
  const int64_t ptiles = ceil_div(rows.m_cap, 2 * gf::kTileRows);
  const unsigned grid = 2u * (unsigned)std::min<int64_t>(ptiles, ctx->sm_count / 2);
  TRK_LAUNCH(ctx, kern, grid, gf::kFusedThreads, gf::kSmemFused, st, tw1, tw2, tout, tout, rows, p);
  return TRK_OK;
}

// ---------------------------------------------------------------- small SIMT kernels
__device__ __forceinline__ int64_t rows_of(const int32_t* m_dev, int64_t m_off, int64_t m_cap) {
  if (!m_dev) return m_cap;
  int64_t m = (int64_t)*m_dev - m_off;
  return m < 0 ? 0 : (m > m_cap ? m_cap : m);
}

// S1 first layer: out[m][n] = bf16(relu(W[n][0..3) . x[m] + b[n])).  A thread owns 8 columns (its 24 weights and 8 biases stay
// in registers) and walks down the rows of its block, so a row costs 3 broadcast loads, 24 FMAs and one 16-byte store:
// the kernel runs at the HBM write rate of the activation instead of re-reading W from L1 for every row.
constexpr int kFirstLayerRowsPerBlock = 64;
__global__ void __launch_bounds__(256)
embed_first_layer_kernel(const float* __restrict__ hits, const float* __restrict__ W, const float* __restrict__ b,
                         bf16* __restrict__ out, int64_t M, int N) {
  TRK_GRID_DEP_WAIT();
  const int groups = N / 8;                       // 16-byte column groups per row
  const int lanes_r = blockDim.x / groups;        // rows in flight per pass (host guarantees groups <= blockDim.x)
  const int g = threadIdx.x % groups, rl = threadIdx.x / groups;
  if (rl >= lanes_r) return;
  float w[8][3], bb[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const float* wp = W + (int64_t)(g * 8 + j) * 3;
    w[j][0] = wp[0]; w[j][1] = wp[1]; w[j][2] = wp[2];
    bb[j] = b[g * 8 + j];
  }
  const int64_t row0 = (int64_t)blockIdx.x * kFirstLayerRowsPerBlock;
  const int64_t row1 = min(row0 + kFirstLayerRowsPerBlock, M);
  for (int64_t row = row0 + rl; row < row1; row += lanes_r) {
    const float x0 = __ldg(hits + row * 3), x1 = __ldg(hits + row * 3 + 1), x2 = __ldg(hits + row * 3 + 2);
    float v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = fmaxf(fmaf(w[j][2], x2, fmaf(w[j][1], x1, fmaf(w[j][0], x0, bb[j]))), 0.f);
    *reinterpret_cast<uint4*>(out + row * N + g * 8) =
        make_uint4(tc::pack_bf16(v[0], v[1]), tc::pack_bf16(v[2], v[3]), tc::pack_bf16(v[4], v[5]), tc::pack_bf16(v[6], v[7]));
  }
}

// S3 input rows: out[m][0..2u) = bf16([feat[src] ; feat[dst]]); 8 columns per thread, 2^cpr_log2 threads per row cover the
// 16-byte chunks that hold data.  Columns [2u, 64) are the zero padding of K: the buffer is zeroed once in trk_create and
// nothing ever writes there.  Rows beyond M keep stale (finite) values; no result of theirs is ever read.
__global__ void filter_gather_kernel(const float* __restrict__ feat, int u, int cpr_log2, const int32_t* __restrict__ src,
                                     const int32_t* __restrict__ dst, const int32_t* __restrict__ m_dev, int64_t m_off, int64_t m_cap,
                                     bf16* __restrict__ out) {
  TRK_GRID_DEP_WAIT();
  const int64_t M = rows_of(m_dev, m_off, m_cap);
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t row = i >> cpr_log2;
  const int c0 = (int)(i & ((1 << cpr_log2) - 1)) * 8;
  if (row >= M || c0 >= 2 * u) return;
  float v[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) v[j] = 0.f;
  {
    const int64_t s = src[m_off + row], d = dst[m_off + row];
    if ((u & 3) == 0 && (reinterpret_cast<uintptr_t>(feat) & 15) == 0) {
      // rows of feat are 16-byte aligned: the thread's eight columns are two float4 pieces, each from one endpoint
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int c = c0 + 4 * h;
        if (c < 2 * u) {
          const float4 x = __ldg(reinterpret_cast<const float4*>(c < u ? feat + s * u + c : feat + d * u + (c - u)));
          v[4 * h] = x.x; v[4 * h + 1] = x.y; v[4 * h + 2] = x.z; v[4 * h + 3] = x.w;
        }
      }
    } else {
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int c = c0 + j;
        if (c < u) v[j] = feat[s * u + c];
        else if (c < 2 * u) v[j] = feat[d * u + (c - u)];
      }
    }
  }
  *reinterpret_cast<uint4*>(out + row * 64 + c0) =
      make_uint4(tc::pack_bf16(v[0], v[1]), tc::pack_bf16(v[2], v[3]), tc::pack_bf16(v[4], v[5]), tc::pack_bf16(v[6], v[7]));
}

__global__ void filter_finish_kernel(const float* __restrict__ partial, int n_tiles, float b_last, const int32_t* __restrict__ m_dev,
                                     int64_t m_off, int64_t m_cap, float* __restrict__ score) {
  TRK_GRID_DEP_WAIT();
  const int64_t M = rows_of(m_dev, m_off, m_cap);
  const int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (row >= M) return;
  float s = b_last;
  for (int t = 0; t < n_tiles; ++t) s += partial[row * n_tiles + t];
  score[m_off + row] = 1.f / (1.f + __expf(-s));
}

// First GNN encoder layers (K = 3 node features or K = 4 edge features): out[m] = bf16(ReLU(LayerNorm(W x + b))).
// A warp takes 32 rows at a time: every lane prepares the input of one row (EDGE: the edge features of (src[m], dst[m]),
// two asinhf per lane instead of per warp), then the warp walks over the 32 rows with shuffles; a lane owns the H/32
// adjacent columns 'per * lane ..' (weights in registers) so one row leaves as one coalesced 2H-byte store.
template <bool EDGE, int PER>
__global__ void __launch_bounds__(256)
encoder_first_layer_kernel(const float* __restrict__ hits, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
                           const float* __restrict__ W, const float* __restrict__ b, int use_ln,
                           const int32_t* __restrict__ m_dev, int64_t m_cap, bf16* __restrict__ out) {
  TRK_GRID_DEP_WAIT();
  constexpr int K = EDGE ? 4 : 3;
  constexpr int H = PER * 32;
  const int64_t M = rows_of(m_dev, 0, m_cap);
  const int lane = threadIdx.x & 31;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  float w[PER][K], bb[PER];
#pragma unroll
  for (int j = 0; j < PER; ++j) {
    const int c = lane * PER + j;
#pragma unroll
    for (int k = 0; k < K; ++k) w[j][k] = W[c * K + k];
    bb[j] = b[c];
  }
  for (int64_t base = warp * 32; base < M; base += n_warps * 32) {
    const int64_t mine = base + lane;
    float x[4] = {0.f, 0.f, 0.f, 0.f};
    if (mine < M) {
      if (EDGE) {
        const float4 a = edge_features(hits, src[mine], dst[mine]);
        x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w;
      } else {
        x[0] = hits[mine * 3]; x[1] = hits[mine * 3 + 1]; x[2] = hits[mine * 3 + 2];
      }
    }
    const int cnt = (int)min((int64_t)32, M - base);
    for (int r = 0; r < cnt; ++r) {
      float xr[K];
#pragma unroll
      for (int k = 0; k < K; ++k) xr[k] = __shfl_sync(0xffffffffu, x[k], r);
      float v[PER];
      float s = 0.f;
#pragma unroll
      for (int j = 0; j < PER; ++j) {
        float a = bb[j];
#pragma unroll
        for (int k = 0; k < K; ++k) a = fmaf(w[j][k], xr[k], a);
        v[j] = a;
        s += a;
      }
      float mean = 0.f, rstd = 1.f;
      if (use_ln) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        mean = s * (1.f / H);
        float q = 0.f;
#pragma unroll
        for (int j = 0; j < PER; ++j) { const float d = v[j] - mean; q = fmaf(d, d, q); }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
        rstd = rsqrtf(q * (1.f / H) + 1e-5f);
      }
#pragma unroll
      for (int j = 0; j < PER; ++j) v[j] = fmaxf((v[j] - mean) * rstd, 0.f);
      bf16* o = out + (base + r) * H + lane * PER;
      if constexpr (PER == 4) {
        *reinterpret_cast<uint2*>(o) = make_uint2(tc::pack_bf16(v[0], v[1]), tc::pack_bf16(v[2], v[3]));
      } else {
        *reinterpret_cast<uint32_t*>(o) = tc::pack_bf16(v[0], v[1]);
      }
    }
  }
}

template <bool EDGE>
trk_status launch_encoder_first(trk_ctx* ctx, const float* hits, const int32_t* src, const int32_t* dst, const DevLinear& L, int H,
                                int use_ln, const int32_t* m_dev, int64_t m_cap, bf16* out, cudaStream_t st) {
  if (m_cap <= 0) return TRK_OK;
  const unsigned blocks = (unsigned)std::min<int64_t>(ceil_div(m_cap, 32 * 8), (int64_t)ctx->sm_count * 8);
  if (H == 128) {
    TRK_LAUNCH(ctx, (encoder_first_layer_kernel<EDGE, 4>), blocks, 256, 0, st, hits, src, dst, L.w_f32, L.b_f32, use_ln, m_dev, m_cap, out);
  } else {
    TRK_LAUNCH(ctx, (encoder_first_layer_kernel<EDGE, 2>), blocks, 256, 0, st, hits, src, dst, L.w_f32, L.b_f32, use_ln, m_dev, m_cap, out);
  }
  return TRK_OK;
}

}  // namespace

// ---------------------------------------------------------------- S1
trk_status embed_forward_bf16(trk_ctx* ctx, const float* hits, int64_t n, float* emb, cudaStream_t st) {
  const auto& L = ctx->embed.layers;
  const int nl = (int)L.size();
  bf16* bufs[2] = {(bf16*)ctx->act0, (bf16*)ctx->act1};
  const int w0 = L[0].out;
  if (w0 / 8 > 256) return fail(ctx, TRK_ERR_SHAPE, "TRK_BF16: the first embedding layer is limited to 2048 outputs");
  TRK_LAUNCH(ctx, embed_first_layer_kernel, (unsigned)ceil_div(n, kFirstLayerRowsPerBlock), 256, 0, st, hits, L[0].w_f32, L[0].b_f32,
             bufs[0], n, w0);
  int cur = 0;
  tc::Rows rows{nullptr, 0, n};
  for (int l = 1; l < nl - 1; ++l) {
    TRK_TRY(gemm_bias_act(ctx, bufs[cur], ctx->act_rows, L[l].in_pad, L[l], bufs[cur ^ 1], ctx->act_rows, L[l].out_pad, 1, rows, st));
    cur ^= 1;
  }
  const DevLinear& last = L[nl - 1];
  tc::EpiBiasF32Narrow::Params ep{last.b_f32, emb, ctx->d_e, ctx->d_e};
  return launch_gemm<16, tc::EpiBiasF32Narrow>(ctx, bufs[cur], ctx->act_rows, last.in_pad, last.in_pad, last.w_bf16, 16, rows, ep, st);
}

// ---------------------------------------------------------------- S3
// All layers of the filter MLP in one persistent CTA-pair kernel (filter_fused.cuh); activations stay in L2-resident scratch.
static trk_status filter_forward_fused(trk_ctx* ctx, const float* feat, const int32_t* src, const int32_t* dst,
                                       const int32_t* n_edges_dev, int64_t n_edges_cap, float* score, cudaStream_t st) {
  const auto& L = ctx->filter.layers;
  const int W = L[0].out_pad;
  const int n_pairs_max = ctx->sm_count / 2;
  const int64_t s_rows = (int64_t)n_pairs_max * 256;
  auto kern = ff::filter_mlp_kernel;
  TRK_TRY(ensure_smem(ctx, kern, ff::kSmemFilter));
  CUtensorMap ts1, ts2, tw1, tw2, tw3, ts1st, ts2st;
  TRK_TRY(make_tmap(ctx, &ts1, ctx->filter_s1, s_rows, W, W, 128));
  TRK_TRY(make_tmap(ctx, &ts2, ctx->filter_s2, s_rows, W, W, 128));
  TRK_TRY(make_tmap(ctx, &tw1, ctx->filter_w1_pad, W, 64, 64, 128));
  TRK_TRY(make_tmap(ctx, &tw2, L[1].w_bf16, W, W, W, 128));
  TRK_TRY(make_tmap(ctx, &tw3, L[2].w_bf16, W, W, W, 128));
  TRK_TRY(make_tmap(ctx, &ts1st, ctx->filter_s1, s_rows, W, W, 32));
  TRK_TRY(make_tmap(ctx, &ts2st, ctx->filter_s2, s_rows, W, W, 32));
  ff::FilterParams p{feat, src, dst, ctx->filter_u, L[0].b_f32, L[1].b_f32, L[2].b_f32, L[3].w_f32, ctx->filter_b_last, score, W};
  const tc::Rows rows{n_edges_dev, 0, n_edges_cap};
  // "filter_max_pairs" (trk_set_option): fewer CTA pairs than the device holds leave SMs to the other stages of another
  // model instance (a pair walks row blocks pair, pair + n_pairs, ...: the scores do not depend on the number of pairs)
  const int64_t pair_cap = ctx->knobs[kKnobFilterPairs] > 0 ? std::min<int64_t>(ctx->knobs[kKnobFilterPairs], n_pairs_max) : n_pairs_max;
  const unsigned grid = 2u * (unsigned)std::min<int64_t>(ceil_div(n_edges_cap, 256), pair_cap);
  // trk_profile_kernel_ms: one CUDA-event pair around the launch
  const bool kprof = ctx->profiling && n_edges_dev == &ctx->counts[0] && ctx->kprof_ev.size() >= 2;
  if (kprof) {
    ctx->kprof_n = 1;
    TRK_CUDA(ctx, cudaEventRecord(ctx->kprof_ev[0], st));
  }
  TRK_LAUNCH(ctx, kern, grid, ff::kThreadsFilter, ff::kSmemFilter, st, ts1, ts2, tw1, tw2, tw3, ts1st, ts2st, rows, p);
  if (kprof) TRK_CUDA(ctx, cudaEventRecord(ctx->kprof_ev[1], st));
  return TRK_OK;
}

trk_status filter_forward_bf16(trk_ctx* ctx, const float* feat, const int32_t* src, const int32_t* dst,
                               const int32_t* n_edges_dev, int64_t n_edges_cap, float* score, cudaStream_t st) {
  if (ctx->filter_fusable && ctx->knobs[kKnobFilterFused] != 0)
    return filter_forward_fused(ctx, feat, src, dst, n_edges_dev, n_edges_cap, score, st);
  const auto& L = ctx->filter.layers;
  const int nl = (int)L.size();
  const int u = ctx->filter_u;
  bf16* bufs[2] = {(bf16*)ctx->act0, (bf16*)ctx->act1};
  bf16* gin = (bf16*)ctx->act_in;
  for (int64_t off = 0; off < n_edges_cap; off += ctx->filter_chunk) {
    const int64_t cap = std::min<int64_t>(ctx->filter_chunk, n_edges_cap - off);
    tc::Rows rows{n_edges_dev, off, cap};
    // first layer with 256-column tiles: its A operand is gathered inside the GEMM (gemm_tc.cuh GATHER_A)
    int cpr_log2 = 0;                                   // threads per gathered row: the 16-byte chunks that hold data, rounded up to 2^k
    while ((8 << cpr_log2) < 2 * u) ++cpr_log2;
    const bool fuse_gather = nl >= 3 && pick_bn(L[0].out_pad) == 256 && ctx->knobs[kKnobEpiSplit] >= 2;
    const tc::AGather ag{feat, src, dst, u};
    if (!fuse_gather)
      TRK_LAUNCH(ctx, filter_gather_kernel, (unsigned)ceil_div(cap << cpr_log2, 256), 256, 0, st, feat, u, cpr_log2, src, dst, n_edges_dev,
                 off, cap, gin);
    const bf16* in = gin;
    int64_t in_rows = ctx->filter_chunk;
    int cur = 0;
    int n_tiles = 1;
    for (int l = 0; l < nl - 1; ++l) {
      // layer 0 reads the gathered rows (K padded to 64) against the K-padded copy of W1
      DevLinear Ll = L[l];
      if (l == 0) { Ll.w_bf16 = ctx->filter_w1_pad; Ll.in_pad = 64; }
      const int64_t lda = l == 0 ? 64 : Ll.in_pad;
      // trk_profile_kernel_ms: one CUDA-event pair around every hidden-layer GEMM launch with K >= 256
      const bool kprof = ctx->profiling && n_edges_dev == &ctx->counts[0] && Ll.in_pad >= 256 &&
                         (size_t)ctx->kprof_n * 2 + 2 <= ctx->kprof_ev.size();   // the event pairs are created by trk_profile_enable
      cudaEvent_t k0 = nullptr, k1 = nullptr;
      if (kprof) {
        k0 = ctx->kprof_ev[(size_t)ctx->kprof_n * 2];
        k1 = ctx->kprof_ev[(size_t)ctx->kprof_n * 2 + 1];
        ++ctx->kprof_n;
        TRK_CUDA(ctx, cudaEventRecord(k0, st));
      }
      if (l == nl - 2) {
        TRK_TRY(gemm_relu_dot(ctx, in, in_rows, lda, Ll, L[nl - 1].w_f32, ctx->partial, &n_tiles, rows, st));
      } else {
        TRK_TRY(gemm_bias_act(ctx, in, in_rows, lda, Ll, bufs[cur], ctx->act_rows, Ll.out_pad, 1, rows, st,
                              l == 0 && fuse_gather ? &ag : nullptr));
        in = bufs[cur];
        in_rows = ctx->act_rows;
        cur ^= 1;
      }
      if (kprof) TRK_CUDA(ctx, cudaEventRecord(k1, st));
    }
    TRK_LAUNCH(ctx, filter_finish_kernel, (unsigned)ceil_div(cap, 256), 256, 0, st, ctx->partial, n_tiles, ctx->filter_b_last,
               n_edges_dev, off, cap, score);
  }
  return TRK_OK;
}

// ---------------------------------------------------------------- S4
trk_status gnn_forward_bf16(trk_ctx* ctx, const float* hits, int64_t n, const int32_t* src, const int32_t* dst,
                            const int32_t* n_edges_dev, int64_t n_edges_cap, float* score, cudaStream_t st) {
  const int H = ctx->H;
  const int ln = ctx->cfg.gnn_layernorm;
  bf16* X = (bf16*)ctx->X;      // [n][3H]: h | m_in | m_out
  bf16* E = (bf16*)ctx->E;      // [E][H]
  bf16* T1 = (bf16*)ctx->T1;    // [max(n,E)][H]
  float* PAB = ctx->PAB;        // [n][2H]
  const int64_t x_rows = ctx->cfg.max_hits, e_rows = ctx->cfg.max_kept_edges, t_rows = std::max(x_rows, e_rows);
  tc::Rows nrows{nullptr, 0, n};
  tc::Rows erows{n_edges_dev, 0, n_edges_cap};
  TRK_TRY(build_gnn_csr(ctx, hits, src, dst, n_edges_dev, n_edges_cap, n, st));

  const bool fused = H == gf::kH && ctx->knobs[kKnobGnnFused] != 0;
  if (fused) {
    // both encoders as fused two-layer kernels: the K = 3 / 4 first layer on the tensor core from hi/lo-split features
    TRK_TRY(launch_encoder_fused(ctx, hits, nullptr, nullptr, ctx->node_enc_w1p, ctx->node_enc.layers[0], ctx->node_enc.layers[1], X, x_rows,
                                 3 * H, nrows, st));
    if (n_edges_cap > 0)
      TRK_TRY(launch_encoder_fused(ctx, hits, src, dst, ctx->edge_enc_w1p, ctx->edge_enc.layers[0], ctx->edge_enc.layers[1], E, e_rows, H,
                                   erows, st));
  } else {
  // node encoder: 3 -> H (SIMT) -> H (GEMM, LNR) -> X[:, 0:H]
  TRK_TRY(launch_encoder_first<false>(ctx, hits, nullptr, nullptr, ctx->node_enc.layers[0], H, ln, nullptr, n, T1, st));
  {
    tc::EpiRowLn::Params ep{ctx->node_enc.layers[1].b_f32, nullptr, nullptr, nullptr, ln, nullptr, 0, X, 3 * H, nullptr, 0.f, nullptr};
    TRK_TRY(gemm_row_ln(ctx, T1, t_rows, H, H, ctx->node_enc.layers[1].w_bf16, ep, nrows, st));
  }
  if (n_edges_cap > 0) {
    // edge encoder: 4 -> H (SIMT on the fly features) -> H (GEMM, LNR) -> E
    TRK_TRY(launch_encoder_first<true>(ctx, hits, src, dst, ctx->edge_enc.layers[0], H, ln, n_edges_dev, n_edges_cap, T1, st));
    tc::EpiRowLn::Params ep{ctx->edge_enc.layers[1].b_f32, nullptr, nullptr, nullptr, ln, nullptr, 0, E, H, nullptr, 0.f, nullptr};
    TRK_TRY(gemm_row_ln(ctx, T1, t_rows, H, H, ctx->edge_enc.layers[1].w_bf16, ep, erows, st));
  }
  }
  for (int t = 0; t < ctx->cfg.gnn_iters; ++t) {
    if (n_edges_cap > 0 && fused) {
      TRK_TRY(launch_edge_fused<gf::kUpdate>(ctx, X, 3 * H, E, e_rows, src, dst, ctx->edge_net.layers[0], ctx->edge_net.layers[1], nullptr,
                                             0.f, nullptr, erows, st));
    } else if (n_edges_cap > 0) {
      // PA|PB = h [Wa ; Wb]^T per node, then e <- e + LNR(W2 LNR(Wc e + PA[src] + PB[dst] + b1) + b2)
      TRK_TRY(gemm_store_f32(ctx, X, x_rows, 3 * H, H, ctx->edge_net_wab, 2 * H, PAB, nrows, st));
      tc::EpiRowLn::Params e1{ctx->edge_net.layers[0].b_f32, PAB, src, dst, ln, nullptr, 0, T1, H, nullptr, 0.f, nullptr};
      TRK_TRY(gemm_row_ln(ctx, E, e_rows, H, H, ctx->edge_net_wc, e1, erows, st));
      tc::EpiRowLn::Params e2{ctx->edge_net.layers[1].b_f32, nullptr, nullptr, nullptr, ln, E, H, E, H, nullptr, 0.f, nullptr};
      TRK_TRY(gemm_row_ln(ctx, T1, t_rows, H, H, ctx->edge_net.layers[1].w_bf16, e2, erows, st));
    }
    TRK_TRY(segment_sums(ctx, E, true, n, X, st));
    // h <- h + LNR(W2 LNR(W1 [h ; m_in ; m_out] + b1) + b2): X is the concatenation already
    if (fused) {
      TRK_TRY(launch_node_fused(ctx, X, x_rows, ctx->node_net.layers[0], ctx->node_net.layers[1], nrows, st));
      continue;
    }
    tc::EpiRowLn::Params n1{ctx->node_net.layers[0].b_f32, nullptr, nullptr, nullptr, ln, nullptr, 0, T1, H, nullptr, 0.f, nullptr};
    TRK_TRY(gemm_row_ln(ctx, X, x_rows, 3 * H, 3 * H, ctx->node_net.layers[0].w_bf16, n1, nrows, st));
    tc::EpiRowLn::Params n2{ctx->node_net.layers[1].b_f32, nullptr, nullptr, nullptr, ln, X, 3 * H, X, 3 * H, nullptr, 0.f, nullptr};
    TRK_TRY(gemm_row_ln(ctx, T1, t_rows, H, H, ctx->node_net.layers[1].w_bf16, n2, nrows, st));
  }
  if (n_edges_cap > 0 && fused) {
    // the decoder's second layer is Linear(H -> 1): its fp32 weights are w_out; the W2 operand of the kernel is unused in this mode
    TRK_TRY(launch_edge_fused<gf::kDecode>(ctx, X, 3 * H, E, e_rows, src, dst, ctx->edge_dec.layers[0], ctx->edge_net.layers[1],
                                           ctx->edge_dec.layers[1].w_f32, ctx->edge_dec_b_last, score, erows, st));
  } else if (n_edges_cap > 0) {
    TRK_TRY(gemm_store_f32(ctx, X, x_rows, 3 * H, H, ctx->edge_dec_wab, 2 * H, PAB, nrows, st));
    tc::EpiRowLn::Params d1{ctx->edge_dec.layers[0].b_f32, PAB, src, dst, ln, nullptr, 0, nullptr, 0,
                            ctx->edge_dec.layers[1].w_f32, ctx->edge_dec_b_last, score};
    TRK_TRY(gemm_row_ln(ctx, E, e_rows, H, H, ctx->edge_dec_wc, d1, erows, st));
  }
  return TRK_OK;
}

// ---------------------------------------------------------------- test hook
trk_status gemm_bf16_hook(trk_ctx* ctx, const void* a, const void* w, const float* bias, void* out, int64_t m, int n, int k, int relu,
                          cudaStream_t st) {
  DevLinear L;
  L.in = L.in_pad = k;
  L.out = L.out_pad = n;
  L.w_bf16 = (bf16*)w;
  L.b_f32 = const_cast<float*>(bias);
  return gemm_bias_act(ctx, (const bf16*)a, m, k, L, (bf16*)out, m, n, relu, tc::Rows{nullptr, 0, m}, st);
}

}  // namespace trk

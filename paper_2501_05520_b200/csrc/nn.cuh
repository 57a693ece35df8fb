// S1 / S3 / S4 entry points of the two precisions and the small device helpers they share.
#pragma once
#include "common.cuh"

namespace trk {

// Edge features of S4: (dr, dphi wrapped to (-1,1], dz, deta), deta = asinh(z_d/r_d) - asinh(z_s/r_s).
__device__ __forceinline__ float4 edge_features(const float* __restrict__ hits, int s, int d) {
  const float rs = hits[3 * (int64_t)s], ps = hits[3 * (int64_t)s + 1], zs = hits[3 * (int64_t)s + 2];
  const float rd = hits[3 * (int64_t)d], pd = hits[3 * (int64_t)d + 1], zd = hits[3 * (int64_t)d + 2];
  float dphi = pd - ps;
  if (dphi > 1.f) dphi -= 2.f;
  if (dphi <= -1.f) dphi += 2.f;
  return make_float4(rd - rs, dphi, zd - zs, asinhf(zd / rd) - asinhf(zs / rs));
}

__global__ void edge_features_kernel(const float* __restrict__ hits, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
                                     const int32_t* __restrict__ m_dev, int64_t m_cap, float4* __restrict__ out);

trk_status embed_forward_fp32(trk_ctx* ctx, const float* hits, int64_t n, float* emb, cudaStream_t st);
trk_status filter_forward_fp32(trk_ctx* ctx, const float* feat, const int32_t* src, const int32_t* dst,
                               const int32_t* n_edges_dev, int64_t n_edges_cap, float* score, cudaStream_t st);
trk_status gnn_forward_fp32(trk_ctx* ctx, const float* hits, int64_t n, const int32_t* src, const int32_t* dst,
                            const int32_t* n_edges_dev, int64_t n_edges_cap, float* score, cudaStream_t st);

trk_status embed_forward_bf16(trk_ctx* ctx, const float* hits, int64_t n, float* emb, cudaStream_t st);
trk_status filter_forward_bf16(trk_ctx* ctx, const float* feat, const int32_t* src, const int32_t* dst,
                               const int32_t* n_edges_dev, int64_t n_edges_cap, float* score, cudaStream_t st);
trk_status gnn_forward_bf16(trk_ctx* ctx, const float* hits, int64_t n, const int32_t* src, const int32_t* dst,
                            const int32_t* n_edges_dev, int64_t n_edges_cap, float* score, cudaStream_t st);

}  // namespace trk

// S4 graph bookkeeping and aggregation (graph.cu).
#pragma once
#include "common.cuh"

namespace trk {

// Builds out_rowptr (edges are src-sorted) and the dst-sorted permutation in_rowptr/in_perm.
trk_status build_gnn_csr(trk_ctx* ctx, const float* hits, const int32_t* src, const int32_t* dst, const int32_t* n_edges_dev, int64_t n_edges_cap,
                         int64_t n_nodes, cudaStream_t st);
// X[v][H:2H] = sum of E rows over in-edges of v, X[v][2H:3H] = over out-edges (fp32 accumulation).
trk_status segment_sums(trk_ctx* ctx, const void* E, bool bf16, int64_t n_nodes, void* X, cudaStream_t st);

}  // namespace trk

// Graph bookkeeping for S4 message passing: the kept edge list is sorted by
// (src, dst) and static over the T iterations, so both aggregations
//     m_out_v = sum_{k: src(k)=v} e_k        m_in_v = sum_{k: dst(k)=v} e_k
// are atomic-free segmented sums over a CSR built once per call: out-edges are already
// contiguous; in-edges go through a dst-sorted permutation whose segments are ordered by edge
// index, so the fp32 summation order is fixed and results are run-to-run identical
// (PAPER.md line 164 identity check; reading C-14: fp32 accumulation).
#include "common.cuh"
#include "graph.cuh"

namespace trk {
namespace {

__device__ __forceinline__ int64_t dev_count(const int32_t* n_dev, int64_t cap) {
  return n_dev ? min((int64_t)max(*n_dev, 0), cap) : cap;
}

// rowptr[v] = first k with key[k] >= v, for sorted keys; rowptr[n_nodes] = n_edges.
__global__ void rowptr_from_sorted_kernel(const int32_t* __restrict__ key, const int32_t* __restrict__ n_dev, int64_t cap,
                                          int32_t* __restrict__ rowptr, int64_t n_nodes) {
  TRK_GRID_DEP_WAIT();
  const int64_t n_edges = dev_count(n_dev, cap);
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k > n_edges) return;
  const int64_t prev = k == 0 ? -1 : key[k - 1];
  const int64_t cur = k == n_edges ? n_nodes : key[k];
  for (int64_t v = prev + 1; v <= cur; ++v) rowptr[v] = (int32_t)k;
}

__global__ void count_keys_kernel(const int32_t* __restrict__ key, const int32_t* __restrict__ n_dev, int64_t cap,
                                  int32_t* __restrict__ count) {
  TRK_GRID_DEP_WAIT();
  const int64_t n_edges = dev_count(n_dev, cap);
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n_edges) atomicAdd(&count[key[k]], 1);
}

__global__ void place_keys_kernel(const int32_t* __restrict__ key, const int32_t* __restrict__ n_dev, int64_t cap,
                                  const int32_t* __restrict__ rowptr, int32_t* __restrict__ fill, int32_t* __restrict__ perm) {
  TRK_GRID_DEP_WAIT();
  const int64_t n_edges = dev_count(n_dev, cap);
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n_edges) {
    const int v = key[k];
    perm[rowptr[v] + atomicSub(&fill[v], 1) - 1] = (int32_t)k;   // fill still holds the segment's count: back to front
  }
}

// Each segment of perm is put in ascending edge order (place_keys_kernel fills a segment in the arbitrary order of its atomics;
// the order of a segmented sum must not depend on it).  One warp per node: the entries of a segment are distinct, so the rank of
// one is the number of smaller ones -- 32 entries per pass live in registers and are compared through shuffles.  Segments longer
// than kSortMaxLen (a node with that many in-edges does not occur in tracking graphs) are sorted in place by a bitonic network.
constexpr int kSortChunks = 8;
constexpr int kSortMaxLen = 32 * kSortChunks;
__global__ void __launch_bounds__(256) sort_segments_kernel(const int32_t* __restrict__ rowptr, int32_t* __restrict__ perm, int64_t n_nodes) {
  TRK_GRID_DEP_WAIT();
  const int lane = threadIdx.x & 31;
  const int64_t v = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (v >= n_nodes) return;
  const int b = rowptr[v], len = rowptr[v + 1] - b;
  if (len <= 1) return;
  if (len <= 32) {
    const int x = lane < len ? perm[b + lane] : 0x7fffffff;
    int rank = 0;
    for (int j = 0; j < len; ++j) rank += __shfl_sync(0xffffffffu, x, j) < x ? 1 : 0;
    __syncwarp();
    if (lane < len) perm[b + rank] = x;
    return;
  }
  if (len <= kSortMaxLen) {
    int x[kSortChunks], rank[kSortChunks];
#pragma unroll
    for (int c = 0; c < kSortChunks; ++c) {
      x[c] = c * 32 + lane < len ? perm[b + c * 32 + lane] : 0x7fffffff;
      rank[c] = 0;
    }
#pragma unroll
    for (int d = 0; d < kSortChunks; ++d) {
      if (d * 32 >= len) break;
      for (int j = 0; j < 32; ++j) {
        const int y = __shfl_sync(0xffffffffu, x[d], j);
#pragma unroll
        for (int c = 0; c < kSortChunks; ++c) rank[c] += y < x[c] ? 1 : 0;
      }
    }
    __syncwarp();
#pragma unroll
    for (int c = 0; c < kSortChunks; ++c)
      if (c * 32 + lane < len) perm[b + rank[c]] = x[c];
    return;
  }
  // Longer segments (a hub): an in-place sorting network over the warp.  Bitonic sort with ascending-only merges -- the first
  // step of a merge of size k pairs i with i ^ (k - 1), the others i with i ^ j -- so entries beyond len, which count as +inf,
  // would stay where they are: a pair that reaches past the segment is skipped.  O(len log^2 len / 32) steps per lane.
  int32_t* seg = perm + b;
  int p2 = 1;
  while (p2 < len) p2 <<= 1;
  for (int k = 2; k <= p2; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      const bool flip = j == (k >> 1);
      for (int t = lane; t < (p2 >> 1); t += 32) {
        const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));      // the t-th index with bit j clear
        const int l = flip ? (i ^ (k - 1)) : (i | j);
        if (l < len) {
          const int32_t x = seg[i], y = seg[l];
          if (x > y) { seg[i] = y; seg[l] = x; }
        }
      }
      __syncwarp();
    }
  }
}

template <typename T>
__device__ __forceinline__ float4 load4(const T* p);
template <>
__device__ __forceinline__ float4 load4<float>(const float* p) { return *reinterpret_cast<const float4*>(p); }
template <>
__device__ __forceinline__ float4 load4<__nv_bfloat16>(const __nv_bfloat16* p) {
  const uint2 u = *reinterpret_cast<const uint2*>(p);
  const __nv_bfloat162 a = *reinterpret_cast<const __nv_bfloat162*>(&u.x);
  const __nv_bfloat162 b = *reinterpret_cast<const __nv_bfloat162*>(&u.y);
  return make_float4(__low2float(a), __high2float(a), __low2float(b), __high2float(b));
}
template <typename T>
__device__ __forceinline__ void store4(T* p, float4 v);
template <>
__device__ __forceinline__ void store4<float>(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }
template <>
__device__ __forceinline__ void store4<__nv_bfloat16>(__nv_bfloat16* p, float4 v) {
  __nv_bfloat162 a = __floats2bfloat162_rn(v.x, v.y), b = __floats2bfloat162_rn(v.z, v.w);
  uint2 u;
  u.x = *reinterpret_cast<unsigned*>(&a);
  u.y = *reinterpret_cast<unsigned*>(&b);
  *reinterpret_cast<uint2*>(p) = u;
}

// ---- the order in which the segmented sums visit the nodes ----
// Every row of E is read twice per iteration: as an out-edge of its source and as an in-edge of its destination.  E (187 MB at
// pileup-200) does not fit the L2, and in hit-index order (the hits arrive shuffled) the two reads are far apart: 307 MB came
// from DRAM.  The endpoints of an edge are neighbours in the detector, so with the nodes visited by azimuth the second read of
// a row follows the first within a few thousand nodes and hits the L2: every row comes from DRAM once (an LRU model of the L2
// reproduces both figures).  Only the ORDER OF VISITS changes -- each node's sum keeps its fixed order of edges -- so the
// results are the same bits; the position of a node inside its bin (atomics) is irrelevant for the same reason.
__device__ __forceinline__ int phi_bin(float phi_over_pi) {
  const int b = (int)((phi_over_pi + 1.f) * (0.5f * kPhiBins));
  return min(max(b, 0), kPhiBins - 1);
}
__global__ void phi_count_kernel(const float* __restrict__ hits, int64_t n, int32_t* __restrict__ count) {
  TRK_GRID_DEP_WAIT();
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) atomicAdd(&count[phi_bin(hits[i * 3 + 1])], 1);
}
// one block of kPhiBins threads: start = exclusive scan of count; count is zeroed for the placement pass
__global__ void __launch_bounds__(kPhiBins) phi_scan_kernel(int32_t* __restrict__ count, int32_t* __restrict__ start) {
  TRK_GRID_DEP_WAIT();
  __shared__ int32_t s[kPhiBins];
  const int t = threadIdx.x;
  const int32_t mine = count[t];
  s[t] = mine;
  __syncthreads();
  for (int o = 1; o < kPhiBins; o <<= 1) {
    const int32_t add = t >= o ? s[t - o] : 0;
    __syncthreads();
    s[t] += add;
    __syncthreads();
  }
  start[t] = s[t] - mine;
  count[t] = 0;
}
__global__ void phi_place_kernel(const float* __restrict__ hits, int64_t n, const int32_t* __restrict__ start, int32_t* __restrict__ fill,
                                 int32_t* __restrict__ order) {
  TRK_GRID_DEP_WAIT();
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) {
    const int b = phi_bin(hits[i * 3 + 1]);
    order[start[b] + atomicAdd(&fill[b], 1)] = (int32_t)i;
  }
}

// The work list of the segmented sums, built once per call: task 2 p + dir = (node at position p of the visiting order, its
// segment bounds), so a warp of segment_sum_kernel starts from ONE coalesced 16-byte load instead of the chain
// order -> row pointer -> ...
__global__ void seg_tasks_kernel(const int32_t* __restrict__ order, const int32_t* __restrict__ in_rowptr,
                                 const int32_t* __restrict__ out_rowptr, int4* __restrict__ tasks, int64_t n_nodes) {
  TRK_GRID_DEP_WAIT();
  const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= 2 * n_nodes) return;
  const int v = order[w >> 1], dir = (int)(w & 1);
  const int32_t* rp = dir == 0 ? in_rowptr : out_rowptr;
  tasks[w] = make_int4(v, rp[v], rp[v + 1], dir);
}

// One warp per (node, direction): X[v][H + dir*H + :] = sum over the segment of E rows (fp32 accumulate).
// H is a multiple of 4; lanes cover H/4 float4 columns in strides of 32.
template <typename T>
__global__ void __launch_bounds__(256)
segment_sum_kernel(const T* __restrict__ E, int H, const int4* __restrict__ tasks, const int32_t* __restrict__ in_perm,
                   T* __restrict__ X, int ldx, int64_t n_nodes) {
  TRK_GRID_DEP_WAIT();
  const int lane = threadIdx.x & 31;
  const int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (w >= 2 * n_nodes) return;
  const int4 task = tasks[w];             // nodes by azimuth (see above)
  const int64_t v = task.x;
  const int dir = task.w;        // 0: in (dst == v, via perm), 1: out (src == v, contiguous)
  const int b = task.y, e = task.z;
  for (int c = lane * 4; c < H; c += 128) {
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    int k = b;
    for (; k + 8 <= e; k += 8) {               // eight independent row loads in flight; the sum keeps its fixed order
      int64_t r[8];
#pragma unroll
      for (int t = 0; t < 8; ++t) r[t] = dir == 0 ? in_perm[k + t] : k + t;
      float4 x[8];
#pragma unroll
      for (int t = 0; t < 8; ++t) x[t] = load4<T>(E + r[t] * H + c);
#pragma unroll
      for (int t = 0; t < 8; ++t) { acc.x += x[t].x; acc.y += x[t].y; acc.z += x[t].z; acc.w += x[t].w; }
    }
    for (; k + 4 <= e; k += 4) {               // four
      int64_t r0, r1, r2, r3;
      if (dir == 0) { r0 = in_perm[k]; r1 = in_perm[k + 1]; r2 = in_perm[k + 2]; r3 = in_perm[k + 3]; }
      else { r0 = k; r1 = k + 1; r2 = k + 2; r3 = k + 3; }
      const float4 x0 = load4<T>(E + r0 * H + c), x1 = load4<T>(E + r1 * H + c), x2 = load4<T>(E + r2 * H + c),
                   x3 = load4<T>(E + r3 * H + c);
      acc.x += x0.x; acc.y += x0.y; acc.z += x0.z; acc.w += x0.w;
      acc.x += x1.x; acc.y += x1.y; acc.z += x1.z; acc.w += x1.w;
      acc.x += x2.x; acc.y += x2.y; acc.z += x2.z; acc.w += x2.w;
      acc.x += x3.x; acc.y += x3.y; acc.z += x3.z; acc.w += x3.w;
    }
    for (; k < e; ++k) {
      const int64_t row = dir == 0 ? in_perm[k] : k;
      const float4 x = load4<T>(E + row * H + c);
      acc.x += x.x; acc.y += x.y; acc.z += x.z; acc.w += x.w;
    }
    store4<T>(X + v * ldx + H + dir * H + c, acc);
  }
}

}  // namespace

trk_status build_gnn_csr(trk_ctx* ctx, const float* hits, const int32_t* src, const int32_t* dst, const int32_t* n_edges_dev,
                         int64_t n_edges_cap, int64_t n_nodes, cudaStream_t st) {
  // the visiting order of the segmented sums: nodes counting-sorted by phi bin (hits[:, 1] = phi / pi in (-1, 1])
  if (n_nodes > 0) {
    int32_t* count = ctx->phi_bins;
    int32_t* start = ctx->phi_bins + kPhiBins + 1;
    const unsigned nb = (unsigned)ceil_div(n_nodes, 256);
    TRK_TRY(fill_i32(ctx, count, 0, kPhiBins, st));
    TRK_LAUNCH(ctx, phi_count_kernel, nb, 256, 0, st, hits, n_nodes, count);
    TRK_LAUNCH(ctx, phi_scan_kernel, 1, kPhiBins, 0, st, count, start);
    TRK_LAUNCH(ctx, phi_place_kernel, nb, 256, 0, st, hits, n_nodes, start, count, ctx->node_order);
  }
  const unsigned eb = (unsigned)ceil_div(n_edges_cap + 1, 256);
  TRK_LAUNCH(ctx, rowptr_from_sorted_kernel, eb, 256, 0, st, src, n_edges_dev, n_edges_cap, ctx->out_rowptr, n_nodes);
  TRK_TRY(fill_i32(ctx, ctx->in_fill, 0, n_nodes + 1, st));
  TRK_LAUNCH(ctx, count_keys_kernel, eb, 256, 0, st, dst, n_edges_dev, n_edges_cap, ctx->in_fill);
  TRK_TRY(exclusive_scan_i32(ctx, ctx->in_fill, ctx->in_rowptr, n_nodes, ctx->scan_tmp, st));
  TRK_LAUNCH(ctx, place_keys_kernel, eb, 256, 0, st, dst, n_edges_dev, n_edges_cap, ctx->in_rowptr, ctx->in_fill, ctx->in_perm);
  TRK_LAUNCH(ctx, sort_segments_kernel, (unsigned)ceil_div(n_nodes * 32, 256), 256, 0, st, ctx->in_rowptr, ctx->in_perm, n_nodes);
  if (n_nodes > 0)
    TRK_LAUNCH(ctx, seg_tasks_kernel, (unsigned)ceil_div(2 * n_nodes, 256), 256, 0, st, ctx->node_order, ctx->in_rowptr, ctx->out_rowptr,
               ctx->seg_tasks, n_nodes);
  return TRK_OK;
}

trk_status segment_sums(trk_ctx* ctx, const void* E, bool bf16, int64_t n_nodes, void* X, cudaStream_t st) {
  const int H = ctx->H;
  const unsigned blocks = (unsigned)ceil_div(2 * n_nodes * 32, 256);
  // (a half-warp-per-row variant for H = 128 was measured slower: 99 vs 80 us per pileup-200 iteration)
  if (bf16) {
    TRK_LAUNCH(ctx, segment_sum_kernel<__nv_bfloat16>, blocks, 256, 0, st, (const __nv_bfloat16*)E, H, ctx->seg_tasks,
               ctx->in_perm, (__nv_bfloat16*)X, 3 * H, n_nodes);
  } else {
    TRK_LAUNCH(ctx, segment_sum_kernel<float>, blocks, 256, 0, st, (const float*)E, H, ctx->seg_tasks, ctx->in_perm,
               (float*)X, 3 * H, n_nodes);
  }
  return TRK_OK;
}

}  // namespace trk

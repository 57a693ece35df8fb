// S5: weakly-connected components by lock-free union-find ("WCC"; the paper
// ran Boost on the CPU, line 87).  Links always point from a larger to a smaller hit index, so
// the root of a set is its minimum and label[v] = root(v) is unique (reading C-17).
#include "common.cuh"

namespace trk {
namespace {

__global__ void cc_init_kernel(int32_t* __restrict__ parent, int64_t n, int32_t* __restrict__ pass_count) {
  TRK_GRID_DEP_WAIT();
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) parent[i] = (int32_t)i;
  if (i == 0 && pass_count) *pass_count = 0;
}

// A parent pointer only ever changes to another ancestor of its node (path halving) or, at a root, to a smaller root (the
// hook below), so a STALE value is still an ancestor: the walk may read through the SM's L1 (ld.global.ca, ~10x shorter
// latency than the L2 round trip of a volatile load), it just may take a step more.  A stale "root" is caught by the hook:
// atomicMin acts on the true value and the caller retries from what it returns.
__device__ __forceinline__ int32_t load_parent(const int32_t* p) {
  int32_t v;
  asm volatile("ld.global.ca.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

__device__ __forceinline__ int32_t find_root(int32_t* parent, int32_t x) {
  // path halving with plain stores: every value ever stored is an ancestor of x (links are only ever added at roots and
  // point to smaller indices), hence valid whatever the interleaving; only the hook below needs an atomic
  int32_t p = load_parent(parent + x);
  while (p != x) {
    const int32_t gp = load_parent(parent + p);
    if (gp != p) parent[x] = gp;
    x = p;
    p = gp;
  }
  return x;
}

__global__ void cc_union_kernel(int32_t* __restrict__ parent, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
                                const float* __restrict__ score, const int32_t* __restrict__ n_edges_dev, int64_t n_edges_cap,
                                float cut, int32_t* __restrict__ pass_count) {
  TRK_GRID_DEP_WAIT();
  const int64_t n_edges = n_edges_dev ? min((int64_t)*n_edges_dev, n_edges_cap) : n_edges_cap;
  int local = 0;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n_edges; k += (int64_t)gridDim.x * blockDim.x) {
    if (!(score[k] > cut)) continue;
    ++local;
    int32_t a = src[k], b = dst[k];
    while (true) {
      a = find_root(parent, a);
      b = find_root(parent, b);
      if (a == b) break;
      const int32_t hi = max(a, b), lo = min(a, b);
      const int32_t old = atomicMin(&parent[hi], lo);
      if (old == hi) break;  // hi was a root and now points to lo
      a = old;               // hi had already been linked to `old`; keep old and lo connected
      b = lo;
    }
  }
  if (pass_count) {
    for (int o = 16; o > 0; o >>= 1) local += __shfl_down_sync(0xffffffffu, local, o);
    if ((threadIdx.x & 31) == 0 && local) atomicAdd(pass_count, local);
  }
}

__global__ void cc_flatten_kernel(const int32_t* __restrict__ parent, int32_t* __restrict__ labels, int64_t n) {
  TRK_GRID_DEP_WAIT();
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int32_t x = (int32_t)i;
  while (true) {
    int32_t p = parent[x];
    if (p == x) break;
    x = p;
  }
  labels[i] = x;
}

}  // namespace

trk_status cc_labels(trk_ctx* ctx, int64_t n, const int32_t* src, const int32_t* dst, const float* score,
                     const int32_t* n_edges_dev, int64_t n_edges_cap, float cut, int32_t* labels, int32_t* pass_count,
                     cudaStream_t st) {
  if (n <= 0) return TRK_OK;
  TRK_LAUNCH(ctx, cc_init_kernel, (unsigned)ceil_div(n, 256), 256, 0, st, ctx->parent, n, pass_count);
  if (n_edges_cap > 0) {
    const int64_t blocks = std::min<int64_t>(ceil_div(n_edges_cap, 256), (int64_t)ctx->sm_count * 16);
    TRK_LAUNCH(ctx, cc_union_kernel, (unsigned)blocks, 256, 0, st, ctx->parent, src, dst, score, n_edges_dev, n_edges_cap, cut,
               pass_count);
  }
  TRK_LAUNCH(ctx, cc_flatten_kernel, (unsigned)ceil_div(n, 256), 256, 0, st, ctx->parent, labels, n);
  return TRK_OK;
}

}  // namespace trk

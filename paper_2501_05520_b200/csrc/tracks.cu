// S6: track-candidate lists from the S5 labels ("Each track candidate is a list of
// spacepoints"; line 89: the output of the service; reading C-23).
//
// A track is a component with >= min_hits hits.  Tracks are ordered by label (= smallest hit index),
// hits inside a track by hit index, so the output is unique:
//   size[label[v]]++                         (integer atomics: order independent)
//   keep[r] = label[r] == r && size[r] >= min_hits;  tidx = exclusive scan(keep);  hoff = exclusive scan(keep ? size : 0)
//   key[v]  = keep[label[v]] ? tidx[label[v]] : N    (N sorts after every track)
//   stable LSD radix sort of (key, v) with 8-bit digits: v starts in index order and every pass is
//   stable, so equal keys stay in ascending hit index; the first hoff[N] values are track_hits.
#include <utility>

#include "common.cuh"

namespace trk {
namespace {

constexpr int kRadixThreads = 256;
constexpr int kRadixBits = 8;
constexpr int kRadixBins = 1 << kRadixBits;

// labels come from S5 (label = smallest hit index of the component); a value outside [0, n) handed to the stage hook is
// read as "v is its own component" so that nothing is indexed out of range
__device__ __forceinline__ int32_t label_of(const int32_t* __restrict__ labels, int64_t v, int64_t n) {
  const int32_t r = labels[v];
  return (r < 0 || r >= n) ? (int32_t)v : r;
}

__global__ void track_size_kernel(const int32_t* __restrict__ labels, int64_t n, int32_t* __restrict__ size) {
  TRK_GRID_DEP_WAIT();
  const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (v < n) atomicAdd(&size[label_of(labels, v, n)], 1);
}

__global__ void track_keep_kernel(const int32_t* __restrict__ labels, const int32_t* __restrict__ size, int64_t n, int min_hits,
                                  int32_t* __restrict__ keep, int32_t* __restrict__ ksize) {
  TRK_GRID_DEP_WAIT();
  const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= n) return;
  const int k = (label_of(labels, v, n) == (int32_t)v && size[v] >= min_hits) ? 1 : 0;
  keep[v] = k;
  ksize[v] = k ? size[v] : 0;
}

// track_offsets[t] = first position of track t; tracks beyond the capacity are dropped (overflow flag set).
__global__ void track_offsets_kernel(const int32_t* __restrict__ keep, const int32_t* __restrict__ tidx, const int32_t* __restrict__ hoff,
                                     int64_t n, int64_t capacity, int32_t* __restrict__ track_offsets, int32_t* __restrict__ track_counts,
                                     int32_t* __restrict__ overflow_flag) {
  TRK_GRID_DEP_WAIT();
  const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (v < n && keep[v] && tidx[v] <= capacity) track_offsets[tidx[v]] = hoff[v];
  if (v == 0) {
    const int64_t total = tidx[n];
    if (total <= capacity) {
      track_offsets[total] = hoff[n];
      track_counts[0] = (int32_t)total;
      track_counts[1] = hoff[n];
    } else {
      track_counts[0] = (int32_t)capacity;
      track_counts[1] = -1;                 // patched by track_emit_kernel from track_offsets[capacity]
      if (overflow_flag) *overflow_flag = 1;
    }
  }
}

__global__ void track_key_kernel(const int32_t* __restrict__ labels, const int32_t* __restrict__ keep, const int32_t* __restrict__ tidx,
                                 int64_t n, int32_t* __restrict__ key, int32_t* __restrict__ val) {
  TRK_GRID_DEP_WAIT();
  const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= n) return;
  const int32_t r = label_of(labels, v, n);
  key[v] = keep[r] ? tidx[r] : (int32_t)n;
  val[v] = (int32_t)v;
}

// hist[d * n_blocks + b] = number of keys of block b whose digit is d (digit-major, so one exclusive scan gives
// every (digit, block) its first output position)
__global__ void __launch_bounds__(kRadixThreads)
radix_hist_kernel(const int32_t* __restrict__ key, int64_t n, int shift, int32_t* __restrict__ hist, int n_blocks) {
  TRK_GRID_DEP_WAIT();
  __shared__ int cnt[kRadixBins];
  cnt[threadIdx.x] = 0;
  __syncthreads();
  const int64_t i = (int64_t)blockIdx.x * kRadixThreads + threadIdx.x;
  if (i < n) atomicAdd(&cnt[((uint32_t)key[i] >> shift) & (kRadixBins - 1)], 1);
  __syncthreads();
  hist[(int64_t)threadIdx.x * n_blocks + blockIdx.x] = cnt[threadIdx.x];
}

// Stable scatter: position = scanned hist of (digit, block) + number of earlier items of the block with the same digit.
__global__ void __launch_bounds__(kRadixThreads)
radix_scatter_kernel(const int32_t* __restrict__ key, const int32_t* __restrict__ val, int64_t n, int shift,
                     const int32_t* __restrict__ hist_scan, int n_blocks, int32_t* __restrict__ key_out, int32_t* __restrict__ val_out) {
  TRK_GRID_DEP_WAIT();
  constexpr int kWarps = kRadixThreads / 32;
  __shared__ int wcnt[kWarps][kRadixBins];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int w = 0; w < kWarps; ++w) wcnt[w][threadIdx.x] = 0;
  __syncthreads();
  const int64_t i = (int64_t)blockIdx.x * kRadixThreads + threadIdx.x;
  const bool active = i < n;
  const int32_t k = active ? key[i] : 0;
  const int d = active ? (int)(((uint32_t)k >> shift) & (kRadixBins - 1)) : kRadixBins + lane;   // inactive lanes match nobody
  const unsigned peers = __match_any_sync(0xffffffffu, d);
  const int rank_in_warp = __popc(peers & ((1u << lane) - 1u));
  if (active && rank_in_warp == 0) wcnt[warp][d] = __popc(peers);
  __syncthreads();
  {
    int run = 0;                       // thread t owns digit t: exclusive prefix over the warps, in warp order
    for (int w = 0; w < kWarps; ++w) {
      const int c = wcnt[w][threadIdx.x];
      wcnt[w][threadIdx.x] = run;
      run += c;
    }
  }
  __syncthreads();
  if (active) {
    const int64_t pos = (int64_t)hist_scan[(int64_t)d * n_blocks + blockIdx.x] + wcnt[warp][d] + rank_in_warp;
    key_out[pos] = k;
    val_out[pos] = val[i];
  }
}

__global__ void track_emit_kernel(const int32_t* __restrict__ val, const int32_t* __restrict__ track_offsets, int64_t n,
                                  int32_t* __restrict__ track_counts, int32_t* __restrict__ track_hits) {
  TRK_GRID_DEP_WAIT();
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int32_t total = track_offsets[track_counts[0]];
  if (i < n) track_hits[i] = i < total ? val[i] : -1;
  if (i == 0) track_counts[1] = total;
}

}  // namespace

trk_status build_tracks(trk_ctx* ctx, const int32_t* labels, int64_t n, int min_hits, int32_t* track_offsets, int64_t capacity,
                        int32_t* track_hits, int32_t* track_counts, int32_t* overflow_flag, cudaStream_t st) {
  if (min_hits < 1) min_hits = 1;
  if (n <= 0) {
    TRK_TRY(fill_i32(ctx, track_offsets, 0, 1, st));
    return fill_i32(ctx, track_counts, 0, 2, st);
  }
  const unsigned nb = (unsigned)ceil_div(n, 256);
  int32_t *size = ctx->tk_a, *keep = ctx->tk_b, *ksize = ctx->tk_c, *tidx = ctx->tk_d, *hoff = ctx->tk_e;
  TRK_TRY(fill_i32(ctx, size, 0, n, st));
  TRK_LAUNCH(ctx, track_size_kernel, nb, 256, 0, st, labels, n, size);
  TRK_LAUNCH(ctx, track_keep_kernel, nb, 256, 0, st, labels, size, n, min_hits, keep, ksize);
  TRK_TRY(exclusive_scan_i32(ctx, keep, tidx, n, ctx->scan_tmp, st));
  TRK_TRY(exclusive_scan_i32(ctx, ksize, hoff, n, ctx->scan_tmp, st));
  TRK_LAUNCH(ctx, track_offsets_kernel, nb, 256, 0, st, keep, tidx, hoff, n, capacity, track_offsets, track_counts, overflow_flag);
  // size / ksize are dead from here on: they become the second (key, value) buffer of the sort
  int32_t *key0 = ctx->tk_f, *val0 = ctx->tk_g, *key1 = size, *val1 = ksize;
  TRK_LAUNCH(ctx, track_key_kernel, nb, 256, 0, st, labels, keep, tidx, n, key0, val0);
  int bits = 1;
  while ((n >> bits) != 0) ++bits;          // keys are in [0, n]
  const int n_blocks = (int)nb;
  for (int shift = 0; shift < bits; shift += kRadixBits) {
    TRK_LAUNCH(ctx, radix_hist_kernel, nb, kRadixThreads, 0, st, key0, n, shift, ctx->tk_hist, n_blocks);
    TRK_TRY(exclusive_scan_i32(ctx, ctx->tk_hist, ctx->tk_hist_scan, (int64_t)kRadixBins * n_blocks, ctx->scan_tmp, st));
    TRK_LAUNCH(ctx, radix_scatter_kernel, nb, kRadixThreads, 0, st, key0, val0, n, shift, ctx->tk_hist_scan, n_blocks, key1, val1);
    std::swap(key0, key1);
    std::swap(val0, val1);
  }
  TRK_LAUNCH(ctx, track_emit_kernel, nb, 256, 0, st, val0, track_offsets, n, track_counts, track_hits);
  return TRK_OK;
}

}  // namespace trk

// Integer utilities: exclusive scan, fill, stable stream compaction (S3 tail).
#include "common.cuh"

namespace trk {

namespace {

constexpr int kScanThreads = 512;
constexpr int kScanItems = 4;
constexpr int kScanTile = kScanThreads * kScanItems;

// Exclusive scan of one int per thread across the block; returns the exclusive prefix, total in *total.
__device__ __forceinline__ int block_exclusive_scan(int v, int* total) {
  __shared__ int warp_sums[kScanThreads / 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  __syncthreads();  // protect warp_sums reuse across calls
  if (lane == 31) warp_sums[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    int w = lane < kScanThreads / 32 ? warp_sums[lane] : 0;
    int wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, wi, o);
      if (lane >= o) wi += t;
    }
    if (lane < kScanThreads / 32) warp_sums[lane] = wi - w;  // exclusive warp offsets
    if (lane == 31) *total = wi;
  }
  __syncthreads();
  return incl - v + warp_sums[warp];
}

__global__ void __launch_bounds__(kScanThreads) scan_local_kernel(const int32_t* __restrict__ in, int32_t* __restrict__ out,
                                                                  int32_t* __restrict__ block_sums, int64_t n) {
  TRK_GRID_DEP_WAIT();
  __shared__ int total;
  const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
  int v[kScanItems];
  int s = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    v[i] = (base + i < n) ? in[base + i] : 0;
    s += v[i];
  }
  int excl = block_exclusive_scan(s, &total);
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    if (base + i < n) out[base + i] = excl;
    excl += v[i];
  }
  if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

// Single block: exclusive scan of the block sums in place; block_sums[n_blocks] = grand total.
__global__ void __launch_bounds__(kScanThreads) scan_sums_kernel(int32_t* __restrict__ block_sums, int64_t n_blocks) {
  TRK_GRID_DEP_WAIT();
  __shared__ int total;
  int carry = 0;
  for (int64_t base = 0; base < n_blocks; base += kScanThreads) {
    int64_t i = base + threadIdx.x;
    int v = i < n_blocks ? block_sums[i] : 0;
    int excl = block_exclusive_scan(v, &total);
    if (i < n_blocks) block_sums[i] = excl + carry;
    carry += total;
    __syncthreads();
  }
  if (threadIdx.x == 0) block_sums[n_blocks] = carry;
}

__global__ void __launch_bounds__(kScanThreads) scan_add_kernel(int32_t* __restrict__ out, const int32_t* __restrict__ block_sums,
                                                                int64_t n, int64_t n_blocks) {
  TRK_GRID_DEP_WAIT();
  const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
  const int add = block_sums[blockIdx.x];
#pragma unroll
  for (int i = 0; i < kScanItems; ++i)
    if (base + i < n) out[base + i] += add;
  if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = block_sums[n_blocks];
}

__global__ void fill_i32_kernel(int32_t* p, int32_t v, int64_t n) {
  TRK_GRID_DEP_WAIT();
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = v;
}

// ---- stable compaction of edges with score > cut ----
__global__ void __launch_bounds__(kScanThreads) compact_count_kernel(const float* __restrict__ score, const int32_t* __restrict__ n_dev,
                                                                     int64_t n_cap, float cut, int32_t* __restrict__ block_sums) {
  TRK_GRID_DEP_WAIT();
  __shared__ int total;
  const int64_t n = min((int64_t)*n_dev, n_cap);
  const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
  int s = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) s += (base + i < n && score[base + i] > cut) ? 1 : 0;
  block_exclusive_scan(s, &total);
  if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kScanThreads) compact_write_kernel(const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
                                                                     const float* __restrict__ score, const int32_t* __restrict__ n_dev,
                                                                     int64_t n_cap, float cut, const int32_t* __restrict__ block_sums,
                                                                     int64_t n_blocks, int32_t* __restrict__ out_src,
                                                                     int32_t* __restrict__ out_dst, int64_t out_cap,
                                                                     int32_t* __restrict__ count_out, int32_t* __restrict__ overflow_flag) {
  TRK_GRID_DEP_WAIT();
  __shared__ int total;
  const int64_t n = min((int64_t)*n_dev, n_cap);
  const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
  bool keep[kScanItems];
  int s = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    keep[i] = (base + i < n) && (score[base + i] > cut);
    s += keep[i] ? 1 : 0;
  }
  int64_t pos = (int64_t)block_sums[blockIdx.x] + block_exclusive_scan(s, &total);
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    if (keep[i]) {
      if (pos < out_cap) {
        out_src[pos] = src[base + i];
        out_dst[pos] = dst[base + i];
      }
      ++pos;
    }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    int64_t tot = block_sums[n_blocks];
    *count_out = (int32_t)min(tot, out_cap);
    if (tot > out_cap) *overflow_flag = 1;
  }
}

}  // namespace

trk_status exclusive_scan_i32(trk_ctx* ctx, const int32_t* in, int32_t* out, int64_t n, int32_t* tmp, cudaStream_t st) {
  // out has n+1 entries (out[n] = total); tmp has ceil(n/2048)+1 entries.
  const int64_t nb = ceil_div(n > 0 ? n : 1, kScanTile);
  TRK_LAUNCH(ctx, scan_local_kernel, (unsigned)nb, kScanThreads, 0, st, in, out, tmp, n);
  TRK_LAUNCH(ctx, scan_sums_kernel, 1, kScanThreads, 0, st, tmp, nb);
  TRK_LAUNCH(ctx, scan_add_kernel, (unsigned)nb, kScanThreads, 0, st, out, tmp, n, nb);
  return TRK_OK;
}

trk_status fill_i32(trk_ctx* ctx, int32_t* p, int32_t v, int64_t n, cudaStream_t st) {
  if (n <= 0) return TRK_OK;
  TRK_LAUNCH(ctx, fill_i32_kernel, (unsigned)ceil_div(n, 256), 256, 0, st, p, v, n);
  return TRK_OK;
}

trk_status compact_edges(trk_ctx* ctx, const int32_t* src, const int32_t* dst, const float* score, const int32_t* n_dev,
                         int64_t n_cap, float cut, int32_t* out_src, int32_t* out_dst, int64_t out_cap, int32_t* count_out,
                         int32_t* overflow_flag, cudaStream_t st) {
  const int64_t nb = ceil_div(n_cap > 0 ? n_cap : 1, kScanTile);
  int32_t* tmp = ctx->scan_tmp;
  TRK_LAUNCH(ctx, compact_count_kernel, (unsigned)nb, kScanThreads, 0, st, score, n_dev, n_cap, cut, tmp);
  TRK_LAUNCH(ctx, scan_sums_kernel, 1, kScanThreads, 0, st, tmp, nb);
  TRK_LAUNCH(ctx, compact_write_kernel, (unsigned)nb, kScanThreads, 0, st, src, dst, score, n_dev, n_cap, cut, tmp, nb,
             out_src, out_dst, out_cap, count_out, overflow_flag);
  return TRK_OK;
}

}  // namespace trk

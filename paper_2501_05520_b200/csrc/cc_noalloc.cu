// trk_cc_noalloc: S5 (weakly-connected components, "WCC") for callers that must not allocate.
//
// Who needs this.  Every other entry point that runs S5 goes through a trk_ctx, and trk_create sizes and cudaMallocs the
// whole workspace, the union-find parent array among it.  Some callers of a tracking library cannot do that: a backend
// that is handed a fixed slice of device memory by its serving framework (the framework, not the
// backend, owns the GPU) and is forbidden to grow it; code that runs inside a region where cudaMalloc is illegal or
// would deadlock (a stream capture in progress on another thread in global capture mode, a host callback on a stream);
// and latency-critical trigger-style loops where an implicit device synchronisation inside cudaMalloc/cudaFree is not
// acceptable.  For them the parent array lives in the library image itself: a file-scope __device__ array that every GPU
// which loads libtrk.so holds from module load until the process exits (TRK_CC_NOALLOC_MAX_HITS x 4 bytes = 4 MiB per GPU).
//
// The array's name means two different things.  Inside device code `g_parent` is the device array.  In host code the same
// name is only a host-side handle of the symbol: passing it to a kernel hands the kernel a host address, which faults or,
// on a system where the GPU can reach host memory, quietly works on the wrong bytes.  So the host code below never passes
// `g_parent`; it asks the runtime for the device address once per device (cudaGetSymbolAddress with that device current,
// return code checked) and passes that pointer.
//
// Same union-find as cc.cu (links point from a larger to a smaller hit index, root = minimum = label, reading C-17), in
// kernels of its own so that the context path is untouched.
#include <algorithm>
#include <mutex>

#include "common.cuh"

// The scratch.  Shared by every call on a device and never cleared between calls: it still holds the forest of the previous
// call.  init_kernel rewrites entries [0, n) at the start of each call and nothing reads an entry >= n, so no state of
// an earlier call can leak into a result.  Two calls that are in flight on the same GPU at the same time (two streams, two
// threads) would both write it: that is a data race, the caller must order them.
static __device__ __align__(256) int32_t g_parent[TRK_CC_NOALLOC_MAX_HITS];

namespace trk {
namespace {

constexpr int64_t kMaxHits = TRK_CC_NOALLOC_MAX_HITS;
constexpr int kMaxDevices = 64;

std::mutex g_setup_mutex;
int32_t* g_parent_dev[kMaxDevices] = {};  // device address of g_parent on device d, nullptr until the first call there
int g_sm_count[kMaxDevices] = {};

__global__ void init_kernel(int32_t* __restrict__ parent, int64_t n) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) parent[i] = (int32_t)i;
}

// A stale parent value is still an ancestor (links are only added at roots and point to smaller indices), so the walk
// may read through L1; the atomicMin of the hook acts on the true value.
__device__ __forceinline__ int32_t load_parent(const int32_t* p) {
  int32_t v;
  asm volatile("ld.global.ca.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

__device__ __forceinline__ int32_t find_root(int32_t* parent, int32_t x) {
  int32_t p = load_parent(parent + x);
  while (p != x) {
    const int32_t gp = load_parent(parent + p);
    if (gp != p) parent[x] = gp;  // path halving
    x = p;
    p = gp;
  }
  return x;
}

__global__ void union_kernel(int32_t* __restrict__ parent, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
                             const float* __restrict__ score, int64_t n_edges, float cut) {
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n_edges; k += (int64_t)gridDim.x * blockDim.x) {
    if (!(score[k] > cut)) continue;
    int32_t a = src[k], b = dst[k];
    while (true) {
      a = find_root(parent, a);
      b = find_root(parent, b);
      if (a == b) break;
      const int32_t hi = max(a, b), lo = min(a, b);
      const int32_t old = atomicMin(&parent[hi], lo);
      if (old == hi) break;
      a = old;
      b = lo;
    }
  }
}

__global__ void flatten_kernel(const int32_t* __restrict__ parent, int32_t* __restrict__ labels, int64_t n) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int32_t x = (int32_t)i;
  while (true) {
    const int32_t p = parent[x];
    if (p == x) break;
    x = p;
  }
  labels[i] = x;
}

// Once per device, with that device current: the device address of g_parent (and the SM count for the grid size).
trk_status setup_device(int dev, int32_t** parent, int* sm_count) {
  std::lock_guard<std::mutex> lk(g_setup_mutex);
  if (!g_parent_dev[dev]) {
    int major = 0, sms = 0;
    TRK_CUDA(nullptr, cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return fail(nullptr, TRK_ERR_UNSUPPORTED_DEVICE, "trk_cc_noalloc: the current device is not compute capability 10.x");
    TRK_CUDA(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    void* p = nullptr;
    TRK_CUDA(nullptr, cudaGetSymbolAddress(&p, g_parent));
    if (!p) return fail(nullptr, TRK_ERR_CUDA, "trk_cc_noalloc: cudaGetSymbolAddress returned a null address");
    g_sm_count[dev] = sms;
    g_parent_dev[dev] = static_cast<int32_t*>(p);
  }
  *parent = g_parent_dev[dev];
  *sm_count = g_sm_count[dev];
  return TRK_OK;
}

}  // namespace
}  // namespace trk

extern "C" trk_status trk_cc_noalloc(int64_t n, const int32_t* src, const int32_t* dst, const float* score, int64_t n_edges,
                                     float cut, int32_t* labels, void* cuda_stream) {
  using namespace trk;
  if (n < 0 || n_edges < 0 || (n > 0 && !labels) || (n_edges > 0 && (!src || !dst || !score)))
    return fail(nullptr, TRK_ERR_INVALID_ARG, "trk_cc_noalloc: bad arguments");
  if (n > kMaxHits)
    return fail(nullptr, TRK_ERR_CAPACITY, "trk_cc_noalloc: n = " + std::to_string(n) + " exceeds TRK_CC_NOALLOC_MAX_HITS = " +
                                               std::to_string(kMaxHits) + " (the size of the built-in scratch array); use a trk_ctx and trk_stage_cc");
  if (n == 0) return TRK_OK;
  int dev = -1;
  TRK_CUDA(nullptr, cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return fail(nullptr, TRK_ERR_UNSUPPORTED_DEVICE, "trk_cc_noalloc: device ordinal out of range");
  int32_t* parent = nullptr;
  int sm_count = 0;
  TRK_TRY(setup_device(dev, &parent, &sm_count));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  init_kernel<<<(unsigned)ceil_div(n, 256), 256, 0, st>>>(parent, n);
  if (n_edges > 0) {
    const int64_t blocks = std::min<int64_t>(ceil_div(n_edges, 256), (int64_t)sm_count * 16);
    union_kernel<<<(unsigned)blocks, 256, 0, st>>>(parent, src, dst, score, n_edges, cut);
  }
  flatten_kernel<<<(unsigned)ceil_div(n, 256), 256, 0, st>>>(parent, labels, n);
  TRK_CUDA(nullptr, cudaPeekAtLastError());
  return TRK_OK;
}

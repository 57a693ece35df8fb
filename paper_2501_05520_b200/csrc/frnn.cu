// S2: fixed-radius nearest-neighbour graph in the latent space (the paper used the
// FRNN CUDA package, line 87).  Definition (readings C-7..C-9, C-11, C-21):
//   edge i -> j  iff  same event, outer(i,j), d2(i,j) <= r^2, and j is among the K smallest (d2, j).
// d2 is accumulated in fp64 from the fp32 embedding, k ascending, with separate multiply and add
// (__dsub_rn/__dmul_rn/__dadd_rn forbid FMA contraction), so accept and rank decisions are exact
// functions of the inputs and the edge list is unique.
//
// Search structure (an implementation detail that cannot change the result): hits are binned on
// g <= 3 coordinates of P^T e (P has orthonormal columns, so projected distance <= true distance)
// into a per-event grid with cell edge >= r; a query looks at the 3^g neighbouring cells.  Inside a
// spatial cell the hits are further binned by kRBuckets monotone buckets of their radius feature r:
// outer(i,j) needs r_j >= r_i, hence bucket(j) >= bucket(i), so a query scans only the part of each
// neighbouring cell that starts at its own bucket (about half of it) -- the counting sort by
// (cell, bucket) makes that part one contiguous range.  One warp serves one query: lanes stride over
// the candidates, accepted ones are appended to a shared-memory buffer via ballot; when the buffer
// fills, a bisection on d2 finds a threshold that keeps at least the K nearest (a warp bitonic sort on
// (d2, j) only when ties defeat it, and once at the end for the exact K nearest); rank counting on j
// gives the (src, dst) output order.
#include <cmath>

#include "common.cuh"

namespace trk {
namespace {

__device__ __forceinline__ int float_to_ordered(float f) {
  int i = __float_as_int(f);
  return i >= 0 ? i : i ^ 0x7fffffff;
}
__device__ __forceinline__ float ordered_to_float(int i) { return __int_as_float(i >= 0 ? i : i ^ 0x7fffffff); }

__global__ void frnn_reset_kernel(int32_t* __restrict__ bbox, int32_t* __restrict__ cell_count, int32_t* __restrict__ cell_fill,
                                  int64_t n_cells_plus1) {
  TRK_GRID_DEP_WAIT();
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < 3) {
    bbox[i] = 0x7fffffff;          // min
    bbox[3 + i] = (int)0x80000000; // max
  }
  if (i == 3) {
    bbox[6] = 0x7fffffff;          // min of the radius feature
    bbox[7] = (int)0x80000000;     // max
    bbox[8] = 0;                   // max |e_k| over all hits and coordinates (bits of a non-negative float)
  }
  if (i < n_cells_plus1) cell_count[i] = 0;
  if (i + 1 < n_cells_plus1) cell_fill[i] = 0;
}

// proj[i] = P^T e_i  (or the first g coordinates), and the global bounding box.
__global__ void frnn_project_kernel(const float* __restrict__ emb, const float* __restrict__ hits, int d_e, const float* __restrict__ P, int g,
                                    float* __restrict__ proj, int32_t* __restrict__ bbox, int64_t n) {
  TRK_GRID_DEP_WAIT();
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  float p[3] = {0.f, 0.f, 0.f};
  float emax = 0.f;
  if (i < n) {
    const float* e = emb + i * d_e;
    if (P) {
      for (int k = 0; k < d_e; ++k) {
        float v = e[k];
        emax = fmaxf(emax, fabsf(v));
        for (int a = 0; a < g; ++a) p[a] = fmaf(v, P[k * 3 + a], p[a]);
      }
    } else {
      for (int a = 0; a < g; ++a) p[a] = e[a];      // exact: no rounding slack needed (emax stays 0)
    }
    proj[i * 3 + 0] = p[0];
    proj[i * 3 + 1] = p[1];
    proj[i * 3 + 2] = p[2];
  }
  // warp-reduce, then block-reduce through shared memory: ONE set of nine atomics per block (the atomics all hit the same nine
  // words, so their number is the kernel's run time: 22 us with one set per warp)
  __shared__ int s_red[9][8];
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
  int red[9];
  for (int a = 0; a < 3; ++a) {
    red[a] = i < n ? float_to_ordered(p[a]) : 0x7fffffff;            // min
    red[3 + a] = i < n ? float_to_ordered(p[a]) : (int)0x80000000;   // max
  }
  {
    const int key = i < n ? float_to_ordered(hits[i * 3]) : 0;
    red[6] = i < n ? key : 0x7fffffff;
    red[7] = i < n ? key : (int)0x80000000;
    red[8] = __float_as_int(emax);       // non-negative floats order like their bit patterns
  }
#pragma unroll
  for (int q = 0; q < 9; ++q) {
    const bool is_min = q < 3 || q == 6;
    for (int o = 16; o > 0; o >>= 1) {
      const int other = __shfl_xor_sync(0xffffffffu, red[q], o);
      red[q] = is_min ? min(red[q], other) : max(red[q], other);
    }
    if (lane == 0) s_red[q][wrp] = red[q];
  }
  __syncthreads();
  if (threadIdx.x < 9) {
    const int q = threadIdx.x;
    const bool is_min = q < 3 || q == 6;
    int v = s_red[q][0];
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) v = is_min ? min(v, s_red[q][w]) : max(v, s_red[q][w]);
    if (is_min) atomicMin(&bbox[q], v);
    else atomicMax(&bbox[q], v);
  }
}

__global__ void frnn_grid_setup_kernel(const int32_t* __restrict__ bbox, float radius, int g, int G, GridParams* __restrict__ gp) {
  TRK_GRID_DEP_WAIT();
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  // Rounding slack of the fp32 projection p = sum_k e_k P_ka (an fmaf chain): |p_hat - p| <= d_e 2^-24 sum_k |e_k| |P_ka|
  // <= d_e^1.5 2^-24 max|e| (unit columns), i.e. <= 2^-18 max|e| for d_e <= 16.  Two computed points are at most 2 sqrt(3) of
  // that further apart than the true ones; proj_eps = 2^-16 max|e| covers it with margin and scales with the data.
  const float proj_eps = __int_as_float(bbox[8]) * 1.52587890625e-05f;
  gp->proj_eps = proj_eps;
  // cell edge >= r with relative slack for the cell-index arithmetic and proj_eps for the projection
  const float cell_min = radius * 1.001f + proj_eps + 1e-30f;
  int cells = 1;
  for (int a = 0; a < 3; ++a) {
    if (a >= g) {
      gp->origin[a] = 0.f;
      gp->inv_cell[a] = 0.f;
      gp->dims[a] = 1;
      continue;
    }
    float lo = ordered_to_float(bbox[a]), hi = ordered_to_float(bbox[3 + a]);
    if (!(hi >= lo)) { lo = 0.f; hi = 0.f; }
    float extent = hi - lo;
    float cell = fmaxf(cell_min, extent / (float)G * 1.0001f);
    int d = (int)floorf(extent / cell) + 1;
    d = max(1, min(d, G));
    gp->origin[a] = lo;
    gp->inv_cell[a] = 1.0f / cell;
    gp->dims[a] = d;
    cells *= d;
  }
  gp->cells_per_event = cells;
  // radius buckets: equal-width bins over [r_min, r_max]; any monotone map keeps the search exact (see r_bucket)
  float rlo = ordered_to_float(bbox[6]), rhi = ordered_to_float(bbox[7]);
  if (!(rhi > rlo)) { rlo = 0.f; rhi = 0.f; }
  gp->r_origin = rlo;
  gp->r_inv = rhi > rlo ? (float)kRBuckets / (rhi - rlo) : 0.f;
}

// Monotone non-decreasing in r (fp32 subtraction of a constant, multiplication by a non-negative constant, floor and clamp
// all are), so r_i <= r_j implies bucket(i) <= bucket(j): a candidate in a lower bucket than the query can never be "outer".
__device__ __forceinline__ int r_bucket(const GridParams& gp, float r) {
  const int b = (int)floorf((r - gp.r_origin) * gp.r_inv);
  return max(0, min(b, kRBuckets - 1));
}

__device__ __forceinline__ void cell_coords(const GridParams& gp, const float* p, int c[3]) {
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    int v = (int)floorf((p[a] - gp.origin[a]) * gp.inv_cell[a]);
    c[a] = max(0, min(v, gp.dims[a] - 1));   // clamping is monotone, so neighbours stay neighbours
  }
}

__global__ void frnn_count_kernel(const float* __restrict__ proj, const float* __restrict__ hits, const int32_t* __restrict__ ev_of_hit,
                                  const GridParams* __restrict__ gpp, int32_t* __restrict__ cell_of_hit,
                                  int32_t* __restrict__ cell_count, int64_t n) {
  TRK_GRID_DEP_WAIT();
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const GridParams gp = *gpp;
  int c[3];
  cell_coords(gp, proj + i * 3, c);
  // (event, spatial cell, radius bucket), the bucket fastest: the part of a spatial cell from bucket b on is contiguous
  int cell = (ev_of_hit[i] * gp.cells_per_event + (c[2] * gp.dims[1] + c[1]) * gp.dims[0] + c[0]) * kRBuckets + r_bucket(gp, hits[i * 3]);
  cell_of_hit[i] = cell;
  atomicAdd(&cell_count[cell], 1);
}

// Sorted records: semb[pos][D] and smeta[pos] = (r, |z|, index, cell).
__global__ void frnn_scatter_kernel(const float* __restrict__ emb, const float* __restrict__ hits, int d_e, int d_pad,
                                    const int32_t* __restrict__ cell_of_hit, const int32_t* __restrict__ cell_start,
                                    int32_t* __restrict__ cell_fill, float* __restrict__ semb, float4* __restrict__ smeta,
                                    const float* __restrict__ proj, float4* __restrict__ sproj, int64_t n) {
  TRK_GRID_DEP_WAIT();
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int cell = cell_of_hit[i];
  const int pos = cell_start[cell] + atomicAdd(&cell_fill[cell], 1);
  for (int k = 0; k < d_pad; ++k) semb[(int64_t)pos * d_pad + k] = k < d_e ? emb[i * d_e + k] : 0.f;
  smeta[pos] = make_float4(hits[i * 3 + 0], fabsf(hits[i * 3 + 2]), __int_as_float((int)i), __int_as_float(cell));
  sproj[pos] = make_float4(proj[i * 3 + 0], proj[i * 3 + 1], proj[i * 3 + 2], 0.f);
}

// ---- warp-level bitonic sort of n (power of two) entries held in shared memory ----
// by_index = false: key (d2 bits, idx);  true: key idx only.
__device__ __forceinline__ void warp_bitonic(unsigned long long* d2, int* idx, int n, bool by_index, int lane) {
  for (int k = 2; k <= n; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int t = lane; t < n; t += 32) {
        const int l = t ^ j;
        if (l > t) {
          const unsigned long long a = d2[t], b = d2[l];
          const int ia = idx[t], ib = idx[l];
          const bool a_gt_b = by_index ? (ia > ib) : (a > b || (a == b && ia > ib));
          const bool up = (t & k) == 0;
          if (a_gt_b == up) {
            d2[t] = b; d2[l] = a;
            idx[t] = ib; idx[l] = ia;
          }
        }
      }
      __syncwarp();
    }
  }
}

constexpr unsigned long long kInfBits = 0x7ff0000000000000ull;
constexpr int kWarpsPerBlock = 4;

// Three-level test per candidate.  Level 0 (all candidates, 16 bytes and 6 flops each): the squared distance of the
// binning coordinates P^T e (the same fp32 values the grid was built from) against lambda r^2 with slack, lambda >= the
// largest eigenvalue of P^T P (1 for orthonormal P), so no pair with d2 <= r2 can fail it; a ball inside the 27 cells keeps
// ~15 % of them.  Survivors are queued and, 32 at a time, take level 1 (fp32 with FMA, all d_e coordinates): d2f <= r2 (1 + 1e-4).
// The fp32 value differs from the exact d2 by at most ~16 ulp relative (all terms are non-negative, so there is no
// cancellation), so no candidate with d2 <= r2 can fail it.  Survivors (a few per cent) are queued in shared memory and, 32 at
// a time, take level 2: the outer() test and the exact fp64 d2 (no FMA) that decides acceptance and rank.
//
// Candidates: for each of the (up to) 27 neighbouring spatial cells the contiguous range of hits whose radius bucket is >=
// the query's (lower buckets cannot be "outer", r_bucket()); empty ranges are skipped.
//
// Buffer of accepted neighbours (CAP = 2 K entries): when it cannot take 32 more, prune() bisects on d2 for a threshold T
// with K <= #{d2 <= T} <= CAP - 32, drops everything above T (none of it can be among the K nearest: K entries are at most
// T) and tightens the accept thresholds of all three levels to T.  Only when ties in d2 defeat the bisection the buffer is
// sorted by (d2, j) and cut to K; the exact K nearest by (d2, j) are selected once, at the end.
template <int D4, int CAP>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
frnn_search_kernel(const float* __restrict__ semb, const float4* __restrict__ smeta, const float4* __restrict__ sproj,
                   const int32_t* __restrict__ cell_start, const GridParams* __restrict__ gpp, double r2_in, float r2_loose_in,
                   float r_proj_in, float proj_scale, int K, int32_t* __restrict__ slots, int32_t* __restrict__ deg, int64_t n) {
  TRK_GRID_DEP_WAIT();
  constexpr int D = D4 * 4;
  constexpr int PER = CAP / 32;            // buffer entries per lane
  __shared__ unsigned long long s_d2[kWarpsPerBlock][CAP];
  __shared__ int s_idx[kWarpsPerBlock][CAP];
  __shared__ int s_queue[kWarpsPerBlock][64];
  __shared__ int s_queue0[kWarpsPerBlock][128];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t q = (int64_t)blockIdx.x * kWarpsPerBlock + warp;
  if (q >= n) return;
  unsigned long long* bd2 = s_d2[warp];
  int* bidx = s_idx[warp];
  int* queue = s_queue[warp];
  int* queue0 = s_queue0[warp];
  const GridParams gp = *gpp;
  const float4 qp = sproj[q];

  const float4 qm = smeta[q];
  const float q_r = qm.x, q_az = qm.y;
  const int q_i = __float_as_int(qm.z);
  int cell = __float_as_int(qm.w);
  const int q_b = cell % kRBuckets;        // the query's radius bucket
  cell /= kRBuckets;
  const int ev = cell / gp.cells_per_event;
  cell -= ev * gp.cells_per_event;
  const int cx = cell % gp.dims[0];
  const int cy = (cell / gp.dims[0]) % gp.dims[1];
  const int cz = cell / (gp.dims[0] * gp.dims[1]);
  float qf[D];
#pragma unroll
  for (int k4 = 0; k4 < D4; ++k4) {
    const float4 v = reinterpret_cast<const float4*>(semb + q * D)[k4];
    qf[k4 * 4 + 0] = v.x; qf[k4 * 4 + 1] = v.y; qf[k4 * 4 + 2] = v.z; qf[k4 * 4 + 3] = v.w;
  }

  int count = 0;  // warp-uniform number of buffered neighbours
  // both queues are rings (64 and 128 entries): entry i lives at (head + i) & (size - 1), so draining moves nothing
  int qn = 0, qh = 0;     // warp-uniform number / head of queued level-1 survivors
  int qn0 = 0, qh0 = 0;   // warp-uniform number / head of queued level-0 survivors
  // Thresholds shrink once K neighbours are known: a candidate with d2 above a value that K buffered entries do not exceed can
  // never enter the K nearest (equal d2 is kept and settled by the (d2, j) order at the end).
  double r2 = r2_in;
  // level-0 threshold on the binning coordinates: (sqrt(lambda) r, with the slack of the grid's cell edge)^2, rounded up
  const float r0_in = __fadd_ru(r_proj_in, gp.proj_eps);
  float r2_loose = r2_loose_in, r2_proj = __fmul_ru(r0_in, r0_in);
  auto tighten = [&](double kth) {
    if (kth < r2) {
      r2 = kth;
      r2_loose = fminf(r2_loose, __double2float_ru(kth * (1.0 + 1e-4)));
      const float r0 = __fadd_ru(__fmul_ru(proj_scale, __double2float_ru(sqrt(kth))), gp.proj_eps);
      r2_proj = fminf(r2_proj, __fmul_ru(r0, r0));
    }
  };
  for (int t = lane; t < CAP; t += 32) { bd2[t] = kInfBits; bidx[t] = 0x7fffffff; }
  __syncwarp();

  // keeps the entries with d2 <= T for a threshold T with K <= #{d2 <= T} <= max_keep (every entry that can still be among the K
  // nearest stays); max_keep = CAP - 32 makes room for 32 more entries, max_keep = K is the final selection of the K nearest
  auto prune = [&](int max_keep) {
    unsigned long long mine[PER];
#pragma unroll
    for (int i = 0; i < PER; ++i) mine[i] = bd2[lane + 32 * i];          // unused slots hold +inf
    // d2 >= 0, so the bit patterns order like the values; bisect on the value between 0 and the largest buffered d2
    unsigned long long mx = 0ull;
#pragma unroll
    for (int i = 0; i < PER; ++i) mx = (mine[i] != kInfBits && mine[i] > mx) ? mine[i] : mx;
    for (int o = 16; o > 0; o >>= 1) {
      const unsigned long long other = __shfl_xor_sync(0xffffffffu, mx, o);
      mx = other > mx ? other : mx;
    }
    double lo = 0.0, hi = __longlong_as_double((long long)mx);
    int cnt_hi = count;
    bool found = false;
    for (int it = 0; it < 48 && !found; ++it) {
      const double mid = 0.5 * (lo + hi);
      const unsigned long long mb = (unsigned long long)__double_as_longlong(mid);
      int c = 0;
#pragma unroll
      for (int i = 0; i < PER; ++i) c += mine[i] <= mb ? 1 : 0;
      c = __reduce_add_sync(0xffffffffu, c);
      if (c < K) {
        lo = mid;
      } else {
        hi = mid;
        cnt_hi = c;
        found = c <= max_keep;
      }
    }
    if (found) {
      // keep the entries with d2 <= hi, in place and in buffer order
      const unsigned long long hb = (unsigned long long)__double_as_longlong(hi);
      int idx[PER];
#pragma unroll
      for (int i = 0; i < PER; ++i) idx[i] = bidx[lane + 32 * i];
      __syncwarp();
      int base = 0;
#pragma unroll
      for (int i = 0; i < PER; ++i) {
        const bool keep = mine[i] <= hb;
        const unsigned m = __ballot_sync(0xffffffffu, keep);
        if (keep) {
          const int slot = base + __popc(m & ((1u << lane) - 1u));
          bd2[slot] = mine[i];
          bidx[slot] = idx[i];
        }
        base += __popc(m);
      }
      __syncwarp();
      for (int t = base + lane; t < CAP; t += 32) { bd2[t] = kInfBits; bidx[t] = 0x7fffffff; }
      __syncwarp();
      count = base;
      tighten(hi);
    } else {
      // ties in d2: the exact K nearest by (d2, j)
      warp_bitonic(bd2, bidx, CAP, false, lane);
      tighten(__longlong_as_double((long long)bd2[K - 1]));
      __syncwarp();
      for (int t = K + lane; t < CAP; t += 32) { bd2[t] = kInfBits; bidx[t] = 0x7fffffff; }
      __syncwarp();
      count = K;
    }
  };

  // level 2 on the first min(qn, 32) queued positions
  auto drain = [&]() {
    const int take = min(qn, 32);
    bool ok = false;
    double d2 = 0.0;
    int c_i = 0;
    if (lane < take) {
      const int pos = queue[(qh + lane) & 63];
      const float4 cm = smeta[pos];
      c_i = __float_as_int(cm.z);
      // outer(i,j): (r_i, |z_i|, i) < (r_j, |z_j|, j)
      const bool outer = (q_r < cm.x) || (q_r == cm.x && (q_az < cm.y || (q_az == cm.y && q_i < c_i)));
      if (outer) {
        const float4* ce = reinterpret_cast<const float4*>(semb + (int64_t)pos * D);
#pragma unroll
        for (int k4 = 0; k4 < D4; ++k4) {
          const float4 v = ce[k4];
          double t;
          t = __dsub_rn((double)qf[k4 * 4 + 0], (double)v.x); d2 = __dadd_rn(d2, __dmul_rn(t, t));
          t = __dsub_rn((double)qf[k4 * 4 + 1], (double)v.y); d2 = __dadd_rn(d2, __dmul_rn(t, t));
          t = __dsub_rn((double)qf[k4 * 4 + 2], (double)v.z); d2 = __dadd_rn(d2, __dmul_rn(t, t));
          t = __dsub_rn((double)qf[k4 * 4 + 3], (double)v.w); d2 = __dadd_rn(d2, __dmul_rn(t, t));
        }
        ok = d2 <= r2;
      }
    }
    qh = (qh + take) & 63;
    qn -= take;
    const unsigned m = __ballot_sync(0xffffffffu, ok);
    if (m) {
      if (count + 32 > CAP) {
        prune(CAP - 32);
        ok = ok && d2 <= r2;                 // the threshold may just have moved
      }
      const unsigned m2 = __ballot_sync(0xffffffffu, ok);
      if (ok) {
        const int slot = count + __popc(m2 & ((1u << lane) - 1u));
        bd2[slot] = (unsigned long long)__double_as_longlong(d2);
        bidx[slot] = c_i;
      }
      count += __popc(m2);
    }
    __syncwarp();
  };

  // level 1 on the first min(qn0, 32) queued level-0 survivors
  auto drain0 = [&]() {
    const int take = min(qn0, 32);
    bool pre = false;
    int pos = 0;
    if (lane < take) {
      pos = queue0[(qh0 + lane) & 127];
      const float4* ce = reinterpret_cast<const float4*>(semb + (int64_t)pos * D);
      float d2f = 0.f;
#pragma unroll
      for (int k4 = 0; k4 < D4; ++k4) {
        const float4 v = __ldg(ce + k4);
        float t;
        t = qf[k4 * 4 + 0] - v.x; d2f = fmaf(t, t, d2f);
        t = qf[k4 * 4 + 1] - v.y; d2f = fmaf(t, t, d2f);
        t = qf[k4 * 4 + 2] - v.z; d2f = fmaf(t, t, d2f);
        t = qf[k4 * 4 + 3] - v.w; d2f = fmaf(t, t, d2f);
      }
      pre = d2f <= r2_loose;
    }
    qh0 = (qh0 + take) & 127;
    qn0 -= take;
    const unsigned m = __ballot_sync(0xffffffffu, pre);
    if (m) {
      if (pre) queue[(qh + qn + __popc(m & ((1u << lane) - 1u))) & 63] = pos;
      qn += __popc(m);
      __syncwarp();
      if (qn >= 32) drain();
    }
    __syncwarp();
  };

  // the (up to) 27 neighbouring spatial cells: lane c < 27 fetches the candidate range of cell c -- its hits from the query's
  // radius bucket on -- so the dependent cell_start look-ups cost one memory latency
  int my_lo = 0, my_hi = 0;
  if (lane < 27) {
    const int z = cz + lane / 9 - 1, y = cy + (lane / 3) % 3 - 1, x = cx + lane % 3 - 1;
    if (z >= 0 && z < gp.dims[2] && y >= 0 && y < gp.dims[1] && x >= 0 && x < gp.dims[0]) {
      const int64_t sp = (int64_t)ev * gp.cells_per_event + (z * gp.dims[1] + y) * gp.dims[0] + x;
      my_lo = cell_start[sp * kRBuckets + q_b];
      my_hi = cell_start[(sp + 1) * kRBuckets];
    }
  }
  unsigned todo = __ballot_sync(0xffffffffu, my_hi > my_lo);
  while (todo) {
    const int rr = __ffs(todo) - 1;
    todo &= todo - 1;
    const int lo = __shfl_sync(0xffffffffu, my_lo, rr), hi = __shfl_sync(0xffffffffu, my_hi, rr);
    // two 32-candidate groups per trip: their loads are independent, the loop and queue bookkeeping is paid once
    for (int base = lo; base < hi; base += 64) {
      const int pos0 = base + lane, pos1 = base + 32 + lane;
      bool pre0 = false, pre1 = false;
      float4 cp0 = make_float4(0.f, 0.f, 0.f, 0.f), cp1 = cp0;
      if (pos0 < hi) cp0 = __ldg(sproj + pos0);
      if (pos1 < hi) cp1 = __ldg(sproj + pos1);
      {
        // both candidates of a lane in packed fp32x2 arithmetic: the same subtractions and fused multiply-adds, component by
        // component, as the scalar form (stale registers of an out-of-range position are masked by the range test)
        const float2 tx = __fadd2_rn(make_float2(qp.x, qp.x), make_float2(-cp0.x, -cp1.x));
        const float2 ty = __fadd2_rn(make_float2(qp.y, qp.y), make_float2(-cp0.y, -cp1.y));
        const float2 tz = __fadd2_rn(make_float2(qp.z, qp.z), make_float2(-cp0.z, -cp1.z));
        const float2 d = __ffma2_rn(tz, tz, __ffma2_rn(ty, ty, __fmul2_rn(tx, tx)));
        pre0 = pos0 < hi && d.x <= r2_proj;
        pre1 = pos1 < hi && d.y <= r2_proj;
      }
      const unsigned m0 = __ballot_sync(0xffffffffu, pre0), m1 = __ballot_sync(0xffffffffu, pre1);
      if (m0 | m1) {
        const unsigned lt = (1u << lane) - 1u;
        const int n0 = __popc(m0);
        if (pre0) queue0[(qh0 + qn0 + __popc(m0 & lt)) & 127] = pos0;
        if (pre1) queue0[(qh0 + qn0 + n0 + __popc(m1 & lt)) & 127] = pos1;
        qn0 += n0 + __popc(m1);
        __syncwarp();
        while (qn0 >= 32) drain0();       // at most 31 + 64 entries were queued: the ring of 128 cannot overflow
      }
    }
  }
  while (qn0 > 0) drain0();
  while (qn > 0) drain();
  if (count > K) prune(K);       // exactly the K nearest: a threshold between the K-th and the (K+1)-th d2, the sort only on ties
  // order the kept neighbours by index: the indices are distinct, so the rank of one is the number of smaller ones
  for (int t = lane; t < count; t += 32) {
    const int mine = bidx[t];
    int rank = 0;
    for (int u = 0; u < count; ++u) rank += bidx[u] < mine ? 1 : 0;
    slots[(int64_t)q_i * K + rank] = mine;
  }
  if (lane == 0) deg[q_i] = count;
}

__global__ void frnn_emit_kernel(const int32_t* __restrict__ slots, const int32_t* __restrict__ rowptr, int K,
                                 int32_t* __restrict__ src, int32_t* __restrict__ dst, int32_t* __restrict__ rowptr_out,
                                 int64_t capacity, int32_t* __restrict__ count_out, int32_t* __restrict__ overflow_flag, int64_t n) {
  TRK_GRID_DEP_WAIT();
  // one warp per hit
  const int lane = threadIdx.x & 31;
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i > n) return;
  if (i == n) {
    if (lane == 0) {
      const int64_t tot = rowptr[n];
      *count_out = (int32_t)min(tot, capacity);
      if (tot > capacity) *overflow_flag = 1;
      if (rowptr_out) rowptr_out[n] = (int32_t)min(tot, capacity);
    }
    return;
  }
  const int64_t b = rowptr[i], e = rowptr[i + 1];
  if (rowptr_out && lane == 0) rowptr_out[i] = (int32_t)min(b, capacity);
  for (int64_t t = lane; t < e - b; t += 32) {
    if (b + t < capacity) {
      src[b + t] = (int32_t)i;
      dst[b + t] = slots[i * K + t];
    }
  }
}

// Event offsets travel as a kernel parameter (by value), so trk_infer needs no staging copy and
// stays graph-capturable.
__global__ void event_of_hit_kernel(const __grid_constant__ EventOffsets offs, int n_events, int32_t* __restrict__ ev_of_hit, int64_t n) {
  TRK_GRID_DEP_WAIT();
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int lo = 0, hi = n_events;  // offsets[lo] <= i < offsets[hi]
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (offs.v[mid] <= i) lo = mid; else hi = mid;
  }
  ev_of_hit[i] = lo;
}

template <int D4>
trk_status launch_search(trk_ctx* ctx, int K, double r2, int64_t n, cudaStream_t st) {
  // level-0 radius on the binning coordinates: sqrt(lambda) r with the relative slack of the grid's cell edge (the kernel adds the
  // data-dependent rounding slack GridParams::proj_eps and squares)
  const double r0 = std::sqrt((double)ctx->proj_gain) * (double)ctx->cfg.frnn_radius * 1.001;
  const float r_proj = r0 >= 1.0e19 ? __builtin_inff() : nextafterf((float)r0, __builtin_inff());
  const float proj_scale = nextafterf((float)(std::sqrt((double)ctx->proj_gain) * 1.001), __builtin_inff());
  const unsigned blocks = (unsigned)ceil_div(n, kWarpsPerBlock);
  // level-1 threshold: r^2 (1 + 1e-4) rounded up, infinite when r^2 overflows fp32 (then every candidate takes level 2)
  const double loose = r2 * (1.0 + 1e-4);
  const float r2_loose = loose >= 3.0e38 ? __builtin_inff() : fmaxf(nextafterf((float)loose, __builtin_inff()), 1e-30f);
  if (K <= 32) {
    TRK_LAUNCH(ctx, (frnn_search_kernel<D4, 64>), blocks, kWarpsPerBlock * 32, 0, st, ctx->semb, ctx->smeta, ctx->sproj, ctx->cell_start,
               ctx->grid, r2, r2_loose, r_proj, proj_scale, K, ctx->slots, ctx->deg, n);
  } else if (K <= 64) {
    TRK_LAUNCH(ctx, (frnn_search_kernel<D4, 128>), blocks, kWarpsPerBlock * 32, 0, st, ctx->semb, ctx->smeta, ctx->sproj, ctx->cell_start,
               ctx->grid, r2, r2_loose, r_proj, proj_scale, K, ctx->slots, ctx->deg, n);
  } else {
    TRK_LAUNCH(ctx, (frnn_search_kernel<D4, 256>), blocks, kWarpsPerBlock * 32, 0, st, ctx->semb, ctx->smeta, ctx->sproj, ctx->cell_start,
               ctx->grid, r2, r2_loose, r_proj, proj_scale, K, ctx->slots, ctx->deg, n);
  }
  return TRK_OK;
}

}  // namespace

// ev_of_hit must already hold the event id of every hit (see set_event_ids in api.cu).
trk_status frnn_build(trk_ctx* ctx, const float* emb, const float* hits, int64_t n, int32_t n_events, int32_t* src,
                      int32_t* dst, int32_t* rowptr_out, int64_t capacity, int32_t* count_out, int32_t* overflow_flag,
                      cudaStream_t st) {
  const int K = ctx->cfg.frnn_k;
  const int g = ctx->grid_dims;
  const int G = ctx->grid_max;
  const int64_t n_cells = (int64_t)n_events * G * G * G * kRBuckets;
  if (n_cells > ctx->max_cells) return fail(ctx, TRK_ERR_CAPACITY, "frnn: n_events exceeds max_events");
  if (n <= 0) return fail(ctx, TRK_ERR_INVALID_ARG, "frnn: empty input");
  const unsigned nb = (unsigned)ceil_div(n, 256);
  // only the cells of this call's events are touched
  TRK_LAUNCH(ctx, frnn_reset_kernel, (unsigned)ceil_div(n_cells + 1, 256), 256, 0, st, ctx->bbox, ctx->cell_count, ctx->cell_fill,
             n_cells + 1);
  TRK_LAUNCH(ctx, frnn_project_kernel, nb, 256, 0, st, emb, hits, ctx->d_e, ctx->grid_proj, g, ctx->proj, ctx->bbox, n);
  TRK_LAUNCH(ctx, frnn_grid_setup_kernel, 1, 32, 0, st, ctx->bbox, ctx->cfg.frnn_radius, g, G, ctx->grid);
  TRK_LAUNCH(ctx, frnn_count_kernel, nb, 256, 0, st, ctx->proj, hits, ctx->ev_of_hit, ctx->grid, ctx->cell_of_hit, ctx->cell_count, n);
  TRK_TRY(exclusive_scan_i32(ctx, ctx->cell_count, ctx->cell_start, n_cells, ctx->scan_tmp, st));
  TRK_LAUNCH(ctx, frnn_scatter_kernel, nb, 256, 0, st, emb, hits, ctx->d_e, ctx->d_e_pad, ctx->cell_of_hit, ctx->cell_start,
             ctx->cell_fill, ctx->semb, ctx->smeta, ctx->proj, ctx->sproj, n);
  const double r = (double)ctx->cfg.frnn_radius;
  const double r2 = r * r;
  switch (ctx->d_e_pad / 4) {
    case 1: TRK_TRY(launch_search<1>(ctx, K, r2, n, st)); break;
    case 2: TRK_TRY(launch_search<2>(ctx, K, r2, n, st)); break;
    case 3: TRK_TRY(launch_search<3>(ctx, K, r2, n, st)); break;
    default: TRK_TRY(launch_search<4>(ctx, K, r2, n, st)); break;
  }
  TRK_TRY(exclusive_scan_i32(ctx, ctx->deg, ctx->rowptr, n, ctx->scan_tmp, st));
  TRK_LAUNCH(ctx, frnn_emit_kernel, (unsigned)ceil_div((n + 1) * 32, 256), 256, 0, st, ctx->slots, ctx->rowptr, K, src, dst,
             rowptr_out, capacity, count_out, overflow_flag, n);
  return TRK_OK;
}

trk_status set_event_ids(trk_ctx* ctx, const int32_t* offsets_host, int n_events, int64_t n, cudaStream_t st) {
  if (n <= 0) return TRK_OK;
  EventOffsets offs;
  for (int i = 0; i <= n_events; ++i) offs.v[i] = offsets_host[i];
  TRK_LAUNCH(ctx, event_of_hit_kernel, (unsigned)ceil_div(n, 256), 256, 0, st, offs, n_events, ctx->ev_of_hit, n);
  return TRK_OK;
}

}  // namespace trk

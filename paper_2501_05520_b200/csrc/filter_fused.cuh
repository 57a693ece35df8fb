// S3 filter MLP as ONE persistent CTA-pair kernel:   score = sigmoid(MLP([u_src ; u_dst])),
// MLP = 2u -> W -> W -> W -> 1 with ReLU, W a multiple of 256 (1024 in BASELINE.json's pileup configs).
//
// A CTA pair owns 256-row blocks of candidate edges (row block rb = pair, pair + n_pairs, ...) and runs ALL layers of a row
// block itself, so no activation of one pair is ever read by another and nothing needs a grid-wide synchronisation.  Per row
// block the tensor core walks 3 x W/256 tiles of 256 x 256 (tcgen05.mma.cta_group::2, accumulators double-buffered in TMEM):
//   layer 1 (K = 2u <= 32)  A = the gathered rows [u_src ; u_dst] rounded to bf16, written by four gather warps straight into a
//                           swizzled operand tile (one K block, only ceil(2u/16) K steps are issued); epilogue bias + ReLU ->
//                           bf16 -> act1 by TMA store;
//   layer 2 (K = W)         A = act1 by TMA; epilogue bias + ReLU -> bf16 -> act2 by TMA store;
//   layer 3 (K = W)         A = act2; the epilogue folds the final Linear(W -> 1) in: every thread keeps the running dot of its row
//                           over the column tiles and writes sigmoid(dot + b) after the last one.
// act1 / act2 are per-pair scratch of 256 x W bf16 each in global memory (n_pairs x 2 x 512 KB = 74 MB for W = 1024 on 148
// SMs): they are rewritten for every row block and are always read back from the 126 MB L2, so the stage reads from HBM only
// the gather, the indices and the weights once -- against one HBM round trip of the 2 KB activation row per layer before.
//
// Dependencies inside a pair (mbarriers; a CTA's epilogue warps and TMA producer only ever touch their own CTA's 128 rows of the
// scratch, so the slab barriers are CTA-local):
//   xfull / xempty      gather warps <-> MMA issuer: the layer-1 operand tile of the next row block (single buffer: it is free
//                       again as soon as the W/256 short layer-1 MMAs of the current row block have been issued and completed)
//   act1_ready[s], act2_ready[s]   epilogue warps (after their TMA stores of column slab s have COMPLETED) -> TMA producer: the
//                       next layer may load the K blocks of slab s.  A layer's first K blocks come from the slabs stored first,
//                       so the tensor pipe does not wait for the last epilogue of the layer before.
// Writes by TMA store and reads by TMA load of the same CTA are ordered by cp.async.bulk.wait_group (completion, not .read)
// followed by the mbarrier.
#pragma once

#include "gemm_tc2.cuh"

namespace trk {
namespace ff {

using namespace tc;

constexpr int kGatherWarpsF = 4;
constexpr int kThreadsFilter = kThreads + 32 * kGatherWarpsF;   // 0 TMA, 1 MMA, 2-5 epilogue, 6-9 gather
constexpr int kBN = 256;
constexpr int kStages = 5;
constexpr int kStage = stage_bytes_pair(kBN);                  // A 16 KB + this CTA's half of W 16 KB
constexpr int kXBytes = BM * BK * 2;                           // layer-1 operand tile of one CTA
constexpr int kMaxSlabs = 4;                                   // W <= 1024
constexpr int kMaxW = kMaxSlabs * kBN;
constexpr int kVecBytes = 4 * kMaxW * 4;                       // b1, b2, b3, w4 in shared memory
constexpr int kSmemFilter = kStages * kStage + kXBytes + kEpiWarps * kStoreStage + kVecBytes + 1024 /*alignment*/ + 1024 /*barriers, dot exchange*/;
static_assert(kSmemFilter <= 232448, "shared memory budget of one CTA");

struct FilterParams {
  const float* feat;          // fp32 [n][u]: the embedding (or the raw hits)
  const int32_t* src;         // candidate edges
  const int32_t* dst;
  int u;                      // 2 u <= 32
  const float* b1;            // [W]
  const float* b2;            // [W]
  const float* b3;            // [W]
  const float* w4;            // [W] final Linear(W -> 1)
  float b4;
  float* score;               // [rows]
  int W;
};

struct FilterBars {
  uint64_t full[8];
  uint64_t empty[8];
  uint64_t tfull[2];
  uint64_t tempty[2];
  uint64_t xfull;                   // L  8 arrivals (4 gather warps x 2 CTAs)
  uint64_t xempty;                  //    own, multicast commit
  uint64_t act1_ready[kMaxSlabs];   //    own, 4 arrivals each (epilogue warps)
  uint64_t act2_ready[kMaxSlabs];
  uint32_t tmem_slot;
  float dots[BM];                   // layer 3: the helper warps' half of each row's dot product
};
static_assert(sizeof(FilterBars) <= 1024, "barrier block");

__device__ __forceinline__ uint32_t pack_relu_bf16x2(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
// L2 eviction priority for the activation scratch: it is rewritten every row block and should not leave the L2 in between
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void tma_store_2d_hint(const CUtensorMap* tmap, const void* smem_src, int c0, int c1, uint64_t pol) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%2, %3}], [%1], %4;" ::"l"(
                   reinterpret_cast<uint64_t>(tmap)),
               "r"(smem_u32(smem_src)), "r"(c0), "r"(c1), "l"(pol)
               : "memory");
}
__device__ __forceinline__ void tma_load_2d_pair_hint(void* smem_dst, const CUtensorMap* tmap, uint32_t bar_cluster_addr, int c0, int c1,
                                                      uint64_t pol) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4}], [%2], %5;" ::"r"(
          smem_u32(smem_dst)),
      "l"(reinterpret_cast<uint64_t>(tmap)), "r"(bar_cluster_addr), "r"(c0), "r"(c1), "l"(pol)
      : "memory");
}
__device__ __forceinline__ void mbar_arrive_remote_cta(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}

// cluster-scope release: the gathered layer-1 operand rows of this CTA are consumed by an MMA issued from the leader CTA
__device__ __forceinline__ void mbar_arrive_remote_release_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}

constexpr int kTemptyArrivals = 2 * kEpiWarps;   // per CTA and tile: 4 epilogue warps x 2 (layers 1, 2) or 4 + 4 helper warps (layer 3)

// sum over 128 accumulator columns of this thread's TMEM lane of ReLU(acc + b) * w, added to `dot`; releases the accumulator
// (one arrival per warp on the leader's tempty barrier) as soon as the last column has been read
__device__ __forceinline__ float relu_dot_half(uint32_t taddr, const float* __restrict__ sb, const float* __restrict__ sw, float dot,
                                               uint32_t rel, int lane) {
#pragma unroll 1
  for (int c = 0; c < kBN / 2; c += 32) {
    uint32_t r[32];
    tmem_ld32(taddr + c, r);
    const float4* b4 = reinterpret_cast<const float4*>(sb + c);
    const float4* w4 = reinterpret_cast<const float4*>(sw + c);
    float4 bb[8], ww[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) { bb[q] = b4[q]; ww[q] = w4[q]; }
    tmem_ld_wait();
    if (c + 32 >= kBN / 2) {
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(rel);
    }
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      dot = fmaf(fmaxf(__uint_as_float(r[q * 4 + 0]) + bb[q].x, 0.f), ww[q].x, dot);
      dot = fmaf(fmaxf(__uint_as_float(r[q * 4 + 1]) + bb[q].y, 0.f), ww[q].y, dot);
      dot = fmaf(fmaxf(__uint_as_float(r[q * 4 + 2]) + bb[q].z, 0.f), ww[q].z, dot);
      dot = fmaf(fmaxf(__uint_as_float(r[q * 4 + 3]) + bb[q].w, 0.f), ww[q].w, dot);
    }
  }
  return dot;
}

// The tile schedule of one CTA pair, the same for every warp role (so accumulator indices and barrier phases agree):
//   layer 1 of the pair's first row block (n_tiles short tiles), then for every row block i:
//     layer 2: n_tiles tiles;   then  layer 3 tile 0, layer 1 tile 0 OF ROW BLOCK i+1, layer 3 tile 1, layer 1 tile 1 of i+1, ...
// Layer 1 of the next row block rides inside the layer-3 phase: act1 is free then (layer 2 has read it), its epilogues (bias,
// ReLU, bf16, TMA store of 256 x 256 values for a few hundred cycles of MMA) overlap the long layer-3 MMAs instead of standing
// alone, and the next layer 2 finds its operand stored.  f(layer, rb index, column tile).
template <class F>
__device__ __forceinline__ void for_each_tile(int n_rb, int n_tiles, F f) {
  if (n_rb <= 0) return;
  for (int nb = 0; nb < n_tiles; ++nb) f(1, 0, nb);
  for (int i = 0; i < n_rb; ++i) {
    for (int nb = 0; nb < n_tiles; ++nb) f(2, i, nb);
    for (int nb = 0; nb < n_tiles; ++nb) {
      f(3, i, nb);
      if (i + 1 < n_rb) f(1, i + 1, nb);
    }
  }
}

__device__ __forceinline__ void named_bar_sync(int id, int threads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

// tmS1 / tmS2: the act1 / act2 scratch as A operands (box 64 x 128); tmW1 (K padded to 64) / tmW2 / tmW3: weights (box 64 x 128 =
// this CTA's half of a 256-column tile); tmS1st / tmS2st: the scratch for the TMA stores of the epilogues (box 64 x 32).
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreadsFilter, 1)
filter_mlp_kernel(const __grid_constant__ CUtensorMap tmS1, const __grid_constant__ CUtensorMap tmS2, const __grid_constant__ CUtensorMap tmW1,
                  const __grid_constant__ CUtensorMap tmW2, const __grid_constant__ CUtensorMap tmW3, const __grid_constant__ CUtensorMap tmS1st,
                  const __grid_constant__ CUtensorMap tmS2st, Rows rows, FilterParams p) {
  TRK_GRID_DEP_WAIT();
  constexpr int A_BYTES = BM * BK * 2;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint8_t* xbuf = smem + kStages * kStage;
  uint8_t* store_stage = xbuf + kXBytes;
  float* svec = reinterpret_cast<float*>(store_stage + kEpiWarps * kStoreStage);   // [4][kMaxW]: b1, b2, b3, w4
  FilterBars* bar = reinterpret_cast<FilterBars*>(reinterpret_cast<uint8_t*>(svec) + kVecBytes);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const bool leader = rank == 0;
  const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
  const int64_t M = resolve_rows(rows);
  const int64_t m_tiles = (M + kPairBM - 1) / kPairBM;
  const int n_rb = pair < m_tiles ? (int)((m_tiles - pair + n_pairs - 1) / n_pairs) : 0;   // row blocks of this pair
  const int n_tiles = p.W / kBN;          // column tiles (= slabs) per layer
  const int k_blocks = p.W / BK;
  const int kb_per_slab = kBN / BK;
  const int k1_steps = (2 * p.u + UMMA_K - 1) / UMMA_K;      // K steps of layer 1 that hold data
  const int scratch_row0 = pair * kPairBM + (int)rank * BM;  // this CTA's rows of the scratch

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmS1); prefetch_tmap(&tmS2); prefetch_tmap(&tmW1); prefetch_tmap(&tmW2); prefetch_tmap(&tmW3);
    prefetch_tmap(&tmS1st); prefetch_tmap(&tmS2st);
    for (int s = 0; s < kStages; ++s) {
      mbar_init(&bar->full[s], 1);
      mbar_init(&bar->empty[s], 1);
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(&bar->tfull[s], 1);
      mbar_init(&bar->tempty[s], 2 * kTemptyArrivals);
    }
    mbar_init(&bar->xfull, 2 * kGatherWarpsF);
    mbar_init(&bar->xempty, 1);
    for (int s = 0; s < kMaxSlabs; ++s) {
      mbar_init(&bar->act1_ready[s], kEpiWarps);
      mbar_init(&bar->act2_ready[s], kEpiWarps);
    }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc_pair<512>(&bar->tmem_slot);
  for (int c = threadIdx.x; c < p.W; c += blockDim.x) {
    svec[c] = p.b1[c];
    svec[kMaxW + c] = p.b2[c];
    svec[2 * kMaxW + c] = p.b3[c];
    svec[3 * kMaxW + c] = p.w4[c];
  }
  __syncthreads();
  tc_fence_before();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = bar->tmem_slot;

  if (warp == 0) {
    // ---------------------------------------------------------------- TMA producer
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      const uint64_t keep = l2_policy_evict_last();
      auto next_stage = [&]() { if (++stage == kStages) { stage = 0; phase ^= 1; } };
      for_each_tile(n_rb, n_tiles, [&](int layer, int i, int nb) {
        if (layer == 1) {
          // only this CTA's half of the W1 tile travels through the ring (the A operand is the gathered tile)
          mbar_wait(&bar->empty[stage], phase ^ 1);
          if (leader) mbar_arrive_expect_tx(&bar->full[stage], 2 * (kStage - A_BYTES));
          const uint32_t full_leader = mapa_u32(smem_u32(&bar->full[stage]), 0);
          tma_load_2d_pair(smem + stage * kStage + A_BYTES, &tmW1, full_leader, 0, nb * kBN + (int)rank * (kBN / 2));
          next_stage();
          return;
        }
        const CUtensorMap* tmA = layer == 2 ? &tmS1 : &tmS2;
        const CUtensorMap* tmB = layer == 2 ? &tmW2 : &tmW3;
        uint64_t* ready = layer == 2 ? bar->act1_ready : bar->act2_ready;
        for (int kb = 0; kb < k_blocks; ++kb) {
          // the first column tile of a layer is the first reader of its operand: slab by slab as the stores complete
          if (nb == 0 && kb % kb_per_slab == 0) mbar_wait(&ready[kb / kb_per_slab], (uint32_t)(i & 1));
          mbar_wait(&bar->empty[stage], phase ^ 1);
          if (leader) mbar_arrive_expect_tx(&bar->full[stage], 2 * kStage);
          const uint32_t full_leader = mapa_u32(smem_u32(&bar->full[stage]), 0);
          uint8_t* sa = smem + stage * kStage;
          tma_load_2d_pair_hint(sa, tmA, full_leader, kb * BK, scratch_row0, keep);
          tma_load_2d_pair(sa + A_BYTES, tmB, full_leader, kb * BK, nb * kBN + (int)rank * (kBN / 2));
          next_stage();
        }
      });
    }
  } else if (warp == 1) {
    // ---------------------------------------------------------------- MMA issuer (leader CTA)
    if (leader && lane == 0) {
      constexpr uint32_t idesc = make_idesc_pair(kBN);
      int stage = 0;
      uint32_t phase = 0;
      int as = 0;
      uint32_t aphase = 0;
      auto next_stage = [&]() { if (++stage == kStages) { stage = 0; phase ^= 1; } };
      const uint64_t xdesc = make_smem_desc(smem_u32(xbuf));
      for_each_tile(n_rb, n_tiles, [&](int layer, int i, int nb) {
        if (layer == 1 && nb == 0) mbar_wait_cluster(&bar->xfull, (uint32_t)(i & 1));   // both CTAs' gathered rows of row block i
        mbar_wait_cluster(&bar->tempty[as], aphase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(as * kBN);
        if (layer == 1) {
          mbar_wait(&bar->full[stage], phase);
          tc_fence_after();
          const uint64_t bdesc = make_smem_desc(smem_u32(smem + stage * kStage) + A_BYTES);
          for (int k = 0; k < k1_steps; ++k)
            tc_mma_bf16_pair(d_tmem, xdesc + (uint64_t)(k * 2), bdesc + (uint64_t)(k * 2), idesc, k != 0 ? 1u : 0u);
          tc_commit_pair(&bar->empty[stage]);
          next_stage();
          if (nb == n_tiles - 1) tc_commit_pair(&bar->xempty);     // the gathered tile may be overwritten
        } else {
          for (int kb = 0; kb < k_blocks; ++kb) {
            mbar_wait(&bar->full[stage], phase);
            tc_fence_after();
            const uint32_t sa = smem_u32(smem + stage * kStage);
            const uint64_t adesc = make_smem_desc(sa);
            const uint64_t bdesc = make_smem_desc(sa + A_BYTES);
#pragma unroll
            for (int k = 0; k < BK / UMMA_K; ++k)
              tc_mma_bf16_pair(d_tmem, adesc + (uint64_t)(k * 2), bdesc + (uint64_t)(k * 2), idesc, (kb | k) != 0 ? 1u : 0u);
            tc_commit_pair(&bar->empty[stage]);
            next_stage();
          }
        }
        tc_commit_pair(&bar->tfull[as]);
        if (++as == 2) { as = 0; aphase ^= 1; }
      });
    }
  } else if (warp < 2 + kEpiWarps) {
    // ---------------------------------------------------------------- epilogue warps
    const int quad = warp & 3;
    int as = 0;
    uint32_t aphase = 0;
    uint8_t* stage_buf = store_stage + (warp - 2) * kStoreStage;
    const uint64_t keep = l2_policy_evict_last();
    const uint32_t tempty_leader0 = mapa_u32(smem_u32(&bar->tempty[0]), 0);
    const uint32_t tempty_leader1 = mapa_u32(smem_u32(&bar->tempty[1]), 0);
    // The TMA stores of a tile are only ASKED about at the start of the next tile's epilogue (a whole tile of MMAs later they
    // have long completed), so the epilogue never sits in the store latency; the last tile of a layer asks at once, because the
    // very next tile of the schedule is the first reader of that slab.
    uint64_t* pending = nullptr;
    float dot = 0.f;
    for_each_tile(n_rb, n_tiles, [&](int layer, int i, int nb) {
      mbar_wait(&bar->tfull[as], aphase);
      tc_fence_after();
      if (pending) {
        if (lane == 0) {
          bulk_wait_all();
          mbar_arrive(pending);
        }
        pending = nullptr;
      }
      const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(as * kBN);
      const uint32_t rel = as == 0 ? tempty_leader0 : tempty_leader1;
      if (layer < 3) {
        // bias + ReLU -> bf16 -> act1 / act2 (this warp's 32 rows x 256 columns, 64 columns per TMA store box)
        const float* bias = svec + (layer == 1 ? 0 : kMaxW) + nb * kBN;
        const CUtensorMap* tmC = layer == 1 ? &tmS1st : &tmS2st;
        uint32_t chunk = 0;
#pragma unroll 1
        for (int c = 0; c < kBN; c += 64) {
          uint32_t ra[32], rb2[32];
          tmem_ld32(taddr + c, ra);
          tmem_ld32(taddr + c + 32, rb2);
          uint8_t* buf = stage_buf + (chunk & 1u) * (kStoreStage / 2);
          if (chunk >= 2) {          // the box staged two chunks ago must have left shared memory
            if (lane == 0) bulk_wait_read<1>();
            __syncwarp();
          }
          const float4* b4 = reinterpret_cast<const float4*>(bias + c);
          float4 bb[16];
#pragma unroll
          for (int j = 0; j < 16; ++j) bb[j] = b4[j];
          tmem_ld_wait();
          if (c + 64 >= kBN) {
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {      // this warp stands for two arrivals: the helper warps only take part in layer-3 tiles
              mbar_arrive_cluster(rel);
              mbar_arrive_cluster(rel);
            }
          }
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            uint32_t w[4];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              const float4 b = bb[q * 2 + h];
              const uint32_t* r = (q < 4 ? ra : rb2) + (q & 3) * 8 + h * 4;
              w[h * 2 + 0] = pack_relu_bf16x2(__uint_as_float(r[0]) + b.x, __uint_as_float(r[1]) + b.y);
              w[h * 2 + 1] = pack_relu_bf16x2(__uint_as_float(r[2]) + b.z, __uint_as_float(r[3]) + b.w);
            }
            *reinterpret_cast<uint4*>(buf + lane * 128 + ((q ^ (lane & 7)) << 4)) = make_uint4(w[0], w[1], w[2], w[3]);
          }
          fence_proxy_async();
          __syncwarp();
          if (lane == 0) {
            tma_store_2d_hint(tmC, buf, nb * kBN + c, scratch_row0 + quad * 32, keep);
            bulk_commit();
          }
          ++chunk;
        }
        // slab nb is complete for this warp's rows once its stores have landed
        uint64_t* ready = layer == 1 ? &bar->act1_ready[nb] : &bar->act2_ready[nb];
        if (nb == n_tiles - 1) {
          if (lane == 0) {
            bulk_wait_all();
            mbar_arrive(ready);
          }
        } else {
          pending = ready;
        }
        __syncwarp();
      } else {
        // ReLU(acc + b3) . w4 over columns [0, 128) of this tile (the helper warp of the same lane quadrant takes [128, 256)),
        // accumulated over the column tiles in the thread's register
        if (nb == 0) dot = 0.f;
        dot = relu_dot_half(taddr, svec + 2 * kMaxW + nb * kBN, svec + 3 * kMaxW + nb * kBN, dot, rel, lane);
        if (nb == n_tiles - 1) {
          // the helper warp of this lane quadrant holds the other half of the row's dot product
          named_bar_sync(1 + quad, 64);
          const float other = bar->dots[quad * 32 + lane];
          const int64_t rb = pair + (int64_t)i * n_pairs;
          const int64_t row = rb * kPairBM + (int64_t)rank * BM + quad * 32 + lane;
          if (row < M) p.score[rows.m_off + row] = fast_sigmoid(dot + other + p.b4);
          __syncwarp();
        }
      }
      if (++as == 2) { as = 0; aphase ^= 1; }
    });
  } else {
    // ---------------------------------------------------------------- helper warps: gather the layer-1 operand rows (one row per
    // thread) and take the upper half of the columns in the layer-3 epilogues
    const int hw = warp - (2 + kEpiWarps);
    const int quad = warp & 3;                       // TMEM lane quadrant this warp may read (the epilogue warp with the same quadrant is its partner)
    const int r = hw * 32 + lane;                    // operand row written by this thread
    const int u = p.u;
    const uint32_t xfull_leader = mapa_u32(smem_u32(&bar->xfull), 0);
    const uint32_t tempty_leader0 = mapa_u32(smem_u32(&bar->tempty[0]), 0);
    const uint32_t tempty_leader1 = mapa_u32(smem_u32(&bar->tempty[1]), 0);
    uint8_t* rowp = xbuf + r * 128;
    auto gather = [&](int i) {
      const int64_t rb = pair + (int64_t)i * n_pairs;
      const int64_t row = rb * kPairBM + (int64_t)rank * BM + r;
      float v[32];
#pragma unroll
      for (int c = 0; c < 32; ++c) v[c] = 0.f;
      if (row < M) {
        const int64_t si = p.src[rows.m_off + row], di = p.dst[rows.m_off + row];
        const float* fs = p.feat + si * u;
        const float* fd = p.feat + di * u;
#pragma unroll
        for (int c = 0; c < 16; ++c)
          if (c < u) v[c] = __ldg(fs + c);
#pragma unroll
        for (int c = 0; c < 32; ++c)
          if (c >= u && c < 2 * u) v[c] = __ldg(fd + (c - u));
      }
      uint32_t pk[16];
#pragma unroll
      for (int c = 0; c < 16; ++c) pk[c] = pack_bf16(v[2 * c], v[2 * c + 1]);
      if (i > 0) mbar_wait(&bar->xempty, (uint32_t)((i - 1) & 1));   // the layer-1 MMAs of the previous row block have read the tile
#pragma unroll
      for (int q = 0; q < 4; ++q)
        *reinterpret_cast<uint4*>(rowp + ((q ^ (r & 7)) << 4)) = make_uint4(pk[q * 4], pk[q * 4 + 1], pk[q * 4 + 2], pk[q * 4 + 3]);
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive_remote_release_cluster(xfull_leader);
    };
    int as = 0;
    uint32_t aphase = 0;
    float dot = 0.f;
    if (n_rb > 0) gather(0);
    for_each_tile(n_rb, n_tiles, [&](int layer, int i, int nb) {
      // the operand of row block i+1 is gathered while layer 2 of row block i runs (its layer-1 tiles follow in the layer-3 phase)
      if (layer == 2 && nb == 0 && i + 1 < n_rb) gather(i + 1);
      // every tile's accumulator barrier is waited for, also where this warp has nothing to do: a parity wait that skipped a
      // phase could be satisfied by an older one
      mbar_wait(&bar->tfull[as], aphase);
      if (layer == 3) {
        tc_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(as * kBN + kBN / 2);
        if (nb == 0) dot = 0.f;
        dot = relu_dot_half(taddr, svec + 2 * kMaxW + nb * kBN + kBN / 2, svec + 3 * kMaxW + nb * kBN + kBN / 2, dot,
                            as == 0 ? tempty_leader0 : tempty_leader1, lane);
        if (nb == n_tiles - 1) {
          bar->dots[quad * 32 + lane] = dot;
          named_bar_sync(1 + quad, 64);
        }
      }
      if (++as == 2) { as = 0; aphase ^= 1; }
    });
  }
  if (warp >= 2 && warp < 2 + kEpiWarps && lane == 0) bulk_wait_all();
  tc_fence_before();
  cluster_sync_all();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_pair<512>(tmem_base);
  }
}

}  // namespace ff
}  // namespace trk

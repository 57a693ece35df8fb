// S3 filter MLP as ONE persistent CTA-pair kernel:   score = sigmoid(MLP([u_src ; u_dst])),
// MLP = 2u -> W -> W -> W -> 1 with ReLU, W a multiple of 256 (1024 in BASELINE.json's pileup configs).
//
// A CTA pair owns 256-row blocks of candidate edges (row block rb = pair, pair + n_pairs, ...) and runs ALL layers of a row
// block itself, so no activation of one pair is ever read by another and nothing needs a grid-wide synchronisation:
//   layer 1 (K = 2u <= 32)  four "side" warps per CTA: the gathered, bf16-rounded rows [u_src ; u_dst] live in mma.sync
//                           A fragments in registers, W1 streams from L2 in fragment order; bias + ReLU -> bf16 -> act1;
//   layer 2 (K = W)         tcgen05.mma.cta_group::2, 256 x 256 tiles, A = act1 by TMA, epilogue bias + ReLU -> bf16 -> act2
//                           by TMA store;
//   layer 3 (K = W)         same MMAs with A = act2; the epilogue folds the final Linear(W -> 1) in: every thread keeps the
//                           running dot of its row over the column tiles and writes sigmoid(dot + b) after the last one.
// act1 / act2 are per-pair scratch of 256 x W bf16 each in global memory (n_pairs x 2 x 512 KB = 74 MB for W = 1024 on 148
// SMs): they are rewritten for every row block and stay in the 126 MB L2, so the only HBM traffic of the stage is the gather,
// the indices and the scores -- against one HBM round trip of the 2 KB activation row per layer before.
//
// Dependencies inside a pair (all mbarriers; the side warps and the TMA producer of a CTA only ever touch their own CTA's 128
// rows of the scratch, so every one of them is CTA-local):
//   act1_ready     side warps -> TMA producer: layer-1 rows of the NEXT row block are in global memory
//   l2_done        MMA issuer (commit after the last layer-2 tile) -> side warps: act1 may be overwritten
//   act2_ready[s]  epilogue warps (after their TMA stores of column slab s completed) -> TMA producer: layer 3 may load the
//                  K blocks of slab s.  Layer 3's first K blocks come from the slabs stored first, so the tensor pipe does not
//                  wait for the last layer-2 epilogue.
// Writes by TMA store and reads by TMA load of the same CTA are ordered by cp.async.bulk.wait_group (completion, not .read);
// the side warps' st.global are made visible to the TMA loads by fence.proxy.async + the mbarrier.
#pragma once

#include "gemm_tc2.cuh"

namespace trk {
namespace ff {

using namespace tc;

constexpr int kSideWarps = 4;
constexpr int kThreadsFilter = kThreads + 32 * kSideWarps;   // 0 TMA, 1 MMA, 2-5 epilogue, 6-9 layer 1
constexpr int kBN = 256;
constexpr int kStages = num_stages_pair(kBN);
constexpr int kStage = stage_bytes_pair(kBN);
constexpr int kSmemFilter = kStages * kStage + kEpiWarps * kStoreStage + 1024 /*alignment*/ + 512 /*barriers*/;
constexpr int kMaxSlabs = 4;                                  // W <= 1024

struct FilterParams {
  const float* feat;          // fp32 [n][u]: the embedding (or the raw hits)
  const int32_t* src;         // candidate edges
  const int32_t* dst;
  int u;                      // 2 u <= 32
  const uint4* w1_frag;       // layer 1 weights in mma.sync B-fragment order: [W / 8][32 lanes] x {b0, b1 (k 0..15), b0, b1 (k 16..31)}
  const float* b1;            // [W]
  const float* b2;            // [W]
  const float* b3;            // [W]
  const float* w4;            // [W] final Linear(W -> 1)
  float b4;
  __nv_bfloat16* act1;        // scratch [n_pairs * 256][W]
  float* score;               // [rows]
  int W;
};

struct FilterBars {
  uint64_t full[8];
  uint64_t empty[8];
  uint64_t tfull[2];
  uint64_t tempty[2];
  uint64_t act1_ready;        // 4 arrivals (side warps)
  uint64_t l2_done;           // multicast commit
  uint64_t act2_ready[kMaxSlabs];   // 4 arrivals each (epilogue warps)
  uint32_t tmem_slot;
};
static_assert(sizeof(FilterBars) <= 512, "barrier block");

__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }

__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

__device__ __forceinline__ uint32_t pack_relu_bf16x2(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

// tmS1 / tmS2: the act1 / act2 scratch as A operands (box 64 x 128); tmW2 / tmW3: weights (box 64 x 128 = this CTA's half of a
// 256-column tile); tmS2st: act2 for the TMA stores of the layer-2 epilogue (box 64 x 32).
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreadsFilter, 1)
filter_mlp_kernel(const __grid_constant__ CUtensorMap tmS1, const __grid_constant__ CUtensorMap tmS2, const __grid_constant__ CUtensorMap tmW2,
                  const __grid_constant__ CUtensorMap tmW3, const __grid_constant__ CUtensorMap tmS2st, Rows rows, FilterParams p) {
  constexpr int A_BYTES = BM * BK * 2;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint8_t* store_stage = smem + kStages * kStage;
  FilterBars* bar = reinterpret_cast<FilterBars*>(store_stage + kEpiWarps * kStoreStage);

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
  const int scratch_row0 = pair * kPairBM + (int)rank * BM;   // this CTA's rows of the scratch

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmS1); prefetch_tmap(&tmS2); prefetch_tmap(&tmW2); prefetch_tmap(&tmW3); prefetch_tmap(&tmS2st);
    for (int s = 0; s < kStages; ++s) {
      mbar_init(&bar->full[s], 1);
      mbar_init(&bar->empty[s], 1);
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(&bar->tfull[s], 1);
      mbar_init(&bar->tempty[s], 2 * kEpiWarps);
    }
    mbar_init(&bar->act1_ready, kSideWarps);
    mbar_init(&bar->l2_done, 1);
    for (int s = 0; s < kMaxSlabs; ++s) mbar_init(&bar->act2_ready[s], kEpiWarps);
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc_pair<512>(&bar->tmem_slot);
  tc_fence_before();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = bar->tmem_slot;

  if (warp == 0) {
    // ---------------------------------------------------------------- TMA producer
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int i = 0; i < n_rb; ++i) {
        for (int layer = 2; layer <= 3; ++layer) {
          const CUtensorMap* tmA = layer == 2 ? &tmS1 : &tmS2;
          const CUtensorMap* tmB = layer == 2 ? &tmW2 : &tmW3;
          for (int nb = 0; nb < n_tiles; ++nb) {
            for (int kb = 0; kb < k_blocks; ++kb) {
              if (nb == 0) {   // the first column tile of a layer is the first reader of its operand
                if (layer == 2 && kb == 0) mbar_wait(&bar->act1_ready, (uint32_t)(i & 1));
                if (layer == 3 && kb % kb_per_slab == 0) mbar_wait(&bar->act2_ready[kb / kb_per_slab], (uint32_t)(i & 1));
              }
              mbar_wait(&bar->empty[stage], phase ^ 1);
              if (leader) mbar_arrive_expect_tx(&bar->full[stage], 2 * kStage);
              const uint32_t full_leader = mapa_u32(smem_u32(&bar->full[stage]), 0);
              uint8_t* sa = smem + stage * kStage;
              tma_load_2d_pair(sa, tmA, full_leader, kb * BK, scratch_row0);
              tma_load_2d_pair(sa + A_BYTES, tmB, full_leader, kb * BK, nb * kBN + (int)rank * (kBN / 2));
              if (++stage == kStages) { stage = 0; phase ^= 1; }
            }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ---------------------------------------------------------------- MMA issuer (leader CTA)
    if (leader && lane == 0) {
      constexpr uint32_t idesc = make_idesc_pair(kBN);
      int stage = 0;
      uint32_t phase = 0;
      int as = 0;
      uint32_t aphase = 0;
      for (int i = 0; i < n_rb; ++i) {
        for (int t = 0; t < 2 * n_tiles; ++t) {
          mbar_wait_cluster(&bar->tempty[as], aphase ^ 1);
          tc_fence_after();
          const uint32_t d_tmem = tmem_base + (uint32_t)(as * kBN);
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
            if (++stage == kStages) { stage = 0; phase ^= 1; }
          }
          tc_commit_pair(&bar->tfull[as]);
          if (t == n_tiles - 1) tc_commit_pair(&bar->l2_done);   // every layer-2 MMA of this row block has read act1
          if (++as == 2) { as = 0; aphase ^= 1; }
        }
      }
    }
  } else if (warp < 2 + kEpiWarps) {
    // ---------------------------------------------------------------- epilogue warps
    const int quad = warp & 3;
    int as = 0;
    uint32_t aphase = 0;
    uint8_t* stage_buf = store_stage + (warp - 2) * kStoreStage;
    uint32_t chunk = 0;
    const uint32_t tempty_leader0 = mapa_u32(smem_u32(&bar->tempty[0]), 0);
    const uint32_t tempty_leader1 = mapa_u32(smem_u32(&bar->tempty[1]), 0);
    for (int i = 0; i < n_rb; ++i) {
      const int64_t rb = pair + (int64_t)i * n_pairs;
      const int64_t row = rb * kPairBM + (int64_t)rank * BM + quad * 32 + lane;
      float dot = 0.f;
      for (int t = 0; t < 2 * n_tiles; ++t) {
        const int layer = t < n_tiles ? 2 : 3;
        const int nb = t < n_tiles ? t : t - n_tiles;
        mbar_wait(&bar->tfull[as], aphase);
        tc_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(as * kBN);
        const uint32_t rel = as == 0 ? tempty_leader0 : tempty_leader1;
        if (layer == 2) {
          // bias + ReLU -> bf16 -> act2 (this warp's 32 rows x 256 columns, 64 columns per TMA store box)
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
            tmem_ld_wait();
            if (c + 64 >= kBN) {
              tc_fence_before();
              __syncwarp();
              if (lane == 0) mbar_arrive_cluster(rel);
            }
            const float4* b4 = reinterpret_cast<const float4*>(p.b2 + nb * kBN + c);
#pragma unroll
            for (int q = 0; q < 8; ++q) {
              uint32_t w[4];
#pragma unroll
              for (int h = 0; h < 2; ++h) {
                const float4 b = __ldg(b4 + q * 2 + h);
                const uint32_t* r = (q < 4 ? ra : rb2) + (q & 3) * 8 + h * 4;
                w[h * 2 + 0] = pack_relu_bf16x2(__uint_as_float(r[0]) + b.x, __uint_as_float(r[1]) + b.y);
                w[h * 2 + 1] = pack_relu_bf16x2(__uint_as_float(r[2]) + b.z, __uint_as_float(r[3]) + b.w);
              }
              *reinterpret_cast<uint4*>(buf + lane * 128 + ((q ^ (lane & 7)) << 4)) = make_uint4(w[0], w[1], w[2], w[3]);
            }
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) {
              tma_store_2d(&tmS2st, buf, nb * kBN + c, scratch_row0 + quad * 32);
              bulk_commit();
            }
            ++chunk;
          }
          // slab nb of act2 is complete for this warp's rows once its stores have landed
          if (lane == 0) {
            bulk_wait_all();
            mbar_arrive(&bar->act2_ready[nb]);
          }
          __syncwarp();
          chunk = 0;   // nothing of this warp is in flight any more
        } else {
          // ReLU(acc + b3) . w4 over this tile's columns, accumulated over the column tiles in the thread's register
#pragma unroll 1
          for (int c = 0; c < kBN; c += 32) {
            uint32_t r[32];
            tmem_ld32(taddr + c, r);
            tmem_ld_wait();
            if (c + 32 >= kBN) {
              tc_fence_before();
              __syncwarp();
              if (lane == 0) mbar_arrive_cluster(rel);
            }
            const float4* b4 = reinterpret_cast<const float4*>(p.b3 + nb * kBN + c);
            const float4* w4 = reinterpret_cast<const float4*>(p.w4 + nb * kBN + c);
#pragma unroll
            for (int q = 0; q < 8; ++q) {
              const float4 b = __ldg(b4 + q), w = __ldg(w4 + q);
              dot = fmaf(fmaxf(__uint_as_float(r[q * 4 + 0]) + b.x, 0.f), w.x, dot);
              dot = fmaf(fmaxf(__uint_as_float(r[q * 4 + 1]) + b.y, 0.f), w.y, dot);
              dot = fmaf(fmaxf(__uint_as_float(r[q * 4 + 2]) + b.z, 0.f), w.z, dot);
              dot = fmaf(fmaxf(__uint_as_float(r[q * 4 + 3]) + b.w, 0.f), w.w, dot);
            }
          }
          if (nb == n_tiles - 1 && row < M) p.score[rows.m_off + row] = fast_sigmoid(dot + p.b4);
        }
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
  } else {
    // ---------------------------------------------------------------- layer 1 on mma.sync: 32 rows per warp
    const int sw = warp - (2 + kEpiWarps);
    const int g = lane >> 2, t4 = lane & 3;
    const int u = p.u;
    __nv_bfloat16* out0 = p.act1 + (int64_t)(scratch_row0 + sw * 32) * p.W;
    const int n8_tiles = p.W / 8;
    for (int i = 0; i < n_rb; ++i) {
      const int64_t rb = pair + (int64_t)i * n_pairs;
      const int64_t row0 = rb * kPairBM + (int64_t)rank * BM + sw * 32;
      // A fragments: rows {g, g+8} of the two 16-row tiles, K = 32 columns = [u_src ; u_dst ; 0]
      uint32_t a[2][2][4];
#pragma unroll
      for (int mt = 0; mt < 2; ++mt) {
#pragma unroll
        for (int hr = 0; hr < 2; ++hr) {
          const int64_t row = row0 + mt * 16 + hr * 8 + g;
          int64_t si = 0, di = 0;
          const bool ok = row < M;
          if (ok) { si = p.src[rows.m_off + row]; di = p.dst[rows.m_off + row]; }
#pragma unroll
          for (int ks = 0; ks < 2; ++ks) {
#pragma unroll
            for (int hc = 0; hc < 2; ++hc) {
              const int c = ks * 16 + hc * 8 + 2 * t4;      // even column; (c, c+1) never straddles u when u is even
              float v0 = 0.f, v1 = 0.f;
              if (ok) {
                if (c < u) v0 = __ldg(p.feat + si * u + c); else if (c < 2 * u) v0 = __ldg(p.feat + di * u + (c - u));
                if (c + 1 < u) v1 = __ldg(p.feat + si * u + c + 1); else if (c + 1 < 2 * u) v1 = __ldg(p.feat + di * u + (c + 1 - u));
              }
              a[mt][ks][hc * 2 + hr] = pack_bf16(v0, v1);
            }
          }
        }
      }
      // act1 of the previous row block must have been read by all of its layer-2 MMAs
      if (i > 0) mbar_wait(&bar->l2_done, (uint32_t)((i - 1) & 1));
#pragma unroll 2
      for (int nt = 0; nt < n8_tiles; ++nt) {
        const uint4 b = __ldg(p.w1_frag + (int64_t)nt * 32 + lane);
        const float2 bias = __ldg(reinterpret_cast<const float2*>(p.b1 + nt * 8 + 2 * t4));
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
          float c[4] = {bias.x, bias.y, bias.x, bias.y};
          mma_bf16_16816(c, a[mt][0], b.x, b.y);
          mma_bf16_16816(c, a[mt][1], b.z, b.w);
          __nv_bfloat16* o = out0 + (int64_t)(mt * 16 + g) * p.W + nt * 8 + 2 * t4;
          *reinterpret_cast<uint32_t*>(o) = pack_relu_bf16x2(c[0], c[1]);
          *reinterpret_cast<uint32_t*>(o + (int64_t)8 * p.W) = pack_relu_bf16x2(c[2], c[3]);
        }
      }
      __threadfence();
      fence_proxy_async_global();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bar->act1_ready);
    }
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

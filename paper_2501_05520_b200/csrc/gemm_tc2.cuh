// CTA-pair variant of gemm_tc.cuh:   acc[m][n] = sum_k A[m][k] * W[n][k]   with tcgen05.mma.cta_group::2.
//
// Two CTAs of a 2-CTA cluster (the two SMs of one TPC) compute one 256 x BN output tile: CTA rank r
// holds rows [128 r, 128 r + 128) of A and rows [BN/2 r, BN/2 (r+1)) of W in its shared memory; the
// leader (rank 0) issues one MMA per K step for both SMs, each SM accumulates its own 128 rows x BN
// columns in its own TMEM.  Per SM and K block this moves 16 KB of A + (BN/2 x 128 B) of W instead of
// 16 KB + (BN x 128 B): with BN = 256 the shared-memory fill per flop drops by a third and six ring
// stages fit where the single-CTA kernel has four.
//
// Pipelines (all mbarriers exist in both CTAs at the same offsets):
//   full[s]    leader's copy only: both CTAs' TMA loads complete_tx on it, the leader expects 2 x STAGE bytes
//   empty[s]   each CTA's own copy, arrived by the leader's tcgen05.commit multicast to both CTAs
//   tfull[a]   each CTA's own copy, same multicast commit after the last K block of a tile
//   tempty[a]  leader's copy only: the epilogue warps of both CTAs arrive on it (2 x kEpiWarps)
#pragma once

#include "gemm_tc.cuh"

namespace trk {
namespace tc {

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of the same shared-memory offset in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa_u32(uint32_t local_addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// TMA load whose completion mbarrier may live in the peer CTA of the pair (cluster address).
__device__ __forceinline__ void tma_load_2d_pair(void* smem_dst, const CUtensorMap* tmap, uint32_t bar_cluster_addr, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
          smem_u32(smem_dst)),
      "l"(reinterpret_cast<uint64_t>(tmap)), "r"(bar_cluster_addr), "r"(c0), "r"(c1)
      : "memory");
}
template <int NCOLS>
__device__ __forceinline__ void tmem_alloc_pair(uint32_t* smem_slot) {
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_slot)), "n"(NCOLS) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
template <int NCOLS>
__device__ __forceinline__ void tmem_dealloc_pair(uint32_t taddr) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "n"(NCOLS) : "memory");
}
// arrives on the mbarrier at this shared-memory offset in both CTAs of the pair once all prior MMAs are done
__device__ __forceinline__ void tc_commit_pair(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(smem_u32(bar)),
               "h"((uint16_t)3)
               : "memory");
}
__device__ __forceinline__ void tc_mma_bf16_pair(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// Instruction descriptor of the pair MMA: M = 256 (128 rows per CTA), N = BN.
__host__ __device__ constexpr uint32_t make_idesc_pair(int bn) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(bn >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
}

constexpr int kPairBM = 256;
constexpr int stage_bytes_pair(int bn) { return (BM + bn / 2) * BK * 2; }   // per CTA
constexpr int num_stages_pair(int bn) { return (192 * 1024) / stage_bytes_pair(bn) > 8 ? 8 : (192 * 1024) / stage_bytes_pair(bn); }
constexpr int smem_bytes_pair(int bn, bool tma_store = false) {
  return num_stages_pair(bn) * stage_bytes_pair(bn) + (tma_store ? kEpiWarps * kStoreStage : 0) + 1024 + 256;
}

template <int BN, class Epi>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
gemm_tc2_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const __grid_constant__ CUtensorMap tmC,
                Rows rows, int n_tiles, int k_blocks, typename Epi::Params ep, int row_major_min) {
  TRK_GRID_DEP_WAIT();
  constexpr int STAGES = num_stages_pair(BN);
  constexpr int A_BYTES = BM * BK * 2;
  constexpr int STAGE = stage_bytes_pair(BN);
  constexpr int TMEM_COLS = tmem_cols_for(BN);
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint8_t* store_stage = smem + STAGES * STAGE;
  uint64_t* full_bar = reinterpret_cast<uint64_t*>(store_stage + (Epi::kTmaStore ? kEpiWarps * kStoreStage : 0));
  uint64_t* empty_bar = full_bar + STAGES;
  uint64_t* tfull_bar = empty_bar + STAGES;
  uint64_t* tempty_bar = tfull_bar + 2;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty_bar + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const bool leader = rank == 0;
  const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
  const int64_t M = resolve_rows(rows);
  const int64_t m_tiles = (M + kPairBM - 1) / kPairBM;
  const int64_t total = m_tiles * n_tiles;
  // This pair's j-th tile.  With many row blocks a pair walks all column tiles of one row block before it takes the next
  // (its A rows are re-read from L2 a few microseconds apart: ncu showed 1.37x the algorithmic DRAM reads when the column
  // tiles of a row block were spread over four pairs that drift apart during a 1.7 ms launch); with few row blocks the
  // tiles are dealt out in pair strides so that every pair has work.
  const bool row_major = row_major_min > 0 && m_tiles >= (int64_t)row_major_min * n_pairs;   // imbalance <= 1 / row_major_min
  const int64_t n_iter = row_major ? (pair < m_tiles ? (m_tiles - pair + n_pairs - 1) / n_pairs * n_tiles : 0)
                                   : (pair < total ? (total - pair + n_pairs - 1) / n_pairs : 0);
  auto tile_of = [&](int64_t j, int& m_blk, int& n_blk) {
    if (row_major) {
      m_blk = (int)(pair + (j / n_tiles) * n_pairs);
      n_blk = (int)(j % n_tiles);
    } else {
      const int64_t tile = pair + j * n_pairs;
      m_blk = (int)(tile / n_tiles);
      n_blk = (int)(tile % n_tiles);
    }
  };

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmA);
    prefetch_tmap(&tmB);
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], 1);
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(&tfull_bar[s], 1);
      mbar_init(&tempty_bar[s], 2 * kEpiWarps);
    }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc_pair<TMEM_COLS>(tmem_slot);
  tc_fence_before();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int64_t j = 0; j < n_iter; ++j) {
        int m_blk, n_blk;
        tile_of(j, m_blk, n_blk);
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(&empty_bar[stage], phase ^ 1);
          if (leader) mbar_arrive_expect_tx(&full_bar[stage], 2 * STAGE);
          const uint32_t full_leader = mapa_u32(smem_u32(&full_bar[stage]), 0);
          uint8_t* sa = smem + stage * STAGE;
          tma_load_2d_pair(sa, &tmA, full_leader, kb * BK, m_blk * kPairBM + (int)rank * BM);
          tma_load_2d_pair(sa + A_BYTES, &tmB, full_leader, kb * BK, n_blk * BN + (int)rank * (BN / 2));
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    if (leader && lane == 0) {
      constexpr uint32_t idesc = make_idesc_pair(BN);
      int stage = 0;
      uint32_t phase = 0;
      int as = 0;
      uint32_t aphase = 0;
      for (int64_t j = 0; j < n_iter; ++j) {
        mbar_wait_cluster(&tempty_bar[as], aphase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(as * BN);
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(smem + stage * STAGE);
          const uint64_t adesc = make_smem_desc(sa);
          const uint64_t bdesc = make_smem_desc(sa + A_BYTES);
#pragma unroll
          for (int k = 0; k < BK / UMMA_K; ++k)
            tc_mma_bf16_pair(d_tmem, adesc + (uint64_t)(k * 2), bdesc + (uint64_t)(k * 2), idesc, (kb | k) != 0 ? 1u : 0u);
          tc_commit_pair(&empty_bar[stage]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        tc_commit_pair(&tfull_bar[as]);
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
  } else {
    const int quad = warp & 3;
    int as = 0;
    uint32_t aphase = 0;
    EpiShared es{store_stage + (warp - 2) * kStoreStage, &tmC, 0u};
    const uint32_t tempty_leader0 = mapa_u32(smem_u32(&tempty_bar[0]), 0);
    const uint32_t tempty_leader1 = mapa_u32(smem_u32(&tempty_bar[1]), 0);
    for (int64_t j = 0; j < n_iter; ++j) {
      int m_blk, n_blk;
      tile_of(j, m_blk, n_blk);
      mbar_wait(&tfull_bar[as], aphase);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(as * BN);
      const uint32_t rel = as == 0 ? tempty_leader0 : tempty_leader1;
      auto release = [&]() {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(rel);
      };
      Epi::template run<BN>(ep, taddr, (int64_t)m_blk * kPairBM + (int64_t)rank * BM + quad * 32 + lane, n_blk * BN, n_blk, M, release, es);
      if (++as == 2) { as = 0; aphase ^= 1; }
    }
    if (Epi::kTmaStore && lane == 0) bulk_wait_all();
  }
  tc_fence_before();
  cluster_sync_all();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_pair<TMEM_COLS>(tmem_base);
  }
}

}  // namespace tc
}  // namespace trk

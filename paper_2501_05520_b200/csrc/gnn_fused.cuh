// Fused interaction-network edge update of S4 for H = 128 on CTA pairs (reading C-12):
//
//   e_k <- e_k + LNR(W2 LNR(W1 [h_src(k) ; h_dst(k) ; e_k] + b1) + b2)           (kUpdate)
//   score_k = sigmoid(w_out . LNR(W1 [h_src ; h_dst ; e_k] + b1) + b_out)        (kDecode)
//
// One 2-CTA cluster handles 256 edges per tile (128 per CTA) and never writes an intermediate to HBM:
//   * both weight matrices stay in shared memory for the whole kernel, split by output row between the
//     two CTAs (tcgen05.mma.cta_group::2 reads the N halves from both SMs): 64 KB per CTA;
//   * the 3H-wide first-layer input is assembled in shared memory as six K blocks: the e rows by TMA,
//     the h rows of the edge's endpoints by cp.async gathers (coalesced 256-byte rows) straight into
//     the 128-byte-swizzled UMMA layout;
//   * layer-1 accumulator (TMEM) -> LayerNorm + ReLU in registers -> bf16 tile T in shared memory ->
//     layer-2 MMA -> LayerNorm + ReLU + residual (read from the e tile still in shared memory) ->
//     the e tile is overwritten in place and leaves by TMA store.
// HBM traffic per edge and iteration: 256 B of e in, 256 B out, 8 B of indices; the h rows (20 MB table)
// come from L2.
//
// Warps: 0 TMA producer, 1 MMA issuer (leader CTA) + TMEM owner, 2-5 epilogue 1, 6-9 epilogue 2,
// 10-13 gather.  TMEM: acc1[2] (columns 0,128) and acc2[2] (256,384), so two tiles are in flight.
// mbarriers marked L are used in the leader CTA's copy only (both CTAs arrive on it).
#pragma once

#include "gemm_tc2.cuh"

namespace trk {
namespace gf {

using namespace tc;

constexpr int kH = 128;
constexpr int kThreadsFused = 14 * 32;
constexpr int kTileRows = 128;            // per CTA
constexpr int kKB = 16384;                // one 128-row x 64-column bf16 K block
constexpr int kWKB = 8192;                // one 64-row x 64-column K block of a weight half
// shared memory carve-up (bytes, per CTA)
constexpr int kOffW1 = 0;                 // 6 K blocks of this CTA's 64 output rows of W1
constexpr int kOffW2 = kOffW1 + 6 * kWKB; // 2 K blocks of W2
constexpr int kOffRing = kOffW2 + 2 * kWKB;   // 4 K blocks: h_src (2), h_dst (2)
constexpr int kOffEHold = kOffRing + 4 * kKB; // 2 x (2 K blocks): the e tile of the two tiles in flight
constexpr int kOffT = kOffEHold + 4 * kKB;    // 2 K blocks: layer-1 output
constexpr int kOffBar = kOffT + 2 * kKB;
constexpr int kSmemFused = kOffBar + 256 + 1024;

enum Mode { kUpdate = 0, kDecode = 1 };

struct FusedParams {
  const __nv_bfloat16* X;     // [n_nodes][ldx] bf16, h = columns [0, 128)
  int64_t ldx;
  const int32_t* src;
  const int32_t* dst;
  const float* b1;
  const float* b2;
  int use_ln;
  const float* w_out;         // kDecode
  float b_out;
  float* score;
};

struct Bars {
  uint64_t w_full;
  uint64_t efull[2];      // L  tx: both CTAs' e tiles
  uint64_t eempty[2];     //    own, 4 arrivals (the warps that last touch the e tile)
  uint64_t gfull[2];      // L  8 arrivals (4 gather warps x 2 CTAs), halves: h_src, h_dst
  uint64_t gempty[2];     //    own, multicast commit
  uint64_t a1full[2];     //    own, multicast commit
  uint64_t a1empty[2];    // L  8 arrivals
  uint64_t tfull;         // L  8 arrivals
  uint64_t tempty;        //    own, multicast commit
  uint64_t a2full[2];     //    own, multicast commit
  uint64_t a2empty[2];    // L  8 arrivals
  uint32_t tmem_slot;
};

__device__ __forceinline__ void cp_async_16(uint32_t smem_dst, const void* gsrc, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_dst), "l"(gsrc), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// LayerNorm statistics of one accumulator row (this thread's TMEM lane), columns [0,128) of `taddr`, after adding bias.
__device__ __forceinline__ void row_stats(uint32_t taddr, const float* __restrict__ bias, int use_ln, float& mean, float& rstd) {
  float s = 0.f, q = 0.f;
#pragma unroll 1
  for (int c = 0; c < kH; c += 32) {
    uint32_t r[32];
    tmem_ld32(taddr + c, r);
    tmem_ld_wait();
#pragma unroll
    for (int i = 0; i < 32; i += 4) {
      const float4 b = __ldg(reinterpret_cast<const float4*>(bias + c + i));
      const float v0 = __uint_as_float(r[i]) + b.x, v1 = __uint_as_float(r[i + 1]) + b.y, v2 = __uint_as_float(r[i + 2]) + b.z,
                  v3 = __uint_as_float(r[i + 3]) + b.w;
      s += (v0 + v1) + (v2 + v3);
      q = fmaf(v0, v0, q); q = fmaf(v1, v1, q); q = fmaf(v2, v2, q); q = fmaf(v3, v3, q);
    }
  }
  if (use_ln) {
    mean = s * (1.f / kH);
    const float var = fmaxf(q * (1.f / kH) - mean * mean, 0.f);
    rstd = rsqrtf(var + 1e-5f);
  } else {
    mean = 0.f;
    rstd = 1.f;
  }
}

template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreadsFused, 1)
gnn_edge_fused_kernel(const __grid_constant__ CUtensorMap tmW1, const __grid_constant__ CUtensorMap tmW2,
                      const __grid_constant__ CUtensorMap tmE, const __grid_constant__ CUtensorMap tmEst, Rows rows, FusedParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  Bars* bar = reinterpret_cast<Bars*>(smem + kOffBar);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const bool leader = rank == 0;
  const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
  const int64_t M = resolve_rows(rows);
  const int64_t total = (M + 2 * kTileRows - 1) / (2 * kTileRows);
  const int n_my = total > pair ? (int)((total - pair + n_pairs - 1) / n_pairs) : 0;

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmW1); prefetch_tmap(&tmW2); prefetch_tmap(&tmE); prefetch_tmap(&tmEst);
    mbar_init(&bar->w_full, 1);
    for (int i = 0; i < 2; ++i) {
      mbar_init(&bar->efull[i], 1);
      mbar_init(&bar->eempty[i], 4);
      mbar_init(&bar->gfull[i], 8);
      mbar_init(&bar->gempty[i], 1);
      mbar_init(&bar->a1full[i], 1);
      mbar_init(&bar->a1empty[i], 8);
      mbar_init(&bar->a2full[i], 1);
      mbar_init(&bar->a2empty[i], 8);
    }
    mbar_init(&bar->tfull, 8);
    mbar_init(&bar->tempty, 1);
    fence_barrier_init();
    // this CTA's halves of the weights: output rows [64 rank, 64 rank + 64)
    mbar_arrive_expect_tx(&bar->w_full, 8 * kWKB);
    for (int kb = 0; kb < 6; ++kb) tma_load_2d(smem + kOffW1 + kb * kWKB, &tmW1, &bar->w_full, kb * 64, (int)rank * 64);
    for (int kb = 0; kb < 2; ++kb) tma_load_2d(smem + kOffW2 + kb * kWKB, &tmW2, &bar->w_full, kb * 64, (int)rank * 64);
  }
  if (warp == 1) tmem_alloc_pair<512>(&bar->tmem_slot);
  __syncthreads();
  mbar_wait(&bar->w_full, 0);
  tc_fence_before();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = bar->tmem_slot;
  const uint32_t sbase = smem_u32(smem);

  if (warp == 0) {
    // ---------------------------------------------------------------- TMA producer: e tiles
    if (lane == 0) {
      for (int tl = 0; tl < n_my; ++tl) {
        const int64_t tile = pair + (int64_t)tl * n_pairs;
        const int b = tl & 1;
        const uint32_t ph = (tl >> 1) & 1;
        mbar_wait(&bar->eempty[b], ph ^ 1);
        if (leader) mbar_arrive_expect_tx(&bar->efull[b], 2 * 2 * kKB);
        const uint32_t full_leader = mapa_u32(smem_u32(&bar->efull[b]), 0);
        const int row0 = (int)(tile * 2 * kTileRows + rank * kTileRows);
        for (int kb = 0; kb < 2; ++kb) tma_load_2d_pair(smem + kOffEHold + (b * 2 + kb) * kKB, &tmE, full_leader, kb * 64, row0);
      }
    }
  } else if (warp == 1) {
    // ---------------------------------------------------------------- MMA issuer (leader CTA)
    if (leader && lane == 0) {
      constexpr uint32_t idesc = make_idesc_pair(kH);
      auto kblock = [&](uint32_t d_tmem, uint32_t a_addr, uint32_t b_addr, bool first) {
        const uint64_t adesc = make_smem_desc(a_addr), bdesc = make_smem_desc(b_addr);
#pragma unroll
        for (int k = 0; k < BK / UMMA_K; ++k)
          tc_mma_bf16_pair(d_tmem, adesc + (uint64_t)(k * 2), bdesc + (uint64_t)(k * 2), idesc, (!first || k != 0) ? 1u : 0u);
      };
      auto mma1 = [&](int tl) {
        const int b = tl & 1;
        const uint32_t ph = (tl >> 1) & 1;
        const uint32_t d = tmem_base + (uint32_t)(b * kH);
        mbar_wait_cluster(&bar->a1empty[b], ph ^ 1);
        mbar_wait(&bar->efull[b], ph);
        tc_fence_after();
        for (int kb = 0; kb < 2; ++kb) kblock(d, sbase + kOffEHold + (b * 2 + kb) * kKB, sbase + kOffW1 + (4 + kb) * kWKB, kb == 0);
        for (int h = 0; h < 2; ++h) {
          mbar_wait_cluster(&bar->gfull[h], (uint32_t)(tl & 1));
          tc_fence_after();
          for (int kb = 0; kb < 2; ++kb) kblock(d, sbase + kOffRing + (h * 2 + kb) * kKB, sbase + kOffW1 + (h * 2 + kb) * kWKB, false);
          tc_commit_pair(&bar->gempty[h]);
        }
        tc_commit_pair(&bar->a1full[b]);
      };
      auto mma2 = [&](int tl) {
        const int b = tl & 1;
        const uint32_t ph = (tl >> 1) & 1;
        const uint32_t d = tmem_base + (uint32_t)(2 * kH + b * kH);
        mbar_wait_cluster(&bar->tfull, (uint32_t)(tl & 1));
        mbar_wait_cluster(&bar->a2empty[b], ph ^ 1);
        tc_fence_after();
        for (int kb = 0; kb < 2; ++kb) kblock(d, sbase + kOffT + kb * kKB, sbase + kOffW2 + kb * kWKB, kb == 0);
        tc_commit_pair(&bar->tempty);
        tc_commit_pair(&bar->a2full[b]);
      };
      if (n_my > 0) mma1(0);
      for (int tl = 0; tl < n_my; ++tl) {
        if (tl + 1 < n_my) mma1(tl + 1);
        if (MODE == kUpdate) mma2(tl);
      }
    }
  } else if (warp < 6) {
    // ---------------------------------------------------------------- epilogue 1: acc1 -> LNR -> T (or score)
    const int quad = warp & 3;
    const int r = quad * 32 + lane;   // row of this thread inside the CTA's 128-row tile == TMEM lane
    const uint32_t a1empty0 = mapa_u32(smem_u32(&bar->a1empty[0]), 0), a1empty1 = mapa_u32(smem_u32(&bar->a1empty[1]), 0);
    const uint32_t tfull_l = mapa_u32(smem_u32(&bar->tfull), 0);
    for (int tl = 0; tl < n_my; ++tl) {
      const int64_t tile = pair + (int64_t)tl * n_pairs;
      const int b = tl & 1;
      const uint32_t ph = (tl >> 1) & 1;
      mbar_wait(&bar->a1full[b], ph);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(b * kH);
      float mean, rstd;
      row_stats(taddr, p.b1, p.use_ln, mean, rstd);
      if (MODE == kUpdate) mbar_wait(&bar->tempty, (uint32_t)(tl & 1) ^ 1);   // layer-2 MMA of the previous tile has read T
      float dot = p.b_out;
#pragma unroll 1
      for (int c = 0; c < kH; c += 32) {
        uint32_t v[32];
        tmem_ld32(taddr + c, v);
        tmem_ld_wait();
        if (c + 32 >= kH) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(b == 0 ? a1empty0 : a1empty1);
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          float f[8];
#pragma unroll
          for (int hh = 0; hh < 2; ++hh) {
            const float4 bb = __ldg(reinterpret_cast<const float4*>(p.b1 + c + q * 8 + hh * 4));
            f[hh * 4 + 0] = fmaxf((__uint_as_float(v[q * 8 + hh * 4 + 0]) + bb.x - mean) * rstd, 0.f);
            f[hh * 4 + 1] = fmaxf((__uint_as_float(v[q * 8 + hh * 4 + 1]) + bb.y - mean) * rstd, 0.f);
            f[hh * 4 + 2] = fmaxf((__uint_as_float(v[q * 8 + hh * 4 + 2]) + bb.z - mean) * rstd, 0.f);
            f[hh * 4 + 3] = fmaxf((__uint_as_float(v[q * 8 + hh * 4 + 3]) + bb.w - mean) * rstd, 0.f);
          }
          if (MODE == kDecode) {
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
              const float4 w = __ldg(reinterpret_cast<const float4*>(p.w_out + c + q * 8 + hh * 4));
              dot = fmaf(f[hh * 4 + 0], w.x, dot); dot = fmaf(f[hh * 4 + 1], w.y, dot);
              dot = fmaf(f[hh * 4 + 2], w.z, dot); dot = fmaf(f[hh * 4 + 3], w.w, dot);
            }
          } else {
            const int col = c + q * 8;                 // 8 columns = one 16-byte chunk
            const int kb = col >> 6, ch = (col & 63) >> 3;
            *reinterpret_cast<uint4*>(smem + kOffT + kb * kKB + r * 128 + ((ch ^ (r & 7)) << 4)) =
                make_uint4(pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
          }
        }
      }
      if (MODE == kDecode) {
        const int64_t row = tile * 2 * kTileRows + rank * kTileRows + r;
        if (row < M) p.score[row] = fast_sigmoid(dot);
        __syncwarp();
        if (lane == 0) mbar_arrive(&bar->eempty[b]);   // the layer-1 MMAs that read the e tile are complete
      } else {
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(tfull_l);
      }
    }
  } else if (warp < 10) {
    // ---------------------------------------------------------------- epilogue 2: acc2 -> LNR -> + e -> store
    if (MODE == kUpdate) {
      const int quad = warp & 3;
      const int r = quad * 32 + lane;
      const uint32_t a2empty0 = mapa_u32(smem_u32(&bar->a2empty[0]), 0), a2empty1 = mapa_u32(smem_u32(&bar->a2empty[1]), 0);
      for (int tl = 0; tl < n_my; ++tl) {
        const int64_t tile = pair + (int64_t)tl * n_pairs;
        const int b = tl & 1;
        const uint32_t ph = (tl >> 1) & 1;
        mbar_wait(&bar->a2full[b], ph);
        tc_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(2 * kH + b * kH);
        float mean, rstd;
        row_stats(taddr, p.b2, p.use_ln, mean, rstd);
        uint8_t* eh = smem + kOffEHold + b * 2 * kKB;
#pragma unroll 1
        for (int c = 0; c < kH; c += 32) {
          uint32_t v[32];
          tmem_ld32(taddr + c, v);
          tmem_ld_wait();
          if (c + 32 >= kH) {
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(b == 0 ? a2empty0 : a2empty1);
          }
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const int col = c + q * 8;
            const int kb = col >> 6, ch = (col & 63) >> 3;
            uint4* cell = reinterpret_cast<uint4*>(eh + kb * kKB + r * 128 + ((ch ^ (r & 7)) << 4));
            const uint4 e = *cell;
            const __nv_bfloat162* e2 = reinterpret_cast<const __nv_bfloat162*>(&e);
            float f[8];
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
              const float4 bb = __ldg(reinterpret_cast<const float4*>(p.b2 + col + hh * 4));
              f[hh * 4 + 0] = fmaxf((__uint_as_float(v[q * 8 + hh * 4 + 0]) + bb.x - mean) * rstd, 0.f) + __low2float(e2[hh * 2]);
              f[hh * 4 + 1] = fmaxf((__uint_as_float(v[q * 8 + hh * 4 + 1]) + bb.y - mean) * rstd, 0.f) + __high2float(e2[hh * 2]);
              f[hh * 4 + 2] = fmaxf((__uint_as_float(v[q * 8 + hh * 4 + 2]) + bb.z - mean) * rstd, 0.f) + __low2float(e2[hh * 2 + 1]);
              f[hh * 4 + 3] = fmaxf((__uint_as_float(v[q * 8 + hh * 4 + 3]) + bb.w - mean) * rstd, 0.f) + __high2float(e2[hh * 2 + 1]);
            }
            *cell = make_uint4(pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
          }
        }
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) {
          const int row0 = (int)(tile * 2 * kTileRows + rank * kTileRows + quad * 32);
          for (int kb = 0; kb < 2; ++kb) tma_store_2d(&tmEst, eh + kb * kKB + quad * 32 * 128, kb * 64, row0);
          bulk_commit();
          bulk_wait_read<0>();          // the tile's rows have left shared memory: the buffer may be refilled
          mbar_arrive(&bar->eempty[b]);
        }
      }
      if (lane == 0) bulk_wait_all();
    }
  } else {
    // ---------------------------------------------------------------- gather: h[src], h[dst] rows -> ring
    const int gw = warp - 10;
    const uint32_t gfull0 = mapa_u32(smem_u32(&bar->gfull[0]), 0), gfull1 = mapa_u32(smem_u32(&bar->gfull[1]), 0);
    const int half = lane >> 4, chunk = lane & 15;
    const int kb = chunk >> 3, ch = chunk & 7;
    for (int tl = 0; tl < n_my; ++tl) {
      const int64_t tile = pair + (int64_t)tl * n_pairs;
      const int64_t row = tile * 2 * kTileRows + rank * kTileRows + gw * 32 + lane;
      const int my_s = row < M ? p.src[row] : -1, my_d = row < M ? p.dst[row] : -1;
#pragma unroll 1
      for (int h = 0; h < 2; ++h) {
        mbar_wait(&bar->gempty[h], (uint32_t)(tl & 1) ^ 1);
        const int mine = h == 0 ? my_s : my_d;
#pragma unroll 4
        for (int i = 0; i < 16; ++i) {
          const int rr = i * 2 + half;                       // row inside this warp's 32 rows
          const int idx = __shfl_sync(0xffffffffu, mine, rr);
          const int rt = gw * 32 + rr;                       // row inside the CTA's tile
          const uint32_t dst = sbase + kOffRing + (h * 2 + kb) * kKB + rt * 128 + ((ch ^ (rt & 7)) << 4);
          const __nv_bfloat16* g = p.X + (int64_t)(idx < 0 ? 0 : idx) * p.ldx + chunk * 8;
          cp_async_16(dst, g, idx < 0 ? 0 : 16);             // rows beyond M are zero filled
        }
        cp_async_commit();
      }
      cp_async_wait<1>();
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(gfull0);
      cp_async_wait<0>();
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(gfull1);
    }
  }
  tc_fence_before();
  cluster_sync_all();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_pair<512>(tmem_base);
  }
}

}  // namespace gf
}  // namespace trk

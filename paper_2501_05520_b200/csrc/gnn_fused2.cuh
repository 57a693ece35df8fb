// Fused interaction-network edge update of S4 for H = 128 on CTA pairs, second version (reading C-12):
//
//   e_k <- e_k + LNR(W2 LNR(W1 [h_src(k) ; h_dst(k) ; e_k] + b1) + b2)           (kUpdate)
//   score_k = sigmoid(w_out . LNR(W1 [h_src ; h_dst ; e_k] + b1) + b_out)        (kDecode)
//
// Same data flow as gnn_fused.cuh (weights resident in shared memory and split by output row between the two CTAs of a
// pair, e tile by TMA, endpoint h rows gathered by cp.async into the swizzled UMMA layout, layer-1 accumulator -> LayerNorm
// -> bf16 tile T in shared memory -> layer-2 MMA -> LayerNorm + residual in place -> TMA store; nothing intermediate
// touches HBM).  What changed, from the per-role wait profile of version 1 (same method as profiles/r1_fused_roles_v3.md): the two
// LayerNorm epilogues were latency-bound single warps (two TMEM passes, 128-long dependent FMA chains, ~7 k cycles per tile
// each) and the e-tile loads came cold from HBM behind them.  Here
//   * an epilogue thread reads its whole 128-column accumulator row from TMEM in one go (4 loads, one wait), releases the
//     accumulator at once, and computes mean / variance / normalise on registers with four independent chains;
//   * biases and the decoder weights are read from shared memory (broadcast LDS.128) instead of the global path;
//   * the TMA warp prefetches the e tiles two tiles ahead into L2 (cp.async.bulk.prefetch.tensor);
//   * the MMA warp polls (mbarrier.test_wait) and issues whichever of layer 1 (next tile) and layer 2 (this tile) has its
//     operands ready, instead of blocking on one in program order;
//   * 12 warps (384 threads, up to 168 registers each): 0 TMA, 1 MMA issuer (leader CTA) + TMEM owner, 2-3 gather,
//     4-7 epilogue 1, 8-11 epilogue 2.
// TMEM: acc1[2] (columns 0,128) and acc2[2] (256,384).  mbarriers marked L live in the leader CTA's copy (both CTAs arrive).
#pragma once

#include "gnn_fused.cuh"

namespace trk {
namespace gf2 {

using namespace tc;
using gf::cp_async_16;
using gf::cp_async_commit;
using gf::cp_async_wait;
using gf::FusedParams;
using gf::kH;
using gf::kKB;
using gf::kTileRows;
using gf::kWKB;
using gf::Mode;

constexpr int kThreads2 = 12 * 32;
constexpr int kOffW1 = 0;                       // 6 K blocks of this CTA's 64 output rows of W1
constexpr int kOffW2 = kOffW1 + 6 * kWKB;       // 2 K blocks of W2
constexpr int kOffRing = kOffW2 + 2 * kWKB;     // 4 K blocks: h_src (2), h_dst (2)
constexpr int kOffEHold = kOffRing + 4 * kKB;   // 2 x (2 K blocks): the e tile of the two tiles in flight
constexpr int kOffT = kOffEHold + 4 * kKB;      // 2 K blocks: layer-1 output
constexpr int kOffVec = kOffT + 2 * kKB;        // b1, b2, w_out: 3 x 128 fp32
constexpr int kOffBar = kOffVec + 3 * kH * 4;
constexpr int kSmemFused2 = kOffBar + 256 + 1024;
static_assert(kSmemFused2 <= 232448, "shared memory budget of one CTA");

struct Bars {
  uint64_t w_full;
  uint64_t efull[2];      // L  tx: both CTAs' e tiles
  uint64_t eempty[2];     //    own, 4 arrivals (the warps that last touch the e tile)
  uint64_t gfull[2];      // L  4 arrivals (2 gather warps x 2 CTAs), halves: h_src, h_dst
  uint64_t gempty[2];     //    own, multicast commit
  uint64_t a1full[2];     //    own, multicast commit
  uint64_t a1empty[2];    // L  8 arrivals
  uint64_t tfull;         // L  8 arrivals
  uint64_t tempty;        //    own, multicast commit
  uint64_t a2full[2];     //    own, multicast commit
  uint64_t a2empty[2];    // L  8 arrivals
  uint32_t tmem_slot;
};

// non-blocking probe of an mbarrier phase (cluster-scope acquire: remote CTAs arrive on some of them)
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "mbarrier.test_wait.parity.acquire.cluster.shared::cta.b64 P1, [%1], %2;\n"
      "selp.u32 %0, 1, 0, P1;\n"
      "}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}

// Arrive on an mbarrier of the pair's leader CTA with CTA-scope release (the form CUTLASS uses for its 2-SM pipelines).
// What the leader's MMA issuer must see before it continues is either a finished TMEM read (ordered by
// tcgen05.fence::before_thread_sync) or shared memory of the ARRIVING CTA that its own tensor core / TMA will read
// (ordered by fence.proxy.async); neither needs the cluster-wide memory barrier of .release.cluster, which cost the
// epilogue warps of version 1 several hundred cycles per arrive (stall_membar in profiles/r1_full_v2.md).
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}

__device__ __forceinline__ void tma_prefetch_l2_2d(const CUtensorMap* tmap, int c0, int c1) {
  asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global.tile [%0, {%1, %2}];" ::"l"(reinterpret_cast<uint64_t>(tmap)), "r"(c0), "r"(c1)
               : "memory");
}

// One accumulator row (this thread's TMEM lane, 128 fp32 columns) -> registers, plus bias; returns after the data has landed.
__device__ __forceinline__ void load_row(uint32_t taddr, const float* __restrict__ sbias, float (&x)[kH]) {
  uint32_t u0[32], u1[32], u2[32], u3[32];
  tmem_ld32(taddr, u0);
  tmem_ld32(taddr + 32, u1);
  tmem_ld32(taddr + 64, u2);
  tmem_ld32(taddr + 96, u3);
  tmem_ld_wait();
#pragma unroll
  for (int i = 0; i < 32; i += 4) {
    const float4 b0 = *reinterpret_cast<const float4*>(sbias + i), b1 = *reinterpret_cast<const float4*>(sbias + 32 + i);
    const float4 b2 = *reinterpret_cast<const float4*>(sbias + 64 + i), b3 = *reinterpret_cast<const float4*>(sbias + 96 + i);
    x[i] = __uint_as_float(u0[i]) + b0.x; x[i + 1] = __uint_as_float(u0[i + 1]) + b0.y;
    x[i + 2] = __uint_as_float(u0[i + 2]) + b0.z; x[i + 3] = __uint_as_float(u0[i + 3]) + b0.w;
    x[32 + i] = __uint_as_float(u1[i]) + b1.x; x[32 + i + 1] = __uint_as_float(u1[i + 1]) + b1.y;
    x[32 + i + 2] = __uint_as_float(u1[i + 2]) + b1.z; x[32 + i + 3] = __uint_as_float(u1[i + 3]) + b1.w;
    x[64 + i] = __uint_as_float(u2[i]) + b2.x; x[64 + i + 1] = __uint_as_float(u2[i + 1]) + b2.y;
    x[64 + i + 2] = __uint_as_float(u2[i + 2]) + b2.z; x[64 + i + 3] = __uint_as_float(u2[i + 3]) + b2.w;
    x[96 + i] = __uint_as_float(u3[i]) + b3.x; x[96 + i + 1] = __uint_as_float(u3[i + 1]) + b3.y;
    x[96 + i + 2] = __uint_as_float(u3[i + 2]) + b3.z; x[96 + i + 3] = __uint_as_float(u3[i + 3]) + b3.w;
  }
}

// LayerNorm statistics of a register row (biased variance, eps 1e-5; two passes, four independent chains each).
__device__ __forceinline__ void row_stats(const float (&x)[kH], int use_ln, float& mean, float& rstd) {
  if (!use_ln) {
    mean = 0.f;
    rstd = 1.f;
    return;
  }
  float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
#pragma unroll
  for (int i = 0; i < kH; i += 4) { s0 += x[i]; s1 += x[i + 1]; s2 += x[i + 2]; s3 += x[i + 3]; }
  mean = ((s0 + s1) + (s2 + s3)) * (1.f / kH);
  float q0 = 0.f, q1 = 0.f, q2 = 0.f, q3 = 0.f;
#pragma unroll
  for (int i = 0; i < kH; i += 4) {
    const float d0 = x[i] - mean, d1 = x[i + 1] - mean, d2 = x[i + 2] - mean, d3 = x[i + 3] - mean;
    q0 = fmaf(d0, d0, q0); q1 = fmaf(d1, d1, q1); q2 = fmaf(d2, d2, q2); q3 = fmaf(d3, d3, q3);
  }
  rstd = rsqrtf(((q0 + q1) + (q2 + q3)) * (1.f / kH) + 1e-5f);
}

#ifdef TRK_FUSED_PROF
__device__ unsigned long long g_fused_prof[4][24][8];
#define FPW(slot, stmt) do { long long _t0 = clock64(); stmt; pw[slot] += clock64() - _t0; } while (0)
#else
#define FPW(slot, stmt) stmt
#endif

template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads2, 1)
gnn_edge_fused2_kernel(const __grid_constant__ CUtensorMap tmW1, const __grid_constant__ CUtensorMap tmW2,
                       const __grid_constant__ CUtensorMap tmE, const __grid_constant__ CUtensorMap tmEst, Rows rows, FusedParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  Bars* bar = reinterpret_cast<Bars*>(smem + kOffBar);
  float* sb1 = reinterpret_cast<float*>(smem + kOffVec);
  float* sb2 = sb1 + kH;
  float* swo = sb2 + kH;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const bool leader = rank == 0;
  const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
  const int64_t M = resolve_rows(rows);
  const int64_t total = (M + 2 * kTileRows - 1) / (2 * kTileRows);
  const int n_my = total > pair ? (int)((total - pair + n_pairs - 1) / n_pairs) : 0;
#ifdef TRK_FUSED_PROF
  long long pw[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  const long long t_begin = clock64();
#endif

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmW1); prefetch_tmap(&tmW2); prefetch_tmap(&tmE); prefetch_tmap(&tmEst);
    mbar_init(&bar->w_full, 1);
    for (int i = 0; i < 2; ++i) {
      mbar_init(&bar->efull[i], 1);
      mbar_init(&bar->eempty[i], 4);
      mbar_init(&bar->gfull[i], 4);
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
  if (threadIdx.x >= 128 && threadIdx.x < 128 + kH) {
    const int c = threadIdx.x - 128;
    sb1[c] = p.b1[c];
    sb2[c] = MODE == gf::kUpdate ? p.b2[c] : 0.f;
    swo[c] = MODE == gf::kDecode ? p.w_out[c] : 0.f;
  }
  __syncthreads();
  mbar_wait(&bar->w_full, 0);
  tc_fence_before();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = bar->tmem_slot;
  const uint32_t sbase = smem_u32(smem);

  if (warp == 0) {
    // ---------------------------------------------------------------- TMA producer: e tiles (+ L2 prefetch two tiles ahead)
    if (lane == 0) {
      auto prefetch = [&](int tl) {
        if (tl < n_my) {
          const int64_t tile = pair + (int64_t)tl * n_pairs;
          const int row0 = (int)(tile * 2 * kTileRows + rank * kTileRows);
          for (int kb = 0; kb < 2; ++kb) tma_prefetch_l2_2d(&tmE, kb * 64, row0);
        }
      };
      prefetch(2);
      prefetch(3);
      for (int tl = 0; tl < n_my; ++tl) {
        const int64_t tile = pair + (int64_t)tl * n_pairs;
        const int b = tl & 1;
        const uint32_t ph = (tl >> 1) & 1;
        FPW(0, mbar_wait(&bar->eempty[b], ph ^ 1));
        if (leader) mbar_arrive_expect_tx(&bar->efull[b], 2 * 2 * kKB);
        const uint32_t full_leader = mapa_u32(smem_u32(&bar->efull[b]), 0);
        const int row0 = (int)(tile * 2 * kTileRows + rank * kTileRows);
        for (int kb = 0; kb < 2; ++kb) tma_load_2d_pair(smem + kOffEHold + (b * 2 + kb) * kKB, &tmE, full_leader, kb * 64, row0);
        prefetch(tl + 4);
      }
    }
  } else if (warp == 1) {
    // ---------------------------------------------------------------- MMA issuer (leader CTA): polls, issues what is ready
    if (leader && lane == 0) {
      constexpr uint32_t idesc = make_idesc_pair(kH);
      auto kblock = [&](uint32_t d_tmem, uint32_t a_addr, uint32_t b_addr, bool first) {
        const uint64_t adesc = make_smem_desc(a_addr), bdesc = make_smem_desc(b_addr);
#pragma unroll
        for (int k = 0; k < BK / UMMA_K; ++k)
          tc_mma_bf16_pair(d_tmem, adesc + (uint64_t)(k * 2), bdesc + (uint64_t)(k * 2), idesc, (!first || k != 0) ? 1u : 0u);
      };
      int n1 = 0, n2 = 0;      // next tile of layer 1 / layer 2
      int stage1 = 0;          // 0: waiting for the e tile and the accumulator, 1: e part issued, waiting for h_src, 2: for h_dst
      const int n2_end = MODE == gf::kUpdate ? n_my : 0;
      while (n1 < n_my || n2 < n2_end) {
        if (n2 < n2_end && n2 < n1) {
          const int b = n2 & 1;
          const uint32_t ph = (n2 >> 1) & 1;
          if (mbar_test(&bar->tfull, (uint32_t)(n2 & 1)) && mbar_test(&bar->a2empty[b], ph ^ 1)) {
            tc_fence_after();
            const uint32_t d = tmem_base + (uint32_t)(2 * kH + b * kH);
            for (int kb = 0; kb < 2; ++kb) kblock(d, sbase + kOffT + kb * kKB, sbase + kOffW2 + kb * kWKB, kb == 0);
            tc_commit_pair(&bar->tempty);
            tc_commit_pair(&bar->a2full[b]);
            ++n2;
          }
        }
        if (n1 < n_my) {
          const int b = n1 & 1;
          const uint32_t ph = (n1 >> 1) & 1;
          const uint32_t d = tmem_base + (uint32_t)(b * kH);
          if (stage1 == 0) {
            if (mbar_test(&bar->a1empty[b], ph ^ 1) && mbar_test(&bar->efull[b], ph)) {
              tc_fence_after();
              for (int kb = 0; kb < 2; ++kb) kblock(d, sbase + kOffEHold + (b * 2 + kb) * kKB, sbase + kOffW1 + (4 + kb) * kWKB, kb == 0);
              stage1 = 1;
            }
          }
          if (stage1 == 1 || stage1 == 2) {
            const int h = stage1 - 1;
            if (mbar_test(&bar->gfull[h], (uint32_t)(n1 & 1))) {
              tc_fence_after();
              for (int kb = 0; kb < 2; ++kb) kblock(d, sbase + kOffRing + (h * 2 + kb) * kKB, sbase + kOffW1 + (h * 2 + kb) * kWKB, false);
              tc_commit_pair(&bar->gempty[h]);
              if (h == 1) {
                tc_commit_pair(&bar->a1full[b]);
                stage1 = 0;
                ++n1;
              } else {
                stage1 = 2;
              }
            }
          }
        }
      }
    }
  } else if (warp < 4) {
    // ---------------------------------------------------------------- gather: h[src], h[dst] rows -> ring (64 rows per warp)
    const int gw = warp - 2;
    const uint32_t gfull0 = mapa_u32(smem_u32(&bar->gfull[0]), 0), gfull1 = mapa_u32(smem_u32(&bar->gfull[1]), 0);
    const int half = lane >> 4, chunk = lane & 15;
    const int kb = chunk >> 3, ch = chunk & 7;
    for (int tl = 0; tl < n_my; ++tl) {
      const int64_t tile = pair + (int64_t)tl * n_pairs;
      const int64_t row = tile * 2 * kTileRows + rank * kTileRows + gw * 64 + lane;
      const int s_lo = row < M ? p.src[row] : -1, d_lo = row < M ? p.dst[row] : -1;
      const int s_hi = row + 32 < M ? p.src[row + 32] : -1, d_hi = row + 32 < M ? p.dst[row + 32] : -1;
#pragma unroll 1
      for (int h = 0; h < 2; ++h) {
        FPW(h, mbar_wait(&bar->gempty[h], (uint32_t)(tl & 1) ^ 1));
        const int lo = h == 0 ? s_lo : d_lo, hi = h == 0 ? s_hi : d_hi;
#pragma unroll 8
        for (int i = 0; i < 32; ++i) {
          const int rr = i * 2 + half;                       // row inside this warp's 64 rows
          const int idx = __shfl_sync(0xffffffffu, rr < 32 ? lo : hi, rr & 31);
          const int rt = gw * 64 + rr;                       // row inside the CTA's tile
          const uint32_t dst = sbase + kOffRing + (h * 2 + kb) * kKB + rt * 128 + ((ch ^ (rt & 7)) << 4);
          const __nv_bfloat16* g = p.X + (int64_t)(idx < 0 ? 0 : idx) * p.ldx + chunk * 8;
          cp_async_16(dst, g, idx < 0 ? 0 : 16);             // rows beyond M are zero filled
        }
        cp_async_commit();
      }
      FPW(2, cp_async_wait<1>());
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive_remote(gfull0);
      FPW(3, cp_async_wait<0>());
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive_remote(gfull1);
    }
  } else if (warp < 8) {
    // ---------------------------------------------------------------- epilogue 1: acc1 -> LNR -> T (or score)
    const int quad = warp & 3;
    const int r = quad * 32 + lane;   // row of this thread inside the CTA's 128-row tile == TMEM lane
    const uint32_t a1empty0 = mapa_u32(smem_u32(&bar->a1empty[0]), 0), a1empty1 = mapa_u32(smem_u32(&bar->a1empty[1]), 0);
    const uint32_t tfull_l = mapa_u32(smem_u32(&bar->tfull), 0);
    for (int tl = 0; tl < n_my; ++tl) {
      const int64_t tile = pair + (int64_t)tl * n_pairs;
      const int b = tl & 1;
      const uint32_t ph = (tl >> 1) & 1;
      FPW(0, mbar_wait(&bar->a1full[b], ph));
      tc_fence_after();
      float x[kH];
      FPW(2, load_row(tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(b * kH), sb1, x));
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_remote(b == 0 ? a1empty0 : a1empty1);     // the accumulator is in registers now
      float mean, rstd;
      row_stats(x, p.use_ln, mean, rstd);
      const float shift = -mean * rstd;
      if (MODE == gf::kDecode) {
        float d0 = p.b_out, d1 = 0.f, d2 = 0.f, d3 = 0.f;
#pragma unroll
        for (int c = 0; c < kH; c += 4) {
          const float4 w = *reinterpret_cast<const float4*>(swo + c);
          d0 = fmaf(fmaxf(fmaf(x[c], rstd, shift), 0.f), w.x, d0);
          d1 = fmaf(fmaxf(fmaf(x[c + 1], rstd, shift), 0.f), w.y, d1);
          d2 = fmaf(fmaxf(fmaf(x[c + 2], rstd, shift), 0.f), w.z, d2);
          d3 = fmaf(fmaxf(fmaf(x[c + 3], rstd, shift), 0.f), w.w, d3);
        }
        const int64_t row = tile * 2 * kTileRows + rank * kTileRows + r;
        if (row < M) p.score[row] = fast_sigmoid((d0 + d1) + (d2 + d3));
        __syncwarp();
        if (lane == 0) mbar_arrive(&bar->eempty[b]);   // a1full: the layer-1 MMAs that read the e tile are complete
      } else {
        FPW(1, mbar_wait(&bar->tempty, (uint32_t)(tl & 1) ^ 1));   // the layer-2 MMA of the previous tile has read T
#pragma unroll
        for (int c = 0; c < kH; c += 8) {                  // 8 columns = one 16-byte chunk of the swizzled K block
          float f[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) f[i] = fmaxf(fmaf(x[c + i], rstd, shift), 0.f);
          const int kb = c >> 6, ch = (c & 63) >> 3;
          *reinterpret_cast<uint4*>(smem + kOffT + kb * kKB + r * 128 + ((ch ^ (r & 7)) << 4)) =
              make_uint4(pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
        }
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) mbar_arrive_remote(tfull_l);
      }
    }
  } else {
    // ---------------------------------------------------------------- epilogue 2: acc2 -> LNR -> + e -> store
    if (MODE == gf::kUpdate) {
      const int quad = warp & 3;
      const int r = quad * 32 + lane;
      const uint32_t a2empty0 = mapa_u32(smem_u32(&bar->a2empty[0]), 0), a2empty1 = mapa_u32(smem_u32(&bar->a2empty[1]), 0);
      for (int tl = 0; tl < n_my; ++tl) {
        const int64_t tile = pair + (int64_t)tl * n_pairs;
        const int b = tl & 1;
        const uint32_t ph = (tl >> 1) & 1;
        FPW(0, mbar_wait(&bar->a2full[b], ph));
        tc_fence_after();
        float x[kH];
        FPW(2, load_row(tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(2 * kH + b * kH), sb2, x));
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_remote(b == 0 ? a2empty0 : a2empty1);
        float mean, rstd;
        row_stats(x, p.use_ln, mean, rstd);
        const float shift = -mean * rstd;
        uint8_t* eh = smem + kOffEHold + b * 2 * kKB;
#pragma unroll
        for (int c = 0; c < kH; c += 8) {
          const int kb = c >> 6, ch = (c & 63) >> 3;
          uint4* cell = reinterpret_cast<uint4*>(eh + kb * kKB + r * 128 + ((ch ^ (r & 7)) << 4));
          const uint4 e = *cell;
          const __nv_bfloat162* e2 = reinterpret_cast<const __nv_bfloat162*>(&e);
          float f[8];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            f[2 * i] = fmaxf(fmaf(x[c + 2 * i], rstd, shift), 0.f) + __low2float(e2[i]);
            f[2 * i + 1] = fmaxf(fmaf(x[c + 2 * i + 1], rstd, shift), 0.f) + __high2float(e2[i]);
          }
          *cell = make_uint4(pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
        }
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) {
          const int row0 = (int)(tile * 2 * kTileRows + rank * kTileRows + quad * 32);
          for (int kb = 0; kb < 2; ++kb) tma_store_2d(&tmEst, eh + kb * kKB + quad * 32 * 128, kb * 64, row0);
          bulk_commit();
          FPW(1, bulk_wait_read<0>());          // the tile's rows have left shared memory: the buffer may be refilled
          mbar_arrive(&bar->eempty[b]);
        }
      }
      if (lane == 0) bulk_wait_all();
    }
  }
#ifdef TRK_FUSED_PROF
  if (MODE == gf::kUpdate && blockIdx.x < 4 && lane == 0) {
    for (int i = 0; i < 7; ++i) g_fused_prof[blockIdx.x][warp][i] = (unsigned long long)pw[i];
    g_fused_prof[blockIdx.x][warp][7] = (unsigned long long)(clock64() - t_begin);
  }
#endif
  tc_fence_before();
  cluster_sync_all();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_pair<512>(tmem_base);
  }
}

}  // namespace gf2
}  // namespace trk

// Fused interaction-network edge update of S4 for H = 128 on CTA pairs, third version (reading C-12):
//
//   e_k <- e_k + LNR(W2 LNR(W1 [h_src(k) ; h_dst(k) ; e_k] + b1) + b2)           (kUpdate)
//   score_k = sigmoid(w_out . LNR(W1 [h_src ; h_dst ; e_k] + b1) + b_out)        (kDecode)
//   h_v <- h_v + LNR(W2 LNR(W1 [h_v ; m_in_v ; m_out_v] + b1) + b2)              (kNode: the node update, rows of X)
//
// kNode runs the same pipeline on the node table X [n][3H] = (h | m_in | m_out): all six K blocks of the operand come by
// TMA (h takes the place of the e tile: operand copy + residual copy, new h stored in place; m_in | m_out take the place of
// the gathered rows), the gather warps idle.
//
// Same arithmetic and data flow as gnn_fused2.cuh.  What changed, from the per-role wait profile of version 2
// (profiles/r1_fused_roles_v3.md: no role busier than 65 %, the tile period set by the chain  e-tile load -> MMA 1 ->
// epilogue 1 -> MMA 2 -> epilogue 2 -> TMA store -> buffer free  with only two e tiles in flight):
//   * the e tile is held twice, for two different lifetimes: EOp (the layer-1 operand, free again as soon as MMA 1 has
//     read it; its K blocks are issued LAST in MMA 1 so the next tile's load hides behind the h blocks) and Res (the
//     residual / output staging of epilogue 2, a second TMA load of the same rows that hits L2).  Both are single
//     buffers, so shared memory stays at 227 KB, but no buffer is held across the whole chain any more;
//   * the TMA warp polls both buffers instead of serving them in program order;
//   * the gather loop is 3 instructions per 16-byte cp.async (shuffle, address, copy): swizzle terms and the destination
//     rows are compile-time offsets; rows beyond M gather row 0 instead of being zero filled (their results are never read);
//   * the LayerNorm epilogues use the packed fp32x2 add / fma of sm_100 (half the issue slots).
// Warps as in version 2: 0 TMA, 1 MMA issuer (leader CTA) + TMEM owner, 2-3 gather, 4-7 epilogue 1, 8-11 epilogue 2.
// TMEM: acc1[2] (columns 0,128) and acc2[2] (256,384).  mbarriers marked L live in the leader CTA's copy (both CTAs arrive).
#pragma once

#include "gnn_fused2.cuh"

namespace trk {
namespace gf3 {

using namespace tc;
using gf::cp_async_16;
using gf::cp_async_commit;
using gf::cp_async_wait;
using gf::FusedParams;
using gf::kH;
using gf::kKB;
using gf::kTileRows;
using gf::kWKB;
using gf2::mbar_arrive_remote;
using gf2::mbar_test;
using gf2::tma_prefetch_l2_2d;

constexpr int kThreads3 = 12 * 32;
constexpr int kNode = 2;                        // third mode besides gf::kUpdate / gf::kDecode
constexpr int kOffW1 = 0;                       // 6 K blocks of this CTA's 64 output rows of W1
constexpr int kOffW2 = kOffW1 + 6 * kWKB;       // 2 K blocks of W2
constexpr int kOffRing = kOffW2 + 2 * kWKB;     // 4 K blocks: h_src (2), h_dst (2)
constexpr int kOffEOp = kOffRing + 4 * kKB;     // 2 K blocks: the e tile as layer-1 operand
constexpr int kOffRes = kOffEOp + 2 * kKB;      // 2 K blocks: the e tile as residual, overwritten in place and stored
constexpr int kOffT = kOffRes + 2 * kKB;        // 2 K blocks: layer-1 output
constexpr int kOffVec = kOffT + 2 * kKB;        // b1, b2, w_out: 3 x 128 fp32
constexpr int kOffBar = kOffVec + 3 * kH * 4;
constexpr int kSmemFused3 = kOffBar + 256 + 1024;
static_assert(kSmemFused3 <= 232448, "shared memory budget of one CTA");

struct Bars {
  uint64_t w_full;
  uint64_t eopfull;       // L  tx: both CTAs' operand tiles
  uint64_t eopempty;      //    own, multicast commit (MMA 1 has read the operand tile)
  uint64_t resfull;       //    own, tx: this CTA's residual tile
  uint64_t resempty;      //    own, 4 arrivals (epilogue-2 warps, after their rows have left shared memory)
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

__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }

// One accumulator row (this thread's TMEM lane, 128 fp32 columns) + bias -> 64 packed pairs.
__device__ __forceinline__ void load_row2(uint32_t taddr, const float* __restrict__ sbias, float2 (&x)[kH / 2]) {
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
    x[i / 2] = __fadd2_rn(f2(__uint_as_float(u0[i]), __uint_as_float(u0[i + 1])), f2(b0.x, b0.y));
    x[i / 2 + 1] = __fadd2_rn(f2(__uint_as_float(u0[i + 2]), __uint_as_float(u0[i + 3])), f2(b0.z, b0.w));
    x[16 + i / 2] = __fadd2_rn(f2(__uint_as_float(u1[i]), __uint_as_float(u1[i + 1])), f2(b1.x, b1.y));
    x[16 + i / 2 + 1] = __fadd2_rn(f2(__uint_as_float(u1[i + 2]), __uint_as_float(u1[i + 3])), f2(b1.z, b1.w));
    x[32 + i / 2] = __fadd2_rn(f2(__uint_as_float(u2[i]), __uint_as_float(u2[i + 1])), f2(b2.x, b2.y));
    x[32 + i / 2 + 1] = __fadd2_rn(f2(__uint_as_float(u2[i + 2]), __uint_as_float(u2[i + 3])), f2(b2.z, b2.w));
    x[48 + i / 2] = __fadd2_rn(f2(__uint_as_float(u3[i]), __uint_as_float(u3[i + 1])), f2(b3.x, b3.y));
    x[48 + i / 2 + 1] = __fadd2_rn(f2(__uint_as_float(u3[i + 2]), __uint_as_float(u3[i + 3])), f2(b3.z, b3.w));
  }
}

// LayerNorm statistics of a register row (biased variance, eps 1e-5; two passes, four independent packed chains each).
__device__ __forceinline__ void row_stats2(const float2 (&x)[kH / 2], int use_ln, float& mean, float& rstd) {
  if (!use_ln) {
    mean = 0.f;
    rstd = 1.f;
    return;
  }
  float2 s0 = f2(0.f, 0.f), s1 = s0, s2 = s0, s3 = s0;
#pragma unroll
  for (int i = 0; i < kH / 2; i += 4) {
    s0 = __fadd2_rn(s0, x[i]); s1 = __fadd2_rn(s1, x[i + 1]); s2 = __fadd2_rn(s2, x[i + 2]); s3 = __fadd2_rn(s3, x[i + 3]);
  }
  const float2 s = __fadd2_rn(__fadd2_rn(s0, s1), __fadd2_rn(s2, s3));
  mean = (s.x + s.y) * (1.f / kH);
  const float2 nm = f2(-mean, -mean);
  float2 q0 = f2(0.f, 0.f), q1 = q0, q2 = q0, q3 = q0;
#pragma unroll
  for (int i = 0; i < kH / 2; i += 4) {
    const float2 d0 = __fadd2_rn(x[i], nm), d1 = __fadd2_rn(x[i + 1], nm), d2 = __fadd2_rn(x[i + 2], nm), d3 = __fadd2_rn(x[i + 3], nm);
    q0 = __ffma2_rn(d0, d0, q0); q1 = __ffma2_rn(d1, d1, q1); q2 = __ffma2_rn(d2, d2, q2); q3 = __ffma2_rn(d3, d3, q3);
  }
  const float2 q = __fadd2_rn(__fadd2_rn(q0, q1), __fadd2_rn(q2, q3));
  rstd = rsqrtf((q.x + q.y) * (1.f / kH) + 1e-5f);
}

template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads3, 1)
gnn_edge_fused3_kernel(const __grid_constant__ CUtensorMap tmW1, const __grid_constant__ CUtensorMap tmW2,
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
  constexpr bool kTwoLayers = MODE != gf::kDecode;
  // K blocks of W1 that go with the operand tile (e, or h in kNode) and with the two ring halves
  constexpr int kbE = MODE == kNode ? 0 : 4;
  constexpr int kbR = MODE == kNode ? 2 : 0;
  constexpr int colE = 0;                        // first column of the operand / residual tile in its tensor
#ifdef TRK_FUSED_PROF
  long long pw[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  const long long t_begin = clock64();
#endif

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmW1); prefetch_tmap(&tmW2); prefetch_tmap(&tmE); prefetch_tmap(&tmEst);
    mbar_init(&bar->w_full, 1);
    mbar_init(&bar->eopfull, 1);
    mbar_init(&bar->eopempty, 1);
    mbar_init(&bar->resfull, 1);
    mbar_init(&bar->resempty, 4);
    for (int i = 0; i < 2; ++i) {
      mbar_init(&bar->gfull[i], MODE == kNode ? 1 : 4);
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
    sb2[c] = kTwoLayers ? p.b2[c] : 0.f;
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
    // ---------------------------------------------------------------- TMA producer: operand and residual copies of the e tiles
    if (lane == 0) {
      auto row0_of = [&](int tl) { return (int)((pair + (int64_t)tl * n_pairs) * 2 * kTileRows + rank * kTileRows); };
      auto prefetch = [&](int tl) {
        if (tl < n_my)
          for (int kb = 0; kb < (MODE == kNode ? 6 : 2); ++kb) tma_prefetch_l2_2d(&tmE, kb * 64, row0_of(tl));
      };
      prefetch(1);
      prefetch(2);
      const uint32_t eopfull_leader = mapa_u32(smem_u32(&bar->eopfull), 0);
      const uint32_t gfull_leader[2] = {mapa_u32(smem_u32(&bar->gfull[0]), 0), mapa_u32(smem_u32(&bar->gfull[1]), 0)};
      int n_op = 0, n_res = 0, n_g[2] = {0, 0};
      const int res_end = kTwoLayers ? n_my : 0;
      const int g_end = MODE == kNode ? n_my : 0;
      while (n_op < n_my || n_res < res_end || n_g[0] < g_end || n_g[1] < g_end) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {              // kNode: m_in | m_out blocks into the ring halves
          if (n_g[h] < g_end && mbar_test(&bar->gempty[h], (uint32_t)(n_g[h] & 1) ^ 1)) {
            if (leader) mbar_arrive_expect_tx(&bar->gfull[h], 2 * 2 * kKB);
            for (int kb = 0; kb < 2; ++kb)
              tma_load_2d_pair(smem + kOffRing + (h * 2 + kb) * kKB, &tmE, gfull_leader[h], kH + h * kH + kb * 64, row0_of(n_g[h]));
            ++n_g[h];
          }
        }
        if (n_op < n_my && mbar_test(&bar->eopempty, (uint32_t)(n_op & 1) ^ 1)) {
          if (leader) mbar_arrive_expect_tx(&bar->eopfull, 2 * 2 * kKB);
          for (int kb = 0; kb < 2; ++kb) tma_load_2d_pair(smem + kOffEOp + kb * kKB, &tmE, eopfull_leader, colE + kb * 64, row0_of(n_op));
          prefetch(n_op + 3);
          ++n_op;
        }
        // the residual copy of tile t is asked for only after its operand copy, so it finds the rows in L2
        if (n_res < res_end && n_res < n_op && mbar_test(&bar->resempty, (uint32_t)(n_res & 1) ^ 1)) {
          mbar_arrive_expect_tx(&bar->resfull, 2 * kKB);
          for (int kb = 0; kb < 2; ++kb) tma_load_2d(smem + kOffRes + kb * kKB, &tmE, &bar->resfull, colE + kb * 64, row0_of(n_res));
          ++n_res;
        }
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
      int stage1 = 0;          // 0: waiting for the accumulator and h_src, 1: for h_dst, 2: for the e operand tile
      const int n2_end = kTwoLayers ? n_my : 0;
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
            if (mbar_test(&bar->a1empty[b], ph ^ 1) && mbar_test(&bar->gfull[0], (uint32_t)(n1 & 1))) {
              tc_fence_after();
              for (int kb = 0; kb < 2; ++kb) kblock(d, sbase + kOffRing + kb * kKB, sbase + kOffW1 + (kbR + kb) * kWKB, kb == 0);
              tc_commit_pair(&bar->gempty[0]);
              stage1 = 1;
            }
          }
          if (stage1 == 1) {
            if (mbar_test(&bar->gfull[1], (uint32_t)(n1 & 1))) {
              tc_fence_after();
              for (int kb = 0; kb < 2; ++kb) kblock(d, sbase + kOffRing + (2 + kb) * kKB, sbase + kOffW1 + (kbR + 2 + kb) * kWKB, false);
              tc_commit_pair(&bar->gempty[1]);
              stage1 = 2;
            }
          }
          if (stage1 == 2) {
            if (mbar_test(&bar->eopfull, (uint32_t)(n1 & 1))) {
              tc_fence_after();
              for (int kb = 0; kb < 2; ++kb) kblock(d, sbase + kOffEOp + kb * kKB, sbase + kOffW1 + (kbE + kb) * kWKB, false);
              tc_commit_pair(&bar->eopempty);
              tc_commit_pair(&bar->a1full[b]);
              stage1 = 0;
              ++n1;
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
    // iteration i copies chunk `chunk` of row rr = 2 i + half of this warp's 64 rows; (rr & 7) = 2 (i & 3) + half
    uint32_t sw[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) sw[j] = (uint32_t)((ch ^ (2 * j + half)) << 4);
    const uint32_t dst0 = sbase + kOffRing + kb * kKB + (gw * 64 + half) * 128;
    const char* xb = reinterpret_cast<const char*>(p.X) + chunk * 16;
    const int64_t ldb = p.ldx * 2;
    for (int tl = 0; tl < (MODE == kNode ? 0 : n_my); ++tl) {
      const int64_t tile = pair + (int64_t)tl * n_pairs;
      const int64_t row = tile * 2 * kTileRows + rank * kTileRows + gw * 64 + lane;
      // rows beyond M gather node 0: their results are computed but never read (segment sums and scores stop at M)
      const int s_lo = row < M ? p.src[row] : 0, d_lo = row < M ? p.dst[row] : 0;
      const int s_hi = row + 32 < M ? p.src[row + 32] : 0, d_hi = row + 32 < M ? p.dst[row + 32] : 0;
#pragma unroll 1
      for (int h = 0; h < 2; ++h) {
        FPW(h, mbar_wait(&bar->gempty[h], (uint32_t)(tl & 1) ^ 1));
        const int lo = h == 0 ? s_lo : d_lo, hi = h == 0 ? s_hi : d_hi;
        const uint32_t dsth = dst0 + h * 2 * kKB;
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          const int idx = __shfl_sync(0xffffffffu, i < 16 ? lo : hi, (2 * i + half) & 31);
          cp_async_16(dsth + i * 256 + sw[i & 3], xb + (int64_t)idx * ldb, 16);
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
      float2 x[kH / 2];
      FPW(2, load_row2(tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(b * kH), sb1, x));
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_remote(b == 0 ? a1empty0 : a1empty1);     // the accumulator is in registers now
      float mean, rstd;
      row_stats2(x, p.use_ln, mean, rstd);
      const float2 rs = f2(rstd, rstd), sh = f2(-mean * rstd, -mean * rstd);
      if (MODE == gf::kDecode) {
        float2 d0 = f2(p.b_out, 0.f), d1 = f2(0.f, 0.f);
#pragma unroll
        for (int c = 0; c < kH; c += 4) {
          const float4 w = *reinterpret_cast<const float4*>(swo + c);
          float2 v0 = __ffma2_rn(x[c / 2], rs, sh), v1 = __ffma2_rn(x[c / 2 + 1], rs, sh);
          v0.x = fmaxf(v0.x, 0.f); v0.y = fmaxf(v0.y, 0.f); v1.x = fmaxf(v1.x, 0.f); v1.y = fmaxf(v1.y, 0.f);
          d0 = __ffma2_rn(v0, f2(w.x, w.y), d0);
          d1 = __ffma2_rn(v1, f2(w.z, w.w), d1);
        }
        const int64_t row = tile * 2 * kTileRows + rank * kTileRows + r;
        if (row < M) p.score[row] = fast_sigmoid((d0.x + d0.y) + (d1.x + d1.y));
      } else {
        FPW(1, mbar_wait(&bar->tempty, (uint32_t)(tl & 1) ^ 1));   // the layer-2 MMA of the previous tile has read T
#pragma unroll
        for (int c = 0; c < kH; c += 8) {                  // 8 columns = one 16-byte chunk of the swizzled K block
          uint32_t w[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const float2 v = __ffma2_rn(x[c / 2 + i], rs, sh);
            w[i] = pack_bf16(fmaxf(v.x, 0.f), fmaxf(v.y, 0.f));
          }
          const int kb = c >> 6, ch = (c & 63) >> 3;
          *reinterpret_cast<uint4*>(smem + kOffT + kb * kKB + r * 128 + ((ch ^ (r & 7)) << 4)) = make_uint4(w[0], w[1], w[2], w[3]);
        }
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) mbar_arrive_remote(tfull_l);
      }
    }
  } else {
    // ---------------------------------------------------------------- epilogue 2: acc2 -> LNR -> + e -> store
    if (kTwoLayers) {
      const int quad = warp & 3;
      const int r = quad * 32 + lane;
      const uint32_t a2empty0 = mapa_u32(smem_u32(&bar->a2empty[0]), 0), a2empty1 = mapa_u32(smem_u32(&bar->a2empty[1]), 0);
      uint8_t* res = smem + kOffRes;
      for (int tl = 0; tl < n_my; ++tl) {
        const int64_t tile = pair + (int64_t)tl * n_pairs;
        const int b = tl & 1;
        const uint32_t ph = (tl >> 1) & 1;
        FPW(0, mbar_wait(&bar->a2full[b], ph));
        tc_fence_after();
        float2 x[kH / 2];
        FPW(2, load_row2(tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(2 * kH + b * kH), sb2, x));
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_remote(b == 0 ? a2empty0 : a2empty1);
        float mean, rstd;
        row_stats2(x, p.use_ln, mean, rstd);
        const float2 rs = f2(rstd, rstd), sh = f2(-mean * rstd, -mean * rstd);
        FPW(3, mbar_wait(&bar->resfull, (uint32_t)(tl & 1)));      // the residual copy of this tile has landed
#pragma unroll
        for (int c = 0; c < kH; c += 8) {
          const int kb = c >> 6, ch = (c & 63) >> 3;
          uint4* cell = reinterpret_cast<uint4*>(res + kb * kKB + r * 128 + ((ch ^ (r & 7)) << 4));
          const uint4 e = *cell;
          const __nv_bfloat162* e2 = reinterpret_cast<const __nv_bfloat162*>(&e);
          uint32_t w[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            float2 v = __ffma2_rn(x[c / 2 + i], rs, sh);
            v.x = fmaxf(v.x, 0.f);
            v.y = fmaxf(v.y, 0.f);
            v = __fadd2_rn(v, __bfloat1622float2(e2[i]));
            w[i] = pack_bf16(v.x, v.y);
          }
          *cell = make_uint4(w[0], w[1], w[2], w[3]);
        }
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) {
          const int row0 = (int)(tile * 2 * kTileRows + rank * kTileRows + quad * 32);
          for (int kb = 0; kb < 2; ++kb) tma_store_2d(&tmEst, res + kb * kKB + quad * 32 * 128, colE + kb * 64, row0);
          bulk_commit();
          FPW(1, bulk_wait_read<0>());  // the tile's rows have left shared memory: the buffer may be refilled
          mbar_arrive(&bar->resempty);
        }
      }
      if (lane == 0) bulk_wait_all();
    }
  }
#ifdef TRK_FUSED_PROF
  if (MODE == gf::kUpdate && blockIdx.x < 4 && lane == 0) {
    for (int i = 0; i < 7; ++i) gf2::g_fused_prof[blockIdx.x][warp][i] = (unsigned long long)pw[i];
    gf2::g_fused_prof[blockIdx.x][warp][7] = (unsigned long long)(clock64() - t_begin);
  }
#endif
  tc_fence_before();
  cluster_sync_all();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_pair<512>(tmem_base);
  }
}

}  // namespace gf3
}  // namespace trk

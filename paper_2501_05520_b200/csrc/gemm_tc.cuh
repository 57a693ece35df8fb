// tcgen05 / TMEM / TMA GEMM for sm_100a:   acc[m][n] = sum_k A[m][k] * W[n][k]   (bf16 x bf16 -> fp32)
// followed by a fused epilogue.  Used by every dense layer of S1, S3 and S4 in TRK_BF16 precision
// (BASELINE.json north_star: "tcgen05/TMEM tensor-core GEMMs fed by TMA with bf16 inputs and fp32
// accumulation").
//
// Shape of one CTA (192 threads, 1 CTA per SM, persistent over output tiles):
//   warp 0      TMA producer: A tile 128 x 64 and W tile BN x 64 (both K-major, 128-byte swizzle)
//               into a STAGES-deep shared-memory ring, completion on mbarriers;
//   warp 1      MMA issuer: one thread issues tcgen05.mma (M = 128, N = BN, K = 16) four times per
//               ring slot; tcgen05.commit frees the slot; accumulators are double buffered in TMEM
//               so the epilogue of tile t overlaps the MMAs of tile t+1;
//   warps 2..5  epilogue: tcgen05.ld (32 lanes x 32 columns per warp) -> registers -> fused math -> global.
// The row count may live on the device (rows = clamp(*m_dev - m_off, 0, m_cap)) so that no stage
// of trk_infer needs a host synchronisation.
#pragma once

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace trk {
namespace tc {

constexpr int BM = 128;
constexpr int BK = 64;          // 64 bf16 = 128 bytes = one SWIZZLE_128B row
constexpr int UMMA_K = 16;
constexpr int kThreads = 192;
constexpr int kEpiWarps = 4;

struct Rows {                   // rows = m_dev ? clamp(*m_dev - m_off, 0, m_cap) : m_cap
  const int32_t* m_dev;
  int64_t m_off;
  int64_t m_cap;
};

__device__ __forceinline__ int64_t resolve_rows(const Rows& r) {
  if (!r.m_dev) return r.m_cap;
  int64_t m = (int64_t)*r.m_dev - r.m_off;
  return m < 0 ? 0 : (m > r.m_cap ? r.m_cap : m);
}

// ------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap* m) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(m)) : "memory");
}
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* tmap, uint64_t* bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
          smem_u32(smem_dst)),
      "l"(reinterpret_cast<uint64_t>(tmap)), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
      : "memory");
}

// TMA store of a shared-memory box (bulk async group completion)
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* tmap, const void* smem_src, int c0, int c1) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];" ::"l"(reinterpret_cast<uint64_t>(tmap)),
               "r"(smem_u32(smem_src)), "r"(c0), "r"(c1)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <int NCOLS>
__device__ __forceinline__ void tmem_alloc(uint32_t* smem_slot) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_slot)), "n"(NCOLS) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
template <int NCOLS>
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "n"(NCOLS) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// D[tmem] (+)= A[smem desc] * B[smem desc]^T, kind::f16 (bf16 operands, fp32 accumulate)
__device__ __forceinline__ void tc_mma_bf16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
        "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]),
        "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Shared-memory matrix descriptor: K-major tile, rows of 128 bytes, SWIZZLE_128B, 8-row groups 1024 B apart.
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t smem_addr) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);  // start address   [0,14)
  d |= (uint64_t)1 << 16;                        // leading byte offset (unused for swizzled K-major) [16,30)
  d |= (uint64_t)(1024 >> 4) << 32;              // stride byte offset: 8 rows x 128 B               [32,46)
  d |= (uint64_t)1 << 46;                        // descriptor version (Blackwell)                   [46,48)
  d |= (uint64_t)2 << 61;                        // SWIZZLE_128B                                      [61,64)
  return d;
}
// Instruction descriptor, kind::f16: D fp32, A/B bf16, both K-major, M = 128, N = BN.
__host__ __device__ constexpr uint32_t make_idesc(int bn) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(bn >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
}

constexpr int tmem_cols_for(int bn) { return 2 * bn <= 32 ? 32 : (2 * bn <= 64 ? 64 : (2 * bn <= 128 ? 128 : (2 * bn <= 256 ? 256 : 512))); }
constexpr int stage_bytes(int bn) { return (BM + bn) * BK * 2; }
constexpr int kStoreStage = 2 * 32 * 128;   // per epilogue warp: two 32-row x 128-byte boxes (TMA-store staging)
// SPLIT = 2 doubles the epilogue warps (two per TMEM lane quadrant, each taking half of the tile's columns): for layers whose
// K loop is one block long the epilogue, not the tensor pipe, paces a tile.  Their staging takes the room of one ring stage.
constexpr int num_stages(int bn, int split = 1) {
  return ((196 - 32 * (split - 1)) * 1024) / stage_bytes(bn) > 8 ? 8 : ((196 - 32 * (split - 1)) * 1024) / stage_bytes(bn);
}
constexpr int smem_bytes(int bn, bool tma_store = false, int split = 1) {
  return num_stages(bn, split) * stage_bytes(bn) + (tma_store ? split * kEpiWarps * kStoreStage : 0) + 1024 /*alignment*/ + 256 /*barriers*/;
}
constexpr int kGatherWarps = 4;
constexpr int threads_for(int split, bool gather = false) { return 64 + 32 * kEpiWarps * split + (gather ? 32 * kGatherWarps : 0); }

// GATHER_A: the A tile of a one-K-block layer is not loaded by TMA but assembled by four gather warps straight into the
// swizzled operand layout: row m = bf16([feat[src[m]] ; feat[dst[m]]]) zero padded to 64 columns (the S3 filter input).
struct AGather {
  const float* feat;      // fp32 [n][u]
  const int32_t* src;     // indexed by rows.m_off + m
  const int32_t* dst;
  int u;                  // 2 u <= 64
};

// What an epilogue may use besides its own parameters: a per-warp staging area and the output tensor map.
struct EpiShared {
  uint8_t* stage;           // kStoreStage bytes, 1024-byte aligned (only when Epi::kTmaStore)
  const CUtensorMap* tmC;
  uint32_t chunk;           // running count of staged boxes of this warp (selects the half of `stage`)
};

// ------------------------------------------------------------------ the kernel
// Epi::run(params, tmem_tile_addr (lane and column base of this warp's quadrant), row0 (first row of the
//          tile), col0 (first column of the tile), n_blk, rows M, lane-row index r, release()) must call
//          `release` exactly once after its last TMEM read.
__device__ __forceinline__ uint32_t pack_bf16(float a, float b);

template <int BN, class Epi, int SPLIT = 1, bool GATHER_A = false>
__global__ void __launch_bounds__(threads_for(SPLIT, GATHER_A), 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const __grid_constant__ CUtensorMap tmC,
               Rows rows, int n_tiles, int k_blocks, typename Epi::Params ep, AGather ag) {
  TRK_GRID_DEP_WAIT();
  constexpr int STAGES = num_stages(BN, SPLIT);
  constexpr int A_BYTES = BM * BK * 2;
  constexpr int STAGE = stage_bytes(BN);
  constexpr int TMEM_COLS = tmem_cols_for(BN);
  static_assert(SPLIT == 1 || (SPLIT == 2 && BN % 128 == 0), "column split of the epilogue");
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint8_t* store_stage = smem + STAGES * STAGE;
  uint64_t* full_bar = reinterpret_cast<uint64_t*>(store_stage + (Epi::kTmaStore ? SPLIT * kEpiWarps * kStoreStage : 0));
  uint64_t* empty_bar = full_bar + STAGES;
  uint64_t* tfull_bar = empty_bar + STAGES;
  uint64_t* tempty_bar = tfull_bar + 2;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty_bar + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t M = resolve_rows(rows);
  const int64_t m_tiles = (M + BM - 1) / BM;
  const int64_t total = m_tiles * n_tiles;
  // This CTA's j-th tile.  Default: tiles in grid strides, n fastest (co-resident CTAs share A rows in L2).  GATHER_A: a CTA
  // takes row blocks in grid strides and walks all their column tiles, so the gathered rows are loaded once per row block.
  const int64_t n_iter = GATHER_A ? ((int64_t)blockIdx.x < m_tiles ? (m_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x * n_tiles : 0)
                                  : ((int64_t)blockIdx.x < total ? (total - blockIdx.x + gridDim.x - 1) / gridDim.x : 0);
  auto tile_of = [&](int64_t j, int& m_blk, int& n_blk) {
    if (GATHER_A) {
      m_blk = (int)(blockIdx.x + (j / n_tiles) * gridDim.x);
      n_blk = (int)(j % n_tiles);
    } else {
      const int64_t tile = blockIdx.x + j * gridDim.x;
      m_blk = (int)(tile / n_tiles);
      n_blk = (int)(tile % n_tiles);
    }
  };

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmA);
    prefetch_tmap(&tmB);
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(&full_bar[s], GATHER_A ? 1 + kGatherWarps : 1);
      mbar_init(&empty_bar[s], 1);
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(&tfull_bar[s], 1);
      mbar_init(&tempty_bar[s], kEpiWarps * SPLIT);
    }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc<TMEM_COLS>(tmem_slot);
  tc_fence_before();
  __syncthreads();
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
          mbar_arrive_expect_tx(&full_bar[stage], GATHER_A ? STAGE - A_BYTES : STAGE);
          uint8_t* sa = smem + stage * STAGE;
          if (!GATHER_A) tma_load_2d(sa, &tmA, &full_bar[stage], kb * BK, m_blk * BM);
          tma_load_2d(sa + A_BYTES, &tmB, &full_bar[stage], kb * BK, n_blk * BN);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      constexpr uint32_t idesc = make_idesc(BN);
      int stage = 0;
      uint32_t phase = 0;
      int as = 0;
      uint32_t aphase = 0;
      for (int64_t j = 0; j < n_iter; ++j) {
        mbar_wait(&tempty_bar[as], aphase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(as * BN);
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(smem + stage * STAGE);
          const uint64_t adesc = make_smem_desc(sa);
          const uint64_t bdesc = make_smem_desc(sa + A_BYTES);
#pragma unroll
          for (int k = 0; k < BK / UMMA_K; ++k)   // +32 bytes per K step inside the 128-byte swizzle row
            tc_mma_bf16(d_tmem, adesc + (uint64_t)(k * 2), bdesc + (uint64_t)(k * 2), idesc, (kb | k) != 0 ? 1u : 0u);
          tc_commit(&empty_bar[stage]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        tc_commit(&tfull_bar[as]);
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
  } else if (GATHER_A && warp >= 2 + kEpiWarps * SPLIT) {
    // gather warps: one row per thread (k_blocks == 1).  The row of the NEXT row block is loaded (2 u scalar loads, packed to
    // bf16 pairs) while the current one is written into the ring once per column tile, so no load latency is exposed.
    const int r = (warp - 2 - kEpiWarps * SPLIT) * 32 + lane;
    int stage = 0;
    uint32_t phase = 0;
    auto load_row = [&](int64_t m_blk, uint32_t (&pk)[BK / 2]) {
      const int64_t m = m_blk * BM + r;
      float v[BK];
#pragma unroll
      for (int c = 0; c < BK; ++c) v[c] = 0.f;
      if (m_blk < m_tiles && m < M) {
        const int64_t si = ag.src[rows.m_off + m], di = ag.dst[rows.m_off + m];
        const float* fs = ag.feat + si * ag.u;
        const float* fd = ag.feat + di * ag.u;
#pragma unroll
        for (int c = 0; c < BK / 2; ++c)
          if (c < ag.u) v[c] = __ldg(fs + c);
#pragma unroll
        for (int c = 0; c < BK; ++c)
          if (c >= ag.u && c < 2 * ag.u) v[c] = __ldg(fd + (c - ag.u));
      }
#pragma unroll
      for (int c = 0; c < BK / 2; ++c) pk[c] = pack_bf16(v[2 * c], v[2 * c + 1]);
    };
    uint32_t cur[BK / 2], nxt[BK / 2];
    load_row(blockIdx.x, cur);
    for (int64_t mb = blockIdx.x; mb < m_tiles; mb += gridDim.x) {
      load_row(mb + gridDim.x, nxt);
      for (int nb = 0; nb < n_tiles; ++nb) {
        mbar_wait(&empty_bar[stage], phase ^ 1);
        uint8_t* sa = smem + stage * STAGE;
#pragma unroll
        for (int q = 0; q < 8; ++q)
          *reinterpret_cast<uint4*>(sa + r * 128 + ((q ^ (r & 7)) << 4)) = make_uint4(cur[q * 4], cur[q * 4 + 1], cur[q * 4 + 2], cur[q * 4 + 3]);
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) mbar_arrive(&full_bar[stage]);
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
#pragma unroll
      for (int c = 0; c < BK / 2; ++c) cur[c] = nxt[c];
    }
  } else {
    const int quad = warp & 3;   // TMEM lane quadrant this warp may access
    const int chalf = (warp - 2) >> 2;   // SPLIT == 2: which half of the tile's columns
    constexpr int BNE = BN / SPLIT;
    int as = 0;
    uint32_t aphase = 0;
    EpiShared es{store_stage + (warp - 2) * kStoreStage, &tmC, 0u};
    for (int64_t j = 0; j < n_iter; ++j) {
      int m_blk, n_blk;
      tile_of(j, m_blk, n_blk);
      mbar_wait(&tfull_bar[as], aphase);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(as * BN + chalf * BNE);
      uint64_t* rel = &tempty_bar[as];
      auto release = [&]() {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(rel);
      };
      Epi::template run<BNE>(ep, taddr, (int64_t)m_blk * BM + quad * 32 + lane, n_blk * BN + chalf * BNE, n_blk, M, release, es);
      if (++as == 2) { as = 0; aphase ^= 1; }
    }
    if (Epi::kTmaStore && lane == 0) bulk_wait_all();   // staged boxes must be read before the CTA's shared memory goes away
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc<TMEM_COLS>(tmem_base);
  }
}

// ------------------------------------------------------------------ epilogues
__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
  __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ float fast_sigmoid(float x) { return 1.f / (1.f + __expf(-x)); }

// out[m][n] = act(acc + bias[n]) as bf16.  Each warp stages 32 rows x 64 columns (one 128-byte swizzled
// box) in shared memory and hands it to the TMA (cp.async.bulk.tensor store): full 128-byte lines leave the
// SM instead of 16-byte pieces of 32 different rows per store instruction.  Rows beyond M inside the last
// tile are written too (finite values computed from zero padded inputs); rows beyond the tensor are clipped.
struct EpiBiasActBf16 {
  static constexpr bool kTmaStore = true;
  struct Params {
    const float* bias;
    int relu;
  };
  template <int BN, class F>
  __device__ static void run(const Params& p, uint32_t taddr, int64_t row, int col0, int n_blk, int64_t M, F release, EpiShared& es) {
    const int lane = threadIdx.x & 31;
#pragma unroll 1
    for (int c = 0; c < BN; c += 64) {
      uint32_t ra[32], rb[32];
      tmem_ld32(taddr + c, ra);
      tmem_ld32(taddr + c + 32, rb);
      uint8_t* buf = es.stage + (es.chunk & 1u) * (kStoreStage / 2);
      if (es.chunk >= 2) {          // the box staged two chunks ago must have left shared memory
        if (lane == 0) bulk_wait_read<1>();
        __syncwarp();
      }
      tmem_ld_wait();
      if (c + 64 >= BN) release();
      const float4* b4 = reinterpret_cast<const float4*>(p.bias + col0 + c);
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        float v[8];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const float4 b = __ldg(b4 + q * 2 + h);
          const uint32_t* r = (q < 4 ? ra : rb) + (q & 3) * 8 + h * 4;
          v[h * 4 + 0] = __uint_as_float(r[0]) + b.x;
          v[h * 4 + 1] = __uint_as_float(r[1]) + b.y;
          v[h * 4 + 2] = __uint_as_float(r[2]) + b.z;
          v[h * 4 + 3] = __uint_as_float(r[3]) + b.w;
        }
        if (p.relu) {
#pragma unroll
          for (int i = 0; i < 8; ++i) v[i] = fmaxf(v[i], 0.f);
        }
        // 128-byte swizzle: 16-byte chunk q of row `lane` lives at chunk position q ^ (lane & 7)
        *reinterpret_cast<uint4*>(buf + lane * 128 + ((q ^ (lane & 7)) << 4)) =
            make_uint4(pack_bf16(v[0], v[1]), pack_bf16(v[2], v[3]), pack_bf16(v[4], v[5]), pack_bf16(v[6], v[7]));
      }
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) {
        tma_store_2d(es.tmC, buf, col0 + c, (int)(row - lane));
        bulk_commit();
      }
      ++es.chunk;
    }
  }
};

// partial[m][n_blk] = sum_n relu(acc + bias[n]) * w_last[n] over this tile's columns (fp32).
// The last Linear(N -> 1) of S3 folded into the epilogue of the layer before it; a tiny kernel adds
// the n_tiles partials in fixed order, so the result is deterministic.
struct EpiReluDot {
  static constexpr bool kTmaStore = false;
  struct Params {
    const float* bias;
    const float* w_last;
    float* partial;
    int n_tiles;
  };
  template <int BN, class F>
  __device__ static void run(const Params& p, uint32_t taddr, int64_t row, int col0, int n_blk, int64_t M, F release, EpiShared&) {
    float s = 0.f;
#pragma unroll 1
    for (int c = 0; c < BN; c += 32) {
      uint32_t r[32];
      tmem_ld32(taddr + c, r);
      tmem_ld_wait();
      if (c + 32 >= BN) release();
      const float4* b4 = reinterpret_cast<const float4*>(p.bias + col0 + c);
      const float4* w4 = reinterpret_cast<const float4*>(p.w_last + col0 + c);
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        const float4 b = __ldg(b4 + q), w = __ldg(w4 + q);
        s = fmaf(fmaxf(__uint_as_float(r[q * 4 + 0]) + b.x, 0.f), w.x, s);
        s = fmaf(fmaxf(__uint_as_float(r[q * 4 + 1]) + b.y, 0.f), w.y, s);
        s = fmaf(fmaxf(__uint_as_float(r[q * 4 + 2]) + b.z, 0.f), w.z, s);
        s = fmaf(fmaxf(__uint_as_float(r[q * 4 + 3]) + b.w, 0.f), w.w, s);
      }
    }
    if (row < M) p.partial[row * p.n_tiles + n_blk] = s;
  }
};

// out[m][0..n_valid) = acc + bias as fp32 (narrow output layer, BN = 16).
struct EpiBiasF32Narrow {
  static constexpr bool kTmaStore = false;
  struct Params {
    const float* bias;
    float* out;
    int ldo;
    int n_valid;
  };
  template <int BN, class F>
  __device__ static void run(const Params& p, uint32_t taddr, int64_t row, int col0, int n_blk, int64_t M, F release, EpiShared&) {
    static_assert(BN == 16, "narrow epilogue is for BN = 16");
    uint32_t r[16];
    tmem_ld16(taddr, r);
    tmem_ld_wait();
    release();
    if (row < M) {
#pragma unroll
      for (int i = 0; i < 16; ++i)
        if (col0 + i < p.n_valid) p.out[row * p.ldo + col0 + i] = __uint_as_float(r[i]) + p.bias[col0 + i];
    }
  }
};

// out[m][n] = acc as fp32 (the per-node halves of a split first layer, no bias).
struct EpiStoreF32 {
  static constexpr bool kTmaStore = false;
  struct Params {
    float* out;
    int ldo;
  };
  template <int BN, class F>
  __device__ static void run(const Params& p, uint32_t taddr, int64_t row, int col0, int n_blk, int64_t M, F release, EpiShared&) {
#pragma unroll 1
    for (int c = 0; c < BN; c += 32) {
      uint32_t r[32];
      tmem_ld32(taddr + c, r);
      tmem_ld_wait();
      if (c + 32 >= BN) release();
      if (row < M) {
        uint4* dst = reinterpret_cast<uint4*>(p.out + row * p.ldo + col0 + c);
#pragma unroll
        for (int q = 0; q < 8; ++q) dst[q] = make_uint4(r[q * 4], r[q * 4 + 1], r[q * 4 + 2], r[q * 4 + 3]);
      }
    }
  }
};

// Full-row epilogue of the GNN layers (BN == H, one tile column):
//   v = acc + bias (+ PA[src[m]] + PB[dst[m]]);  v = ReLU(LayerNorm(v)) or ReLU(v);
//   score mode:  score[m] = sigmoid(dot(v, w_out) + b_out)
//   else:        out[m] = (res ? res[m] : 0) + v   as bf16   (out may alias res)
struct EpiRowLn {
  static constexpr bool kTmaStore = false;
  struct Params {
    const float* bias;
    const float* pab;        // fp32 [nodes][2*BN]: columns [0,BN) belong to src, [BN,2BN) to dst; may be null
    const int32_t* src;
    const int32_t* dst;
    int use_ln;
    const __nv_bfloat16* res;
    int ldr;
    __nv_bfloat16* out;
    int ldo;
    const float* w_out;      // score mode when non-null
    float b_out;
    float* score;
  };
  template <int BN, class F>
  __device__ static void run(const Params& p, uint32_t taddr, int64_t row, int col0, int n_blk, int64_t M, F release, EpiShared&) {
    float v[BN];
#pragma unroll
    for (int c = 0; c < BN; c += 32) {
      uint32_t r[32];
      tmem_ld32(taddr + c, r);
      tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 32; ++i) v[c + i] = __uint_as_float(r[i]);
    }
    release();
    if (row >= M) return;
#pragma unroll
    for (int c = 0; c < BN; c += 4) {
      const float4 b = __ldg(reinterpret_cast<const float4*>(p.bias + c));
      v[c] += b.x; v[c + 1] += b.y; v[c + 2] += b.z; v[c + 3] += b.w;
    }
    if (p.pab) {
      const float4* ga = reinterpret_cast<const float4*>(p.pab + (int64_t)p.src[row] * (2 * BN));
      const float4* gb = reinterpret_cast<const float4*>(p.pab + (int64_t)p.dst[row] * (2 * BN) + BN);
#pragma unroll
      for (int c = 0; c < BN; c += 4) {
        const float4 a = __ldg(ga + c / 4), b = __ldg(gb + c / 4);
        v[c] += a.x + b.x; v[c + 1] += a.y + b.y; v[c + 2] += a.z + b.z; v[c + 3] += a.w + b.w;
      }
    }
    float mean = 0.f, rstd = 1.f;
    if (p.use_ln) {
      float s = 0.f;
#pragma unroll
      for (int c = 0; c < BN; ++c) s += v[c];
      mean = s * (1.f / BN);
      float q = 0.f;
#pragma unroll
      for (int c = 0; c < BN; ++c) { const float d = v[c] - mean; q = fmaf(d, d, q); }
      rstd = rsqrtf(q * (1.f / BN) + 1e-5f);
    }
#pragma unroll
    for (int c = 0; c < BN; ++c) v[c] = fmaxf((v[c] - mean) * rstd, 0.f);
    if (p.w_out) {
      float s = p.b_out;
#pragma unroll
      for (int c = 0; c < BN; c += 4) {
        const float4 w = __ldg(reinterpret_cast<const float4*>(p.w_out + c));
        s = fmaf(v[c], w.x, s); s = fmaf(v[c + 1], w.y, s); s = fmaf(v[c + 2], w.z, s); s = fmaf(v[c + 3], w.w, s);
      }
      p.score[row] = fast_sigmoid(s);
      return;
    }
    if (p.res) {
      const uint4* rp = reinterpret_cast<const uint4*>(p.res + row * p.ldr);
#pragma unroll
      for (int c = 0; c < BN; c += 8) {
        const uint4 u = rp[c / 8];
        const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&u);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          v[c + 2 * i] += __low2float(h[i]);
          v[c + 2 * i + 1] += __high2float(h[i]);
        }
      }
    }
    uint4* op = reinterpret_cast<uint4*>(p.out + row * p.ldo);
#pragma unroll
    for (int c = 0; c < BN; c += 8)
      op[c / 8] = make_uint4(pack_bf16(v[c], v[c + 1]), pack_bf16(v[c + 2], v[c + 3]), pack_bf16(v[c + 4], v[c + 5]),
                             pack_bf16(v[c + 6], v[c + 7]));
  }
};

}  // namespace tc
}  // namespace trk

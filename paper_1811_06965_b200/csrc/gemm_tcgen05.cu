// gemm_tcgen05.cu - bf16 GEMM on the 5th-generation tensor cores of sm_100a.
//
//   C[M,N] = epilogue( op(A)[M,K] * op(B)[K,N] ),   fp32 accumulation in TMEM.
//
// Design:
//   * CTA pairs (cta_group::2): the two CTAs on the two SMs of a TPC compute one 256 x BN output
//     tile.  Each CTA stages its own 128 rows of A and HALF of the B tile (BN/2 columns); the
//     leader's tcgen05.mma.cta_group::2 reads both halves of B and writes rows [0,128) of the tile
//     into its own TMEM and rows [128,256) into the peer's.  Per SM that is (128 + BN/2) x 64 x 2 B
//     of L2->shared traffic per 128 x BN x 64 MACs, 1.5x less than a 1-CTA 128 x 256 tile;
//   * persistent pairs (one per TPC), static tile schedule, K-blocks of 64 elements, a 5-stage
//     TMA -> shared-memory ring guarded by mbarriers; TMA of both CTAs completes on the LEADER's
//     "full" barrier, tcgen05.commit multicasts "stage free" / "accumulator ready" to both CTAs,
//     both CTAs' epilogue warps arrive on the leader's "accumulator drained" barrier;
//   * warp-specialised: warp 0 = TMA producer (one lane), warp 1 = tcgen05.mma issuer (one lane of
//     the leader), warp 2 = TMEM allocator, warps 4-7 = epilogue (one TMEM lane quadrant each);
//   * two TMEM accumulator stages (2 x BN columns): the epilogue of tile i overlaps the main loop
//     of tile i+1;
//   * all four operand layouts through the shared-memory descriptors: a K-major operand is one TMA
//     box [rows x 64] per stage (128-byte swizzle, 8-row atoms 1024 B apart), an MN-major operand
//     is [64 k x 64 mn] boxes, so forward (NN), dgrad (NT) and wgrad (TN) read the tensors where
//     they are - no transposed copies in HBM;
//   * epilogue: TMEM -> registers (+bias from shared memory, ReLU, bit-packed ReLU mask in/out,
//     +fp32 residual) -> 128-byte-swizzled shared staging -> TMA store; fp32 accumulation across
//     micro-batches (wgrad) is a TMA reduce-add (cp.reduce.async.bulk.tensor .add), so the
//     gradient tile is never read into registers.  All global writes of C are full-line TMA
//     transactions; TMA clips ragged edges.
// Roofline: bf16 tensor pipe (wgrad with fp32 accumulate sits near the HBM ridge).
#include <cuda.h>
#include <stdlib.h>

#include <mutex>
#include <unordered_map>

#include "common.cuh"
#include "tcgen05.cuh"

namespace gp {

namespace tc {

constexpr int BK = 64;
constexpr int NUM_THREADS = 384;
constexpr int EPI_WARP0 = 4;
constexpr int NUM_EPI_THREADS = 256;             // 8 epilogue warps

struct Params {
  int M, N, K;
  int a_mn_major, b_mn_major;   // 1: operand is MN-major in global memory (transA / !transB)
  const float *bias;
  const float *resid;           // fp32 [M, ldr]
  int64_t ldr;
  uint32_t *maskbits;           // EPI_MASK: read, EPI_BITS_OUT: written; [M, ldmask] words
  int64_t ldmask;
  int flags;
  int tiles_m, tiles_n;
  float *colpart;               // EPI_COLSUM: fp32 [ceil(M/128), N] per-128-row column sums
  // split-K (few output tiles, long K): `splits` work units per tile, each a contiguous range of
  // kb_per_split K-blocks.  The first splits-1 CTAs to finish a (tile, rank) write their raw fp32
  // accumulators to ws_part; the last one adds them to its own IN SPLIT ORDER (bitwise
  // deterministic, whoever is last) and runs the epilogue.  Nobody waits on a CTA that is not
  // already running.  ws_cnt: 2 self-resetting counters per (tile, rank).
  int splits, kb_per_split;
  float *ws_part;               // [tile][split][rank][128][BN] fp32
  unsigned int *ws_cnt;         // [tile][rank][2]: arrivals, partials ready
#if GP_PROBES
  unsigned long long *tl;       // optional timeline probe: 8 globaltimer stamps per CTA (gemm_tc_set_timeline)
  int dbg;                      // GPIPE_GEMM_DBG: 1 = epilogue only drains TMEM, 2 = no TMA loads, 4 = half of B's rows loaded (garbage results)
#endif
};
#if GP_PROBES
#define GP_DBG(p, bit) (((p).dbg & (bit)) != 0)
#else
#define GP_DBG(p, bit) false
#endif

#if GP_PROBES
__device__ __forceinline__ void tl_stamp(const Params &p, int slot) {
  if (p.tl) {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    p.tl[(size_t)blockIdx.x * 32 + slot] = t;
  }
}
// fine-grained: SM clock stamps of the first tile's first four chunks (epilogue warp 0, lane 0)
__device__ __forceinline__ void tl_clock(const Params &p, bool on, int c, int which) {
  if (p.tl && on && c < 6) p.tl[(size_t)blockIdx.x * 32 + 8 + c * 4 + which] = (unsigned long long)clock64();
}
#else
__device__ __forceinline__ void tl_stamp(const Params &, int) {}
__device__ __forceinline__ void tl_clock(const Params &, bool, int, int) {}
#endif

// Dynamic shared memory: operand ring (5 stages of 32 KB), epilogue staging (one [32 rows x 128 B] buffer per
// epilogue warp), bias (2 x BN floats, only with EPI_BIAS), column-sum exchange (4 x BN floats, only with
// EPI_COLSUM), 1 KB alignment slack.  An instantiation whose flags are compile-time constants carries only the
// auxiliary buffers it uses.  STG = 2 (a second staging buffer per warp, which fits for the flag sets without
// column sums) was measured in the config-5 step against STG = 1 on one box: 1500-1504 ms vs 1492 ms - the extra
// shared-memory footprint buys nothing, the epilogue is not waiting on its staging buffer.
template <int BN, int F> struct PairCfg {
  static constexpr int BNH = BN / 2;
  static constexpr uint32_t A_BYTES = 128 * BK * 2, B_BYTES = BNH * BK * 2, STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int STAGES = BN == 256 ? 5 : 4;   // BN 512 with 3 stages + a second staging buffer per warp: +8 ms per config-5 step
  static constexpr int STG = 1;
  static constexpr uint32_t BIAS_BYTES = (BN == 256 && (F < 0 || (F & EPI_BIAS))) ? 2 * BN * 4 : 0;   // BN 512: bias from L1
  static constexpr uint32_t COLBUF_BYTES = (F < 0 || (F & EPI_COLSUM)) ? 4 * BN * 4 : 0;
  static constexpr uint32_t AUX_BYTES = BIAS_BYTES + COLBUF_BYTES;
  static constexpr uint32_t LIMIT = 227 * 1024 - 512;                // opt-in maximum minus the static barriers etc.
  static constexpr uint32_t STAGING_BYTES = 8 * STG * 4096;
  static constexpr uint32_t TMEM_COLS = 512;
  static constexpr int NBLK = BN / 256;                               // 256-column accumulator blocks of one tile
  static constexpr int NACC = 2 / NBLK;                               // accumulator stages in the 512 TMEM columns
  static constexpr size_t SMEM = (size_t)STAGES * STAGE_BYTES + STAGING_BYTES + AUX_BYTES + 1024;
  static_assert(SMEM <= LIMIT, "shared-memory budget");
};

// Column sums over a warp's 32 rows: transpose-reduce across lanes (31 shuffles); afterwards
// v[0] of lane j is the sum of column col0 + j.
__device__ __forceinline__ void warp_colsum32(float (&v)[32], const int lane) {
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) {
    const bool hi = (lane & off) != 0;
#pragma unroll
    for (int i = 0; i < off; ++i) {
      float send = hi ? v[i] : v[i + off];
      float keep = hi ? v[i + off] : v[i];
      v[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
    }
  }
}

// ------------------------------------------------------------------------------------------
// the kernel
// ------------------------------------------------------------------------------------------
// F >= 0: the epilogue flags are this compile-time constant (compact straight-line epilogue: the generic one is
// instruction-fetch bound); F < 0: p.flags at run time.  SPLITK: the launch may be split along K (p.splits).
template <int BN, int F, bool SPLITK>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NUM_THREADS, 1)
gemm_tcgen05_pair_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b,
                         const __grid_constant__ CUtensorMap map_c, const Params p) {
  using Cfg = PairCfg<BN, F>;
  constexpr int NST = Cfg::STAGES, BNH = Cfg::BNH, STG = Cfg::STG;
  constexpr uint32_t A_BYTES = Cfg::A_BYTES, STAGE_BYTES = Cfg::STAGE_BYTES;
  static_assert(BN == 256 || (BN == 512 && F >= 0 && !SPLITK && !(F & EPI_COLSUM)),
                "256 x 512: compile-time flags, unsplit, no column sums (shared-memory budget)");
  constexpr int NBLK = Cfg::NBLK, NACC = Cfg::NACC;
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * NST + 4];
  __shared__ uint32_t tmem_base_smem;
  __shared__ int split_last_s;

  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t staging_base = smem_base + NST * STAGE_BYTES;
  float *bias_s = reinterpret_cast<float *>(smem_raw + (staging_base - smem_u32(smem_raw)) + Cfg::STAGING_BYTES);  // [2][BN]
  float *colbuf = bias_s + Cfg::BIAS_BYTES / 4;                                                                   // [4][BN]
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int pair = blockIdx.x >> 1, num_pairs = gridDim.x >> 1;
  const uint32_t bar0 = smem_u32(bars);
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (NST + s); };
  auto tfull_bar = [&](int s) { return bar0 + 8u * (2 * NST + s); };
  auto tempty_bar = [&](int s) { return bar0 + 8u * (2 * NST + 2 + s); };

  if (threadIdx.x == 0) tl_stamp(p, 0);                // kernel entry
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&map_a);
    tma_prefetch_desc(&map_b);
    tma_prefetch_desc(&map_c);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < NST; ++s) {
      mbar_init(full_bar(s), 1);                   // leader's: its producer's arrive.expect_tx (both CTAs' bytes)
      mbar_init(empty_bar(s), 1);                  // one multicast tcgen05.commit
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(tfull_bar(s), 1);
      mbar_init(tempty_bar(s), 16);                // leader's: 8 epilogue warps of each CTA
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // Both CTAs of the pair are running (and their barriers initialised) before the pair-wide TMEM
  // allocation is attempted, and - see the teardown - neither SM is handed to another kernel before
  // BOTH CTAs have returned their columns: a pair dealloc that lands after the peer's SM already hosts
  // a CTA of another TMEM-using kernel wedges that SM's allocator (observed as a later kernel stuck
  // in its prologue).
  cluster_sync_all();
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_smem)),
                 "n"(Cfg::TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;");
  }
  tcgen05_fence_before();
  cluster_sync_all();
  tcgen05_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  if (threadIdx.x == 0) tl_stamp(p, 1);                // prologue done

  const int flags = F >= 0 ? F : p.flags;
  const int splits = SPLITK ? p.splits : 1;
  const int num_units = p.tiles_m * p.tiles_n * splits;       // work units: (tile, split), splits adjacent
  const int num_kb = (p.K + BK - 1) / BK;

  if (warp == 0) {
    // ===================== TMA producer (both CTAs) =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int u = pair; u < num_units; u += num_pairs) {
        const int t = u / splits, sp = u - t * splits;
        const int m0 = (t % p.tiles_m) * 256 + (int)rank * 128, n0 = (t / p.tiles_m) * BN + (int)rank * BNH;
        const int kb0 = sp * p.kb_per_split, kb1 = min(num_kb, kb0 + p.kb_per_split);
        for (int kb = kb0; kb < kb1; ++kb) {
          mbar_wait(empty_bar(stage), phase ^ 1, 0x11);
          const uint32_t sa = smem_base + stage * STAGE_BYTES, sb = sa + A_BYTES;
          if (GP_DBG(p, 2)) {
            if (rank == 0) mbar_arrive(full_bar(stage));
            if (++stage == NST) { stage = 0; phase ^= 1; }
            continue;
          }
          const bool half_b = GP_DBG(p, 4);            // probe: deliver only half of the B rows (25 % fewer bytes)
          if (rank == 0) mbar_expect_tx(full_bar(stage), half_b ? 2 * (A_BYTES + Cfg::B_BYTES / 2) : 2 * STAGE_BYTES);
          const uint32_t fb = mapa_shared(full_bar(stage), 0);
          const int k0 = kb * BK;
          if (!p.a_mn_major) {
            tma_load_2d_pair(sa, &map_a, fb, k0, m0);                          // box [128 rows x 64 k]
          } else {
#pragma unroll
            for (int c = 0; c < 2; ++c)                                        // boxes [64 k x 64 m]
              tma_load_2d_pair(sa + c * (BK * 128), &map_a, fb, m0 + c * 64, k0);
          }
          if (!p.b_mn_major) {
            tma_load_2d_pair(sb, &map_b, fb, k0, n0);                          // box [BN/2 rows x 64 k]
          } else {
#pragma unroll
            for (int c = 0; c < (half_b ? BNH / 128 : BNH / 64); ++c)          // boxes [64 k x 64 n]
              tma_load_2d_pair(sb + c * (BK * 128), &map_b, fb, n0 + c * 64, k0);
          }
          if (++stage == NST) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA only) =====================
    if (lane == 0 && rank == 0) {
      // instruction descriptor: D fp32, A/B bf16, majorness, N >> 3, M >> 4 (M = 256 over the pair)
      const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)p.a_mn_major << 15) |
                             ((uint32_t)p.b_mn_major << 16) | ((uint32_t)(256 >> 3) << 17) |
                             ((uint32_t)(256 >> 4) << 24);
      // K-major: 8-row atoms 1024 B apart, +32 B per 16 k.  MN-major: 64-element chunks BK*128 B
      // apart (LBO), 8-k groups 1024 B apart (SBO), +2048 B per 16 k.
      const uint32_t a_lbo = p.a_mn_major ? BK * 128 : 16, a_sbo = 1024, a_kstep = p.a_mn_major ? 2048 : 32;
      const uint32_t b_lbo = p.b_mn_major ? BK * 128 : 16, b_sbo = 1024, b_kstep = p.b_mn_major ? 2048 : 32;
      int stage = 0;
      uint32_t phase = 0;
      int as = 0;
      uint32_t aphase = 0;
      auto issue = [&](uint32_t d_tmem, int st, uint32_t b_off, bool fresh) {     // one K-block into one accumulator block
        const uint32_t sa = smem_base + st * STAGE_BYTES, sb = sa + A_BYTES + b_off;
#pragma unroll
        for (int k = 0; k < BK / 16; ++k) {
          const uint64_t ad = make_smem_desc(sa + k * a_kstep, a_lbo, a_sbo);
          const uint64_t bd = make_smem_desc(sb + k * b_kstep, b_lbo, b_sbo);
          umma_bf16_pair(d_tmem, ad, bd, idesc, (!fresh || k) ? 1u : 0u);
        }
      };
      for (int u = pair; u < num_units; u += num_pairs) {
        const int sp = u % splits;
        const int kb0 = sp * p.kb_per_split, kb1 = min(num_kb, kb0 + p.kb_per_split);
        if constexpr (NBLK == 1) {
          mbar_wait(tempty_bar(as), aphase ^ 1, 0x12);       // both CTAs' epilogues have drained this accumulator
          tcgen05_fence_after();
          const uint32_t d_tmem = tmem_base + (uint32_t)(as * BN);
          for (int kb = kb0; kb < kb1; ++kb) {
            mbar_wait(full_bar(stage), phase, 0x13);
            tcgen05_fence_after();
            if (u == pair && kb == kb0) tl_stamp(p, 2);  // first operands landed
            issue(d_tmem, stage, 0u, kb == kb0);
            tcgen05_commit_pair(empty_bar(stage), 3);  // frees this stage in both CTAs
            if (++stage == NST) { stage = 0; phase ^= 1; }
          }
          tcgen05_commit_pair(tfull_bar(as), 3);       // accumulator complete -> both epilogues
          if (++as == 2) { as = 0; aphase ^= 1; }
        } else {
          // 256 x 512: one accumulator of two 256-column blocks (all 512 TMEM columns), block b = the tile columns
          // [b*128, b*128+128) of each CTA's 256 B rows (16 KB into its B stage).  The epilogue of the previous tile
          // drains block 0 first: the first `pre` K-blocks (what the ring holds) go into block 0 while block 1 is
          // still being drained, then into block 1; after that both blocks per K-block.
          const int nkb = kb1 - kb0, pre = nkb < NST ? nkb : NST;
          mbar_wait(tempty_bar(0), aphase ^ 1, 0x12);
          tcgen05_fence_after();
          {
            int st = stage;
            uint32_t ph = phase;
            for (int i = 0; i < pre; ++i) {
              mbar_wait(full_bar(st), ph, 0x13);
              tcgen05_fence_after();
              if (u == pair && i == 0) tl_stamp(p, 2);
              issue(tmem_base, st, 0u, i == 0);
              if (++st == NST) { st = 0; ph ^= 1; }
            }
          }
          mbar_wait(tempty_bar(1), aphase ^ 1, 0x15);
          tcgen05_fence_after();
          for (int i = 0; i < pre; ++i) {
            issue(tmem_base + 256u, stage, 16384u, i == 0);
            tcgen05_commit_pair(empty_bar(stage), 3);
            if (++stage == NST) { stage = 0; phase ^= 1; }
          }
          for (int i = pre; i < nkb; ++i) {
            mbar_wait(full_bar(stage), phase, 0x13);
            tcgen05_fence_after();
            issue(tmem_base, stage, 0u, false);
            issue(tmem_base + 256u, stage, 16384u, false);
            tcgen05_commit_pair(empty_bar(stage), 3);
            if (++stage == NST) { stage = 0; phase ^= 1; }
          }
          tcgen05_commit_pair(tfull_bar(0), 3);
          aphase ^= 1;
        }
      }
      tl_stamp(p, 3);                                  // every MMA issued
    }
  } else if (warp >= EPI_WARP0) {
    // ===================== epilogue (both CTAs): own 128 rows of the tile =====================
    // 8 warps: warp ew reads TMEM lane quadrant ew & 3 (rows) and column half ew >> 2 (4 chunks of 32
    // columns).  The tcgen05.ld of chunk c+1 is in flight while chunk c is converted and staged.
    const int ew = warp - EPI_WARP0;
    const int quad = ew & 3, chalf = ew >> 2;
    const int et = threadIdx.x - EPI_WARP0 * 32;     // 0..255 within the epilogue warps
    const bool out_f32 = (flags & (EPI_OUT_F32 | EPI_ACCUM)) != 0;
    const uint32_t stg0 = staging_base + (uint32_t)ew * (uint32_t)(STG * 4096);
    const uint32_t tempty_leader0 = mapa_shared(tempty_bar(0), 0), tempty_leader1 = mapa_shared(tempty_bar(1), 0);
    const uint32_t swz = (uint32_t)(lane & 7);
    int as = 0, it = 0, sbuf = 0;
    uint32_t aphase = 0;
    for (int u = pair; u < num_units; u += num_pairs, ++it) {
      const int t = u / splits, sp = u - t * splits;
      const int m0 = (t % p.tiles_m) * 256 + (int)rank * 128, n0 = (t / p.tiles_m) * BN;
      const int row0 = m0 + quad * 32, row = row0 + lane;
      const bool row_ok = row < p.M;
      float *bs = bias_s + (it & 1) * BN;
      if constexpr (BN == 256) {
        if (flags & EPI_BIAS) {
          for (int i = et; i < BN; i += NUM_EPI_THREADS) bs[i] = (n0 + i < p.N) ? __ldg(p.bias + n0 + i) : 0.f;
        }
      }
      // this row's ReLU-pattern words for this warp's chunks (16 bytes per 256-column block), fetched before the wait
      uint4 mbq[NBLK];
#pragma unroll
      for (int jb = 0; jb < NBLK; ++jb) {
        mbq[jb] = make_uint4(0u, 0u, 0u, 0u);
        if ((flags & EPI_MASK) && row_ok) {
          const uint32_t *mp = p.maskbits + (int64_t)row * p.ldmask + (n0 >> 5) + (chalf * NBLK + jb) * 4;
          if (n0 + BN <= p.N && (p.ldmask & 3) == 0) {
            mbq[jb] = __ldg(reinterpret_cast<const uint4 *>(mp));
          } else {
            const int cb = n0 + (chalf * NBLK + jb) * 128;
            if (cb < p.N) mbq[jb].x = __ldg(mp);
            if (cb + 32 < p.N) mbq[jb].y = __ldg(mp + 1);
            if (cb + 64 < p.N) mbq[jb].z = __ldg(mp + 2);
            if (cb + 96 < p.N) mbq[jb].w = __ldg(mp + 3);
          }
        }
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");       // bias_s visible; colbuf of the previous tile consumed
      mbar_wait(tfull_bar(as), aphase, 0x14);
      tcgen05_fence_after();
      if (it == 0 && et == 0) tl_stamp(p, 4);          // first accumulator complete
      const uint32_t t_row0 = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(as * 256 + chalf * 128);
      uint32_t rn[32];
      tmem_ld32(t_row0, rn);                             // first chunk in flight during the split-K handshake
      // ---- split-K: am I the last of this (tile, rank)'s splits to finish? ----
      bool write_partial = false;
      if constexpr (SPLITK) if (splits > 1) {
        unsigned int *cnt = p.ws_cnt + ((size_t)t * 2 + rank) * 2;
        if (et == 0) {
          const unsigned int arrived = atomicAdd(cnt, 1u);
          if (arrived == (unsigned int)splits - 1) {          // last: wait for the partials already being written
            while (atomicAdd(cnt + 1, 0u) < (unsigned int)splits - 1) __nanosleep(64);
            cnt[0] = 0u;                                        // self-reset for the next launch on this stream
            cnt[1] = 0u;
            __threadfence();
            split_last_s = 1;
          } else {
            split_last_s = 0;
          }
        }
        asm volatile("bar.sync 2, 256;" ::: "memory");
        write_partial = split_last_s == 0;
      }
      // partials: [tile][split][rank][chunk][row 128][32 floats] - the 32 x 128 B a warp writes per chunk are contiguous
      float *part_row = p.ws_part + (((size_t)t * splits) * 2 + rank) * (size_t)(128 * BN) +
                        (size_t)(quad * 32 + lane) * 32;          // split 0 of this (tile, rank), chunk 0, this lane's row
      const size_t part_split_stride = (size_t)2 * 128 * BN;
      // One 256-column accumulator block per outer iteration (256 x 512 tiles have two; TMEM block jb holds the
      // tile columns jb*128 + [0, 128) of each CTA's half, so this warp's 4 * NBLK chunks are consecutive tile columns).
#pragma unroll 1
      for (int jb = 0; jb < NBLK; ++jb) {
      const uint32_t t_row = t_row0 + (uint32_t)(jb * 256);
      const uint32_t mb0 = jb ? mbq[NBLK - 1].x : mbq[0].x, mb1 = jb ? mbq[NBLK - 1].y : mbq[0].y,
                     mb2 = jb ? mbq[NBLK - 1].z : mbq[0].z, mb3 = jb ? mbq[NBLK - 1].w : mbq[0].w;
      uint32_t wb0 = 0u, wb1 = 0u, wb2 = 0u, wb3 = 0u;     // EPI_BITS_OUT words of this row
      // one 32-column chunk per iteration; NOT unrolled in the run-time-flag kernel: the epilogue has to stay
      // resident in the instruction cache next to the other warp roles
#pragma unroll (F >= 0 ? 4 : 1)
      for (int cl = 0; cl < 4; ++cl) {
        const int c = (chalf * NBLK + jb) * 4 + cl;
        const int col0 = n0 + c * 32;
        const bool col_ok = col0 < p.N;                      // uniform over the warp
        float4 rr[8];
        if ((flags & EPI_RESID) && row_ok && col_ok) {
          const float *rp = p.resid + (int64_t)row * p.ldr + col0;
          if (col0 + 32 <= p.N) {
#pragma unroll
            for (int j = 0; j < 8; ++j) rr[j] = *reinterpret_cast<const float4 *>(rp + 4 * j);
          } else {
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              rr[j].x = col0 + 4 * j + 0 < p.N ? rp[4 * j + 0] : 0.f;
              rr[j].y = col0 + 4 * j + 1 < p.N ? rp[4 * j + 1] : 0.f;
              rr[j].z = col0 + 4 * j + 2 < p.N ? rp[4 * j + 2] : 0.f;
              rr[j].w = col0 + 4 * j + 3 < p.N ? rp[4 * j + 3] : 0.f;
            }
          }
        } else {
#pragma unroll
          for (int j = 0; j < 8; ++j) rr[j] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(rn[j]);
        if (cl < 3) tmem_ld32(t_row + (cl + 1) * 32, rn);    // next chunk: overlaps this chunk's arithmetic and staging
        else if (jb + 1 < NBLK) tmem_ld32(t_row + 256, rn);
        const bool tlon = it == 0 && et == 0;
        tl_clock(p, tlon, cl, 0);
        if (!col_ok) continue;
        if (GP_DBG(p, 1)) continue;
        if (splits > 1) {
          if (write_partial) {                               // raw accumulators -> workspace; no epilogue
            float4 *dst = reinterpret_cast<float4 *>(part_row + sp * part_split_stride + (size_t)c * (128 * 32));
#pragma unroll
            for (int j = 0; j < 8; ++j) __stcg(dst + j, make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]));
            continue;
          }
          // fixed summation order: split 0, 1, ... with the own accumulators at position sp
          float acc[32];
          bool first = true;
          for (int s2 = 0; s2 < splits; ++s2) {
            if (s2 == sp) {
              if (first) {
#pragma unroll
                for (int j = 0; j < 32; ++j) acc[j] = v[j];
              } else {
#pragma unroll
                for (int j = 0; j < 32; ++j) acc[j] += v[j];
              }
            } else {
              const float4 *src = reinterpret_cast<const float4 *>(part_row + s2 * part_split_stride + (size_t)c * (128 * 32));
#pragma unroll
              for (int j = 0; j < 8; ++j) {
                const float4 q4 = __ldcg(src + j);
                if (first) { acc[4 * j] = q4.x; acc[4 * j + 1] = q4.y; acc[4 * j + 2] = q4.z; acc[4 * j + 3] = q4.w; }
                else { acc[4 * j] += q4.x; acc[4 * j + 1] += q4.y; acc[4 * j + 2] += q4.z; acc[4 * j + 3] += q4.w; }
              }
            }
            first = false;
          }
#pragma unroll
          for (int j = 0; j < 32; ++j) v[j] = acc[j];
        }
        if (flags & EPI_BIAS) {
          if constexpr (BN == 256) {
#pragma unroll
            for (int j = 0; j < 32; j += 4) {
              float4 b = *reinterpret_cast<const float4 *>(bs + c * 32 + j);
              v[j] += b.x; v[j + 1] += b.y; v[j + 2] += b.z; v[j + 3] += b.w;
            }
          } else if (col0 + 32 <= p.N) {                     // warp-uniform 16-byte loads (the launcher checked alignment)
            const float4 *bp = reinterpret_cast<const float4 *>(p.bias + col0);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              const float4 b = __ldg(bp + j);
              v[4 * j] += b.x; v[4 * j + 1] += b.y; v[4 * j + 2] += b.z; v[4 * j + 3] += b.w;
            }
          } else {
#pragma unroll
            for (int j = 0; j < 32; ++j) v[j] += col0 + j < p.N ? __ldg(p.bias + col0 + j) : 0.f;
          }
        }
        if (flags & EPI_RELU) {
#pragma unroll
          for (int j = 0; j < 32; ++j) v[j] = fmaxf(v[j], 0.f);          // max(-0, +0) = +0
        }
        if ((flags & EPI_BITS_OUT) && (flags & EPI_RELU) && !out_f32) {
          // bit j = [v_j > 0]: after the ReLU v_j >= +0, so v_j > 0 <=> its bit pattern is a positive integer <=> the
          // top bit of (0 - pattern) is set; one subtract + one funnel shift per unit.  RNE to bf16 maps a positive
          // fp32 normal to a positive bf16, so this is also [stored h > 0].
          uint32_t w = 0;
#pragma unroll
          for (int j = 31; j >= 0; --j) w = __funnelshift_l(0u - __float_as_uint(v[j]), w, 1);
          wb0 = cl == 0 ? w : wb0; wb1 = cl == 1 ? w : wb1; wb2 = cl == 2 ? w : wb2; wb3 = cl == 3 ? w : wb3;
        }
        if (flags & EPI_MASK) {
          const uint32_t w01 = (cl & 1) ? mb1 : mb0, w23 = (cl & 1) ? mb3 : mb2;
          const uint32_t mw = (cl & 2) ? w23 : w01;
#pragma unroll
          for (int j = 0; j < 32; ++j) v[j] = ((mw >> j) & 1u) ? v[j] : 0.f;
        }
        if (flags & EPI_RESID) {
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            v[4 * j] += rr[j].x; v[4 * j + 1] += rr[j].y; v[4 * j + 2] += rr[j].z; v[4 * j + 3] += rr[j].w;
          }
        }
        // ---- registers -> swizzled staging -> TMA ----
        if (out_f32) {
          const uint32_t buf = stg0 + (uint32_t)sbuf * 4096u;
          if (lane == 0) bulk_wait_read<STG - 1>();          // the store that last used this buffer has read it
          __syncwarp();
#pragma unroll
          for (int q = 0; q < 8; ++q)
            st_shared_v4(buf + (uint32_t)lane * 128u + (((uint32_t)q ^ swz) << 4), __float_as_uint(v[4 * q]),
                         __float_as_uint(v[4 * q + 1]), __float_as_uint(v[4 * q + 2]), __float_as_uint(v[4 * q + 3]));
          tl_clock(p, tlon, cl, 1);
          fence_proxy_async_smem();
          __syncwarp();
          tl_clock(p, tlon, cl, 2);
          if (lane == 0) {
            if (flags & EPI_ACCUM) tma_reduce_add_2d(&map_c, buf, col0, row0);
            else tma_store_2d(&map_c, buf, col0, row0);
            bulk_commit();
          }
          if (STG > 1) sbuf ^= 1;
          tl_clock(p, tlon, cl, 3);
        } else {
          const uint32_t buf = stg0 + (uint32_t)sbuf * 4096u;
          const int half = cl & 1;
          if (!half) {
            if (lane == 0) bulk_wait_read<STG - 1>();
            __syncwarp();
          }
          uint32_t pk[16];
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            __nv_bfloat162 h = __floats2bfloat162_rn(v[2 * j], v[2 * j + 1]);
            pk[j] = *reinterpret_cast<uint32_t *>(&h);
            float2 f = __bfloat1622float2(h);               // the stored values (EPI_COLSUM, EPI_BITS_OUT)
            v[2 * j] = f.x;
            v[2 * j + 1] = f.y;
          }
#pragma unroll
          for (int q = 0; q < 4; ++q)
            st_shared_v4(buf + (uint32_t)lane * 128u + (((uint32_t)(half * 4 + q) ^ swz) << 4), pk[4 * q],
                         pk[4 * q + 1], pk[4 * q + 2], pk[4 * q + 3]);
          const bool flush = half || col0 + 32 >= p.N;
          tl_clock(p, tlon, cl, 1);
          if (flush) {
            fence_proxy_async_smem();
            __syncwarp();
            tl_clock(p, tlon, cl, 2);
            if (lane == 0) {
              tma_store_2d(&map_c, buf, col0 - half * 32, row0);      // columns past N are clipped
              bulk_commit();
            }
            if (STG > 1) sbuf ^= 1;
          }
          tl_clock(p, tlon, cl, 3);
        }
        if ((flags & EPI_BITS_OUT) && !((flags & EPI_RELU) && !out_f32)) {
          uint32_t w = 0;
#pragma unroll
          for (int j = 0; j < 32; ++j) w |= (v[j] > 0.f ? 1u : 0u) << j;
          wb0 = cl == 0 ? w : wb0; wb1 = cl == 1 ? w : wb1; wb2 = cl == 2 ? w : wb2; wb3 = cl == 3 ? w : wb3;
        }
        if (flags & EPI_COLSUM) {
          const bool ragged = col0 + 32 > p.N;
#pragma unroll
          for (int j = 0; j < 32; ++j) v[j] = (row_ok && !(ragged && col0 + j >= p.N)) ? v[j] : 0.f;
          warp_colsum32(v, lane);
          colbuf[quad * BN + c * 32 + lane] = v[0];
        }
      }
      // every TMEM read of this accumulator block has completed (tcgen05.wait::ld): release it
      tcgen05_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster_relaxed((NBLK == 1 ? as : jb) ? tempty_leader1 : tempty_leader0);
      if ((flags & EPI_BITS_OUT) && row_ok && !write_partial) {   // this row's four pattern words: one 16-byte store
        uint32_t *mp = p.maskbits + (int64_t)row * p.ldmask + (n0 >> 5) + (chalf * NBLK + jb) * 4;
        const int cb = n0 + (chalf * NBLK + jb) * 128;
        if (cb + 128 <= p.N && (p.ldmask & 3) == 0) {
          *reinterpret_cast<uint4 *>(mp) = make_uint4(wb0, wb1, wb2, wb3);
        } else {
          if (cb < p.N) mp[0] = wb0;
          if (cb + 32 < p.N) mp[1] = wb1;
          if (cb + 64 < p.N) mp[2] = wb2;
          if (cb + 96 < p.N) mp[3] = wb3;
        }
      }
      }                                                      // jb
      if (++as == NACC) { as = 0; aphase ^= 1; }
      if (write_partial) {                                   // publish: all 8 warps' partial rows, then one ready tick
        __threadfence();
        asm volatile("bar.sync 2, 256;" ::: "memory");
        if (et == 0) atomicAdd(p.ws_cnt + ((size_t)t * 2 + rank) * 2 + 1, 1u);
        continue;
      }
      if (flags & EPI_COLSUM) {
        asm volatile("bar.sync 2, 256;" ::: "memory");
        for (int cc = et; cc < BN; cc += NUM_EPI_THREADS) {
          float ssum = (colbuf[cc] + colbuf[BN + cc]) + (colbuf[2 * BN + cc] + colbuf[3 * BN + cc]);
          if (n0 + cc < p.N && m0 < p.M) p.colpart[(int64_t)(m0 >> 7) * p.N + n0 + cc] = ssum;
        }
      }
    }
    if (et == 0) tl_stamp(p, 5);                       // last chunk handed to the TMA
    if (lane == 0) bulk_wait_all();                    // staging must outlive the TMA reads; C complete at exit
    if (et == 0) tl_stamp(p, 6);                       // stores complete
  }

  tcgen05_fence_before();
  cluster_sync_all();                                  // the peer's smem / TMEM / barriers stay valid until both are done
  if (threadIdx.x == 0) tl_stamp(p, 7);                // both CTAs done
  if (warp == 2) {
    tcgen05_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(Cfg::TMEM_COLS));
  }
  cluster_sync_all();                                  // no CTA of the pair exits before both deallocations
}

// ------------------------------------------------------------------------------------------
// host side: tensor maps (driver entry point fetched through the runtime, no -lcuda) and launch
// ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  });
  return fn;
}

struct MapKey {
  const void *ptr;
  uint64_t inner, outer, ld;
  uint32_t box_inner, box_outer, esize;
  bool operator==(const MapKey &o) const {
    return ptr == o.ptr && inner == o.inner && outer == o.outer && ld == o.ld && box_inner == o.box_inner &&
           box_outer == o.box_outer && esize == o.esize;
  }
};
struct MapKeyHash {
  size_t operator()(const MapKey &k) const {
    size_t h = (size_t)k.ptr;
    auto mix = [&](uint64_t v) { h ^= v + 0x9e3779b97f4a7c15ull + (h << 6) + (h >> 2); };
    mix(k.inner); mix(k.outer); mix(k.ld); mix(k.box_inner); mix(k.box_outer); mix(k.esize);
    return h;
  }
};

// 2-D tensor [outer, inner] of bf16 (esize 2) or fp32 (esize 4) with row pitch ld elements; box
// [box_outer, box_inner], 128-byte swizzle.
static bool get_map(const void *ptr, uint32_t esize, uint64_t inner, uint64_t outer, uint64_t ld, uint32_t box_inner,
                    uint32_t box_outer, CUtensorMap *out) {
  static std::unordered_map<MapKey, CUtensorMap, MapKeyHash> cache;
  static std::mutex mu;
  MapKey key{ptr, inner, outer, ld, box_inner, box_outer, esize};
  std::lock_guard<std::mutex> lock(mu);
  auto it = cache.find(key);
  if (it != cache.end()) {
    *out = it->second;
    return true;
  }
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {inner, outer};
  cuuint64_t strides[1] = {ld * esize};
  cuuint32_t box[2] = {box_inner, box_outer};
  cuuint32_t estr[2] = {1, 1};
  CUtensorMap m;
  CUresult r = fn(&m, esize == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2,
                  const_cast<void *>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return false;
  if (cache.size() > 65536) cache.clear();
  cache.emplace(key, m);
  *out = m;
  return true;
}

// Split-K when the output has too few 256 x 256 tiles to occupy the CTA pairs (tiles <= pairs / 2) and K is so long
// that each split still runs a main loop of >= 192 K-blocks (12288 deep): only the dlogits W_out^T product (K = V)
// qualifies.  Measured, isolated (us, unsplit vs split): K = 2048 20.5 / 43.6 (run-time-flag kernel, round 1),
// K = 16384 85.8 / 68.0, K = 64000 296.6 / 207.1 - and in the step: with every [T_mb x 1024] output split (>= 32
// K-blocks per split, specialised kernels) config 2 ran 6 % slower (20.8 vs 19.6 ms) and config 5 5 % slower: a split
// launch takes twice the SMs for 0.8x the time, and the step is bound by SM-time, not by single-kernel latency.
// All units run in ONE wave; the first splits-1 CTAs of a (tile, rank) to finish leave raw fp32 accumulators in the
// workspace, the last one sums them in split order (bitwise deterministic, whoever is last).
constexpr int kSplitMinKb = 192;
static int splitk_factor(int tiles, int num_kb, int pairs) {
  int min_kb = kSplitMinKb;
#if GP_PROBES
  static const int off = getenv("GPIPE_NO_SPLITK") ? atoi(getenv("GPIPE_NO_SPLITK")) : 0;
  if (off) return 1;
  static const int mk = getenv("GPIPE_SPLITK_MINKB") ? atoi(getenv("GPIPE_SPLITK_MINKB")) : 0;
  if (mk > 0) min_kb = mk;
#endif
  if (tiles * 2 > pairs) return 1;
  int s = pairs / tiles;
  if (s > 4) s = 4;
  while (s > 1 && num_kb / s < min_kb) --s;
  return s;
}
static size_t splitk_cnt_bytes(int tiles) { return (((size_t)tiles * 2 * 2 * sizeof(unsigned int)) + 1023) & ~(size_t)1023; }

#if GP_PROBES
static unsigned long long *g_timeline = nullptr;
#endif

template <int BN, int F, bool SPLITK>
static cudaError_t launch_pair(const Ctx &c, const GemmArgs &a) {
  using Cfg = PairCfg<BN, F>;
  Params p{};
  p.M = a.M; p.N = a.N; p.K = a.K;
  p.a_mn_major = a.transA ? 1 : 0;
  p.b_mn_major = a.transB ? 0 : 1;
  p.bias = a.bias; p.resid = a.resid; p.ldr = a.ldc; p.maskbits = (uint32_t *)a.mask; p.ldmask = a.ldmask;
  p.flags = a.flags;
  p.colpart = a.colsum_scratch;
  p.tiles_m = (a.M + 255) / 256;
  p.tiles_n = (a.N + BN - 1) / BN;
  int pairs = c.sm_count / 2;
#if GP_PROBES
  {                                                  // experiment knob: run on fewer CTA pairs
    static const int lim = getenv("GPIPE_GEMM_PAIRS") ? atoi(getenv("GPIPE_GEMM_PAIRS")) : 0;
    if (lim > 0 && lim < pairs) pairs = lim;
  }
#endif
  const int num_kb = (a.K + BK - 1) / BK;
  p.splits = SPLITK ? splitk_factor(p.tiles_m * p.tiles_n, num_kb, pairs) : 1;
  if (p.splits > 1 && (!a.ws || a.ws_bytes < gemm_splitk_ws_bytes(a.M, a.N, a.K, c.sm_count))) p.splits = 1;
  p.kb_per_split = (num_kb + p.splits - 1) / p.splits;
  p.splits = (num_kb + p.kb_per_split - 1) / p.kb_per_split;             // no empty split
#if GP_PROBES
  p.tl = g_timeline;
  {
    static const int dbg = getenv("GPIPE_GEMM_DBG") ? atoi(getenv("GPIPE_GEMM_DBG")) : 0;
    p.dbg = dbg;
  }
#endif
  p.ws_cnt = (unsigned int *)a.ws;
  p.ws_part = (float *)((char *)a.ws + splitk_cnt_bytes(p.tiles_m * p.tiles_n));
  const bool out_f32 = (a.flags & (EPI_OUT_F32 | EPI_ACCUM)) != 0;
  CUtensorMap ma, mb, mc;
  bool ok;
  if (!a.transA) ok = get_map(a.A, 2, (uint64_t)a.K, (uint64_t)a.M, (uint64_t)a.lda, BK, 128, &ma);     // [M,K], K inner
  else ok = get_map(a.A, 2, (uint64_t)a.M, (uint64_t)a.K, (uint64_t)a.lda, 64, BK, &ma);                // [K,M], M inner
  if (!ok) return cudaErrorInvalidValue;
  int b_rows = Cfg::BNH;
#if GP_PROBES
  if (p.dbg & 4) b_rows /= 2;
#endif
  if (a.transB) ok = get_map(a.B, 2, (uint64_t)a.K, (uint64_t)a.N, (uint64_t)a.ldb, BK, b_rows, &mb);    // [N,K], K inner
  else ok = get_map(a.B, 2, (uint64_t)a.N, (uint64_t)a.K, (uint64_t)a.ldb, 64, BK, &mb);                // [K,N], N inner
  if (!ok) return cudaErrorInvalidValue;
  // C: boxes of 32 rows x 128 bytes (32 fp32 / 64 bf16 columns), written from swizzled staging
  ok = get_map(a.C, out_f32 ? 4 : 2, (uint64_t)a.N, (uint64_t)a.M, (uint64_t)a.ldc, out_f32 ? 32 : 64, 32, &mc);
  if (!ok) return cudaErrorInvalidValue;
  {
    cudaError_t e = ensure_dyn_smem<gemm_tcgen05_pair_kernel<BN, F, SPLITK>>(Cfg::SMEM, c.device);
    if (e != cudaSuccess) return e;
  }
  int units = p.tiles_m * p.tiles_n * p.splits;
  int grid = 2 * (units < pairs ? units : pairs);
  gemm_tcgen05_pair_kernel<BN, F, SPLITK><<<grid, NUM_THREADS, Cfg::SMEM, c.stream>>>(ma, mb, mc, p);
  GP_LAUNCH_CHECK(c);
}

}  // namespace tc

// Profiling hook: when set, every tcgen05 GEMM launch writes 8 %globaltimer stamps per CTA to buf
// (entry, prologue done, first operands landed, all MMAs issued, first accumulator complete, last
// chunk handed to the TMA, stores complete, exit) plus 24 SM-clock stamps of the first tile's epilogue
// chunks.  buf must hold 32 * SM-count uint64.
#if GP_PROBES
void gemm_tc_set_timeline(unsigned long long *buf) { tc::g_timeline = buf; }
#endif
cudaError_t gemm_tc_set_watchdog(unsigned long long *mapped) {
  return cudaMemcpyToSymbol(tc::g_watchdog, &mapped, sizeof(mapped));
}

// Workspace a split-K launch of this shape needs (0 when the shape is not split); the first
// splitk_cnt_bytes() bytes are the counters and must be ZERO before the first launch (they reset
// themselves afterwards).
size_t gemm_splitk_ws_bytes(int M, int N, int K, int sm_count) {
  const int tiles = ((M + 255) / 256) * ((N + 255) / 256);
  const int s = tc::splitk_factor(tiles, (K + tc::BK - 1) / tc::BK, sm_count / 2);
  if (s <= 1) return 0;
  return tc::splitk_cnt_bytes(tiles) + (size_t)tiles * s * 2 * 128 * 256 * sizeof(float);
}

bool gemm_tc_supported(int dt, const GemmArgs &a) {
  if (dt != GP_BF16) return false;
  if (a.M <= 0 || a.N <= 0 || a.K <= 0) return false;
  auto al16 = [](const void *p) { return ((uintptr_t)p & 15) == 0; };
  if (!al16(a.A) || !al16(a.B) || !al16(a.C)) return false;
  // TMA: 16-byte aligned bases and row pitches
  if (a.lda % 8 || a.ldb % 8) return false;
  const bool out_f32 = (a.flags & (EPI_OUT_F32 | EPI_ACCUM)) != 0;
  if (a.ldc % (out_f32 ? 4 : 8)) return false;
  if ((a.flags & EPI_RESID) && (!al16(a.resid) || a.ldc % 4)) return false;
  if ((a.flags & (EPI_MASK | EPI_BITS_OUT)) && (a.N % 32 || !a.mask)) return false;
  return true;
}

// The epilogue combinations the engine launches get their own instantiation - the two that occur on few-tile,
// deep-K shapes (plain bf16 output: dgrads; fp32 accumulate: FFN2 / out-projection forward, wgrads) also as a
// split-K variant; anything else takes the run-time-flag kernel.
// 256 x 512 pair tiles (BN = 512).  The full-grid GEMMs are bound by what the L2 can deliver to the SMs (DESIGN.md
// "K1-K3"); a pair tile twice as wide needs (128 + 256) instead of 2 x (128 + 128) operand rows per 128 x 512 outputs of
// a CTA - 25 % fewer delivered bytes per FLOP - at the price of the epilogue / main-loop overlap (one accumulator fills
// all 512 TMEM columns; only the first ring's worth of K-blocks of the next tile overlaps the drain of block 1) and of
// half as many, twice as long work units.  Results are bitwise those of the 256 x 256 tiles (same K order per output).
// Measured (profiles/gemm_wide_r02.md): alone, the wgrads (K = T_mb = 2048, 256 tiles) run 66 us instead of 70-74, the
// K = 1024 forward GEMMs 76 instead of 57 (16 K-blocks do not hide a 4 us drain), the 32-tile deep-K products twice as
// long on half the SMs; in the step, with >= 8 cells in flight everything that can go wide should (config 5:
// 1471 -> 1427 ms, config 4: 547 -> 532), with 2-4 cells only the >= 64-tile products with K >= 2048 (config 3:
// 159.5 -> 157.7 ms, config 2 unchanged; all-wide there is 2-13 % SLOWER: nothing fills the SMs a 16-tile launch
// leaves idle).  gemm_backend 3 forbids the wide tile, 4 forces it (the per-kernel tests).
static bool wide_tile_supported(const GemmArgs &a) {
  const bool flags_ok = a.flags == 0 || a.flags == (EPI_ACCUM | EPI_OUT_F32) ||
                        a.flags == (EPI_BIAS | EPI_RELU | EPI_BITS_OUT);
  return flags_ok && a.N >= 512 && (!(a.flags & EPI_BIAS) || ((uintptr_t)a.bias & 15) == 0);
}
static bool wide_tile(const Ctx &c, const GemmArgs &a, bool split) {
  if (c.gemm_backend == 3 || split || !wide_tile_supported(a)) return false;
  if (c.gemm_backend == 4) return true;
  if (a.N % 512 || (a.flags & EPI_BIAS)) return false;
  const int tiles = ((a.M + 255) / 256) * ((a.N + 255) / 256);
#if GP_PROBES
  // experiment knobs: GPIPE_GEMM_WIDE bit 0 plain bf16 output, bit 1 fp32 accumulate (default 3); MINK / MAXK / MINTILES
  static const int wide = getenv("GPIPE_GEMM_WIDE") ? atoi(getenv("GPIPE_GEMM_WIDE")) : 3;
  static const int mink = getenv("GPIPE_GEMM_WIDE_MINK") ? atoi(getenv("GPIPE_GEMM_WIDE_MINK")) : -1;
  static const int maxk = getenv("GPIPE_GEMM_WIDE_MAXK") ? atoi(getenv("GPIPE_GEMM_WIDE_MAXK")) : 1 << 30;
  static const int mintiles = getenv("GPIPE_GEMM_WIDE_MINTILES") ? atoi(getenv("GPIPE_GEMM_WIDE_MINTILES")) : -1;
  if (!(wide & (a.flags == 0 ? 1 : 2)) || a.K > maxk) return false;
  if (mink >= 0 || mintiles >= 0) return a.K >= mink && tiles >= mintiles;
#endif
  return c.streams >= 8 || (tiles >= 64 && a.K >= 2048);
}

cudaError_t gemm_tc(const Ctx &c, const GemmArgs &a) {
#if GP_PROBES
  static const int generic_only = getenv("GPIPE_GEMM_GENERIC") ? atoi(getenv("GPIPE_GEMM_GENERIC")) : 0;
#else
  constexpr int generic_only = 0;
#endif
  const int tiles = ((a.M + 255) / 256) * ((a.N + 255) / 256);
  const bool split = a.ws && tc::splitk_factor(tiles, (a.K + tc::BK - 1) / tc::BK, c.sm_count / 2) > 1 &&
                     a.ws_bytes >= gemm_splitk_ws_bytes(a.M, a.N, a.K, c.sm_count);
  if (c.gemm_backend == 4 && !wide_tile(c, a, split)) return cudaErrorNotSupported;
  if (wide_tile(c, a, split)) {
    switch (a.flags) {
      case 0: return tc::launch_pair<512, 0, false>(c, a);
      case EPI_ACCUM | EPI_OUT_F32: return tc::launch_pair<512, EPI_ACCUM | EPI_OUT_F32, false>(c, a);
      default: return tc::launch_pair<512, EPI_BIAS | EPI_RELU | EPI_BITS_OUT, false>(c, a);
    }
  }
  if (!generic_only) {
    switch (a.flags) {
      case 0: return split ? tc::launch_pair<256, 0, true>(c, a) : tc::launch_pair<256, 0, false>(c, a);
      case EPI_ACCUM | EPI_OUT_F32:
        return split ? tc::launch_pair<256, EPI_ACCUM | EPI_OUT_F32, true>(c, a)
                     : tc::launch_pair<256, EPI_ACCUM | EPI_OUT_F32, false>(c, a);
      case EPI_BIAS: if (!split) return tc::launch_pair<256, EPI_BIAS, false>(c, a); break;
      case EPI_BIAS | EPI_RELU | EPI_BITS_OUT:
        if (!split) return tc::launch_pair<256, EPI_BIAS | EPI_RELU | EPI_BITS_OUT, false>(c, a);
        break;
      case EPI_MASK | EPI_COLSUM: if (!split) return tc::launch_pair<256, EPI_MASK | EPI_COLSUM, false>(c, a); break;
      default: break;
    }
  }
  return tc::launch_pair<256, -1, true>(c, a);
}

}  // namespace gp

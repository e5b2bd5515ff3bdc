// gemm_tcgen05.cu - bf16 GEMM on the 5th-generation tensor cores of sm_100a.
//
//   C[M,N] = epilogue( op(A)[M,K] * op(B)[K,N] ),   fp32 accumulation in TMEM.
//
// Design:
//   * persistent CTAs (one per SM), static tile schedule, 128 x BN output tiles (BN = 256 or 128),
//     K-blocks of 64 elements, a 4-stage TMA -> shared-memory ring guarded by mbarriers;
//   * warp-specialised: warp 0 = TMA producer (one lane), warp 1 = tcgen05.mma issuer (one lane),
//     warp 2 = TMEM allocator, warps 4-7 = epilogue (one TMEM lane quadrant each);
//   * two TMEM accumulator stages (2 x BN columns), so the epilogue of tile i overlaps the main
//     loop of tile i+1;
//   * all four operand layouts through the shared-memory descriptors: a K-major operand is one TMA
//     box [rows x 64] per stage (128-byte swizzle, 8-row atoms 1024 B apart), an MN-major operand
//     is [64 k x 64 mn] boxes (one per 64 elements of M/N), so forward (NN), dgrad (NT) and wgrad
//     (TN) all read the tensors where they are - no transposed copies in HBM;
//   * fused epilogue straight from TMEM: +bias, ReLU, ReLU-mask, +fp32 residual, fp32
//     read-modify-write accumulation (wgrad across micro-batches), bf16 or fp32 output;
//   * out-of-bounds parts of a box are zero-filled by TMA, so ragged M/N/K only need store guards.
// Roofline: bf16 tensor pipe (wgrad with fp32 RMW sits near the HBM ridge).
#include <cuda.h>

#include <stdlib.h>

#include <mutex>
#include <unordered_map>

#include "common.cuh"
#include "tcgen05.cuh"

namespace gp {

namespace tc {

constexpr int BM = 128, BK = 64, STAGES = 4;
constexpr int NUM_THREADS = 256;
constexpr int EPI_WARP0 = 4;

struct Params {
  int M, N, K;
  int a_mn_major, b_mn_major;   // 1: operand is MN-major in global memory (transA / !transB)
  void *C;
  int64_t ldc;
  const float *bias;
  const float *resid;
  const bf16 *mask;
  int64_t ldmask;
  int flags;
  int tiles_m, tiles_n;
  float *colpart;               // EPI_COLSUM: fp32 [tiles_m, N] per-tile-row column sums
};

// Epilogue of one 32-column chunk of one accumulator row: +bias, ReLU, ReLU-mask, +residual, fp32
// accumulate, store (bf16 or fp32).  On return v[] holds the values as stored (0 where nothing was
// stored), which is what EPI_COLSUM sums.
__device__ __forceinline__ void epilogue_chunk(const Params &p, const int row, const bool row_ok, const int col0,
                                               const bool out_f32, float (&v)[32]) {
  const bool active = row_ok && col0 < p.N;
  const bool full = col0 + 32 <= p.N;
  if (active) {
    if (full) {
      if (p.flags & EPI_BIAS) {
#pragma unroll
        for (int j = 0; j < 32; j += 4) {
          float4 b = __ldg(reinterpret_cast<const float4 *>(p.bias + col0 + j));
          v[j] += b.x; v[j + 1] += b.y; v[j + 2] += b.z; v[j + 3] += b.w;
        }
      }
      if (p.flags & EPI_RELU) {
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = fmaxf(v[j], 0.f);
      }
      if (p.flags & EPI_MASK) {
        const bf16 *mp = p.mask + (int64_t)row * p.ldmask + col0;
#pragma unroll
        for (int j = 0; j < 32; j += 8) {
          uint4 u = *reinterpret_cast<const uint4 *>(mp + j);
          const __nv_bfloat162 *h = reinterpret_cast<const __nv_bfloat162 *>(&u);
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            float2 f = __bfloat1622float2(h[q]);
            v[j + 2 * q] = f.x > 0.f ? v[j + 2 * q] : 0.f;
            v[j + 2 * q + 1] = f.y > 0.f ? v[j + 2 * q + 1] : 0.f;
          }
        }
      }
      if (p.flags & EPI_RESID) {
        const float *rp = p.resid + (int64_t)row * p.ldc + col0;
#pragma unroll
        for (int j = 0; j < 32; j += 4) {
          float4 b = *reinterpret_cast<const float4 *>(rp + j);
          v[j] += b.x; v[j + 1] += b.y; v[j + 2] += b.z; v[j + 3] += b.w;
        }
      }
      if (out_f32) {
        float *cp = (float *)p.C + (int64_t)row * p.ldc + col0;
        if (p.flags & EPI_ACCUM) {
#pragma unroll
          for (int j = 0; j < 32; j += 4) {
            float4 b = *reinterpret_cast<const float4 *>(cp + j);
            v[j] += b.x; v[j + 1] += b.y; v[j + 2] += b.z; v[j + 3] += b.w;
          }
        }
#pragma unroll
        for (int j = 0; j < 32; j += 4)
          *reinterpret_cast<float4 *>(cp + j) = make_float4(v[j], v[j + 1], v[j + 2], v[j + 3]);
      } else {
        bf16 *cp = (bf16 *)p.C + (int64_t)row * p.ldc + col0;
#pragma unroll
        for (int j = 0; j < 32; j += 8) {
          uint4 u;
          __nv_bfloat162 *h = reinterpret_cast<__nv_bfloat162 *>(&u);
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            h[q] = __floats2bfloat162_rn(v[j + 2 * q], v[j + 2 * q + 1]);
            float2 f = __bfloat1622float2(h[q]);          // the stored values (for EPI_COLSUM)
            v[j + 2 * q] = f.x;
            v[j + 2 * q + 1] = f.y;
          }
          *reinterpret_cast<uint4 *>(cp + j) = u;
        }
      }
    } else {
      // ragged right edge: element-wise, guarded
#pragma unroll
      for (int j = 0; j < 32; ++j) {
        const int col = col0 + j;
        float x = v[j];
        if (col < p.N) {
          if (p.flags & EPI_BIAS) x += p.bias[col];
          if (p.flags & EPI_RELU) x = fmaxf(x, 0.f);
          if (p.flags & EPI_MASK) x = __bfloat162float(p.mask[(int64_t)row * p.ldmask + col]) > 0.f ? x : 0.f;
          if (p.flags & EPI_RESID) x += p.resid[(int64_t)row * p.ldc + col];
          if (out_f32) {
            float *cp = (float *)p.C + (int64_t)row * p.ldc + col;
            if (p.flags & EPI_ACCUM) x += *cp;
            *cp = x;
          } else {
            bf16 xb = __float2bfloat16_rn(x);
            ((bf16 *)p.C)[(int64_t)row * p.ldc + col] = xb;
            x = __bfloat162float(xb);
          }
        } else {
          x = 0.f;
        }
        v[j] = x;
      }
    }
  }
  if (!active) {
#pragma unroll
    for (int j = 0; j < 32; ++j) v[j] = 0.f;
  }
}

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
template <int BN>
__global__ void __launch_bounds__(NUM_THREADS, 1)
gemm_tcgen05_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b,
                    const Params p) {
  constexpr uint32_t A_BYTES = BM * BK * 2, B_BYTES = BN * BK * 2;
  constexpr uint32_t STAGE_BYTES = A_BYTES + B_BYTES;
  constexpr uint32_t TMEM_COLS = 2 * BN;
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * STAGES + 4];
  __shared__ uint32_t tmem_base_smem;
  __shared__ float colbuf[4][BN];                  // EPI_COLSUM: per-warp column sums of one tile

  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;      // 1024-B aligned (swizzle atoms)
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t bar0 = smem_u32(bars);
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (STAGES + s); };
  auto tfull_bar = [&](int s) { return bar0 + 8u * (2 * STAGES + s); };
  auto tempty_bar = [&](int s) { return bar0 + 8u * (2 * STAGES + 2 + s); };

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&map_a);
    tma_prefetch_desc(&map_b);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full_bar(s), 1);
      mbar_init(empty_bar(s), 1);
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(tfull_bar(s), 1);
      mbar_init(tempty_bar(s), 4);               // one arrive per epilogue warp
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_smem)),
                 "n"(TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem_base = tmem_base_smem;

  const int num_tiles = p.tiles_m * p.tiles_n;
  const int num_kb = (p.K + BK - 1) / BK;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
        const int m0 = (t % p.tiles_m) * BM, n0 = (t / p.tiles_m) * BN;
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(empty_bar(stage), phase ^ 1);
          const uint32_t sa = smem_base + stage * STAGE_BYTES, sb = sa + A_BYTES;
          mbar_expect_tx(full_bar(stage), STAGE_BYTES);
          const int k0 = kb * BK;
          if (!p.a_mn_major) {
            tma_load_2d(sa, &map_a, full_bar(stage), k0, m0);                 // box [BM rows x 64 k]
          } else {
#pragma unroll
            for (int c = 0; c < BM / 64; ++c)                                  // boxes [64 k x 64 m]
              tma_load_2d(sa + c * (BK * 128), &map_a, full_bar(stage), m0 + c * 64, k0);
          }
          if (!p.b_mn_major) {
            tma_load_2d(sb, &map_b, full_bar(stage), k0, n0);                 // box [BN rows x 64 k]
          } else {
#pragma unroll
            for (int c = 0; c < BN / 64; ++c)                                  // boxes [64 k x 64 n]
              tma_load_2d(sb + c * (BK * 128), &map_b, full_bar(stage), n0 + c * 64, k0);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      // instruction descriptor: D fp32, A/B bf16, majorness, N >> 3, M >> 4
      const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)p.a_mn_major << 15) |
                             ((uint32_t)p.b_mn_major << 16) | ((uint32_t)(BN >> 3) << 17) |
                             ((uint32_t)(BM >> 4) << 24);
      // K-major: 8-row atoms 1024 B apart, +32 B per 16 k.  MN-major: 64-element chunks BK*128 B
      // apart (LBO), 8-k groups 1024 B apart (SBO), +2048 B per 16 k.
      const uint32_t a_lbo = p.a_mn_major ? BK * 128 : 16, a_sbo = 1024, a_kstep = p.a_mn_major ? 2048 : 32;
      const uint32_t b_lbo = p.b_mn_major ? BK * 128 : 16, b_sbo = 1024, b_kstep = p.b_mn_major ? 2048 : 32;
      int stage = 0;
      uint32_t phase = 0;
      int as = 0;
      uint32_t aphase = 0;
      for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
        mbar_wait(tempty_bar(as), aphase ^ 1);       // epilogue has drained this accumulator
        tcgen05_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(as * BN);
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(full_bar(stage), phase);
          tcgen05_fence_after();
          const uint32_t sa = smem_base + stage * STAGE_BYTES, sb = sa + A_BYTES;
#pragma unroll
          for (int k = 0; k < BK / 16; ++k) {
            const uint64_t ad = make_smem_desc(sa + k * a_kstep, a_lbo, a_sbo);
            const uint64_t bd = make_smem_desc(sb + k * b_kstep, b_lbo, b_sbo);
            umma_bf16(d_tmem, ad, bd, idesc, (kb | k) ? 1u : 0u);
          }
          tcgen05_commit(empty_bar(stage));          // frees the smem stage when the MMAs retire
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        tcgen05_commit(tfull_bar(as));               // accumulator complete -> epilogue
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
  } else if (warp >= EPI_WARP0) {
    // ===================== epilogue: TMEM -> registers -> global =====================
    const int quad = warp & 3;                       // TMEM lane quadrant of this warp
    int as = 0;
    uint32_t aphase = 0;
    const bool out_f32 = (p.flags & (EPI_OUT_F32 | EPI_ACCUM)) != 0;
    for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
      const int m0 = (t % p.tiles_m) * BM, n0 = (t / p.tiles_m) * BN;
      mbar_wait(tfull_bar(as), aphase);
      tcgen05_fence_after();
      const int row = m0 + quad * 32 + lane;
      const bool row_ok = row < p.M;
      const uint32_t t_row = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(as * BN);
#pragma unroll 1
      for (int c = 0; c < BN / 32; ++c) {
        uint32_t r[32];
        tmem_ld32(t_row + c * 32, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]);
        epilogue_chunk(p, row, row_ok, n0 + c * 32, out_f32, v);
        if (p.flags & EPI_COLSUM) {
          warp_colsum32(v, lane);
          colbuf[quad][c * 32 + lane] = v[0];
        }
      }
      if (p.flags & EPI_COLSUM) {
        asm volatile("bar.sync 1, 128;" ::: "memory");
        const int e = threadIdx.x - EPI_WARP0 * 32;
        for (int cc = e; cc < BN; cc += 128) {
          float ssum = (colbuf[0][cc] + colbuf[1][cc]) + (colbuf[2][cc] + colbuf[3][cc]);
          if (n0 + cc < p.N) p.colpart[(int64_t)(t % p.tiles_m) * p.N + n0 + cc] = ssum;
        }
        asm volatile("bar.sync 1, 128;" ::: "memory");
      }
      tcgen05_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty_bar(as));
      if (++as == 2) { as = 0; aphase ^= 1; }
    }
  }

  tcgen05_fence_before();
  __syncthreads();
  if (warp == 2) {
    tcgen05_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(TMEM_COLS));
  }
}

// ------------------------------------------------------------------------------------------
// CTA-pair kernel (cta_group::2): two CTAs on the two SMs of a TPC compute one 256 x BN tile.
// Each CTA stages its own 128 rows of A and HALF of the B tile (BN/2 columns); the leader's
// tcgen05.mma.cta_group::2 reads both halves of B and writes rows [0,128) of the tile into its own
// TMEM and rows [128,256) into the peer's.  Per SM this needs (128 + BN/2) x 64 x 2 B of
// L2->shared traffic per 128 x BN x 64 MACs: 1.5x less than the 1-CTA 128 x 256 tile, which the
// L2->SM fabric (not the tensor pipe) bounds.  Barriers: TMA of both CTAs
// completes on the LEADER's full barrier; tcgen05.commit multicasts the "stage free" and
// "accumulator ready" arrivals to both CTAs; both CTAs' epilogue warps arrive on the leader's
// "accumulator drained" barrier.
// ------------------------------------------------------------------------------------------
template <int BN> struct PairCfg {
  static constexpr int BNH = BN / 2;
  static constexpr uint32_t A_BYTES = 128 * BK * 2, B_BYTES = BNH * BK * 2, STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int STAGES = (200 * 1024) / STAGE_BYTES > 8 ? 8 : (200 * 1024) / STAGE_BYTES;
  static constexpr uint32_t TMEM_COLS = 2 * BN > 256 ? 512 : 256;
  static constexpr size_t SMEM = (size_t)STAGES * STAGE_BYTES + 1024;
};

template <int BN>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NUM_THREADS, 1)
gemm_tcgen05_pair_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b,
                         const Params p) {
  using Cfg = PairCfg<BN>;
  constexpr int NST = Cfg::STAGES, BNH = Cfg::BNH;
  constexpr uint32_t A_BYTES = Cfg::A_BYTES, STAGE_BYTES = Cfg::STAGE_BYTES;
  static_assert(BN % 32 == 0 && BN <= 256 && BNH % 8 == 0, "tile N");
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * NST + 4];
  __shared__ uint32_t tmem_base_smem;
  __shared__ float colbuf[4][BN];

  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int pair = blockIdx.x >> 1, num_pairs = gridDim.x >> 1;
  const uint32_t bar0 = smem_u32(bars);
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (NST + s); };
  auto tfull_bar = [&](int s) { return bar0 + 8u * (2 * NST + s); };
  auto tempty_bar = [&](int s) { return bar0 + 8u * (2 * NST + 2 + s); };

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&map_a);
    tma_prefetch_desc(&map_b);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < NST; ++s) {
      mbar_init(full_bar(s), 1);                   // leader's: its producer's arrive.expect_tx (both CTAs' bytes)
      mbar_init(empty_bar(s), 1);                  // one multicast tcgen05.commit
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(tfull_bar(s), 1);
      mbar_init(tempty_bar(s), 8);                 // leader's: 4 epilogue warps of each CTA
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_smem)),
                 "n"(Cfg::TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;");
  }
  tcgen05_fence_before();
  cluster_sync_all();
  tcgen05_fence_after();
  const uint32_t tmem_base = tmem_base_smem;

  const int num_tiles = p.tiles_m * p.tiles_n;
  const int num_kb = (p.K + BK - 1) / BK;

  if (warp == 0) {
    // ===================== TMA producer (both CTAs) =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int t = pair; t < num_tiles; t += num_pairs) {
        const int m0 = (t % p.tiles_m) * 256 + (int)rank * 128, n0 = (t / p.tiles_m) * BN + (int)rank * BNH;
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(empty_bar(stage), phase ^ 1);
          const uint32_t sa = smem_base + stage * STAGE_BYTES, sb = sa + A_BYTES;
          if (rank == 0) mbar_expect_tx(full_bar(stage), 2 * STAGE_BYTES);
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
            for (int c = 0; c < BNH / 64; ++c)                                 // boxes [64 k x 64 n]
              tma_load_2d_pair(sb + c * (BK * 128), &map_b, fb, n0 + c * 64, k0);
          }
          if (++stage == NST) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA only) =====================
    if (lane == 0 && rank == 0) {
      const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)p.a_mn_major << 15) |
                             ((uint32_t)p.b_mn_major << 16) | ((uint32_t)(BN >> 3) << 17) |
                             ((uint32_t)(256 >> 4) << 24);
      const uint32_t a_lbo = p.a_mn_major ? BK * 128 : 16, a_sbo = 1024, a_kstep = p.a_mn_major ? 2048 : 32;
      const uint32_t b_lbo = p.b_mn_major ? BK * 128 : 16, b_sbo = 1024, b_kstep = p.b_mn_major ? 2048 : 32;
      int stage = 0;
      uint32_t phase = 0;
      int as = 0;
      uint32_t aphase = 0;
      for (int t = pair; t < num_tiles; t += num_pairs) {
        mbar_wait(tempty_bar(as), aphase ^ 1);       // both CTAs' epilogues have drained this accumulator
        tcgen05_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(as * BN);
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(full_bar(stage), phase);
          tcgen05_fence_after();
          const uint32_t sa = smem_base + stage * STAGE_BYTES, sb = sa + A_BYTES;
#pragma unroll
          for (int k = 0; k < BK / 16; ++k) {
            const uint64_t ad = make_smem_desc(sa + k * a_kstep, a_lbo, a_sbo);
            const uint64_t bd = make_smem_desc(sb + k * b_kstep, b_lbo, b_sbo);
            umma_bf16_pair(d_tmem, ad, bd, idesc, (kb | k) ? 1u : 0u);
          }
          tcgen05_commit_pair(empty_bar(stage), 3);  // frees this stage in both CTAs
          if (++stage == NST) { stage = 0; phase ^= 1; }
        }
        tcgen05_commit_pair(tfull_bar(as), 3);       // accumulator complete -> both epilogues
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
  } else if (warp >= EPI_WARP0) {
    // ===================== epilogue (both CTAs): own 128 rows of the tile =====================
    const int quad = warp & 3;
    int as = 0;
    uint32_t aphase = 0;
    const bool out_f32 = (p.flags & (EPI_OUT_F32 | EPI_ACCUM)) != 0;
    for (int t = pair; t < num_tiles; t += num_pairs) {
      const int m0 = (t % p.tiles_m) * 256 + (int)rank * 128, n0 = (t / p.tiles_m) * BN;
      mbar_wait(tfull_bar(as), aphase);
      tcgen05_fence_after();
      const int row = m0 + quad * 32 + lane;
      const bool row_ok = row < p.M;
      const uint32_t t_row = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(as * BN);
#pragma unroll 1
      for (int c = 0; c < BN / 32; ++c) {
        uint32_t r[32];
        tmem_ld32(t_row + c * 32, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]);
        epilogue_chunk(p, row, row_ok, n0 + c * 32, out_f32, v);
        if (p.flags & EPI_COLSUM) {
          warp_colsum32(v, lane);
          colbuf[quad][c * 32 + lane] = v[0];
        }
      }
      if (p.flags & EPI_COLSUM) {
        asm volatile("bar.sync 1, 128;" ::: "memory");
        const int e = threadIdx.x - EPI_WARP0 * 32;
        for (int cc = e; cc < BN; cc += 128) {
          float ssum = (colbuf[0][cc] + colbuf[1][cc]) + (colbuf[2][cc] + colbuf[3][cc]);
          if (n0 + cc < p.N && m0 < p.M) p.colpart[(int64_t)(m0 >> 7) * p.N + n0 + cc] = ssum;
        }
        asm volatile("bar.sync 1, 128;" ::: "memory");
      }
      tcgen05_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(mapa_shared(tempty_bar(as), 0));
      if (++as == 2) { as = 0; aphase ^= 1; }
    }
  }

  tcgen05_fence_before();
  cluster_sync_all();                                // the peer's smem / TMEM / barriers stay valid until both are done
  if (warp == 2) {
    tcgen05_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(Cfg::TMEM_COLS));
  }
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
  uint32_t box_inner, box_outer;
  bool operator==(const MapKey &o) const {
    return ptr == o.ptr && inner == o.inner && outer == o.outer && ld == o.ld && box_inner == o.box_inner &&
           box_outer == o.box_outer;
  }
};
struct MapKeyHash {
  size_t operator()(const MapKey &k) const {
    size_t h = (size_t)k.ptr;
    auto mix = [&](uint64_t v) { h ^= v + 0x9e3779b97f4a7c15ull + (h << 6) + (h >> 2); };
    mix(k.inner); mix(k.outer); mix(k.ld); mix(k.box_inner); mix(k.box_outer);
    return h;
  }
};

// 2-D bf16 tensor [outer, inner] with row pitch ld elements; box [box_outer, box_inner]
static bool get_map(const void *ptr, uint64_t inner, uint64_t outer, uint64_t ld, uint32_t box_inner,
                    uint32_t box_outer, CUtensorMap *out) {
  static std::unordered_map<MapKey, CUtensorMap, MapKeyHash> cache;
  static std::mutex mu;
  MapKey key{ptr, inner, outer, ld, box_inner, box_outer};
  std::lock_guard<std::mutex> lock(mu);
  auto it = cache.find(key);
  if (it != cache.end()) {
    *out = it->second;
    return true;
  }
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {inner, outer};
  cuuint64_t strides[1] = {ld * 2};
  cuuint32_t box[2] = {box_inner, box_outer};
  cuuint32_t estr[2] = {1, 1};
  CUtensorMap m;
  CUresult r = fn(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(ptr), dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return false;
  if (cache.size() > 65536) cache.clear();
  cache.emplace(key, m);
  *out = m;
  return true;
}

template <int BN>
static cudaError_t launch(const Ctx &c, const GemmArgs &a) {
  Params p{};
  p.M = a.M; p.N = a.N; p.K = a.K;
  p.a_mn_major = a.transA ? 1 : 0;
  p.b_mn_major = a.transB ? 0 : 1;
  p.C = a.C; p.ldc = a.ldc; p.bias = a.bias; p.resid = a.resid; p.mask = (const bf16 *)a.mask; p.ldmask = a.ldmask;
  p.flags = a.flags;
  p.colpart = a.colsum_scratch;
  p.tiles_m = (a.M + BM - 1) / BM;
  p.tiles_n = (a.N + BN - 1) / BN;
  CUtensorMap ma, mb;
  bool ok;
  if (!a.transA) ok = get_map(a.A, (uint64_t)a.K, (uint64_t)a.M, (uint64_t)a.lda, BK, BM, &ma);     // [M,K], K inner
  else ok = get_map(a.A, (uint64_t)a.M, (uint64_t)a.K, (uint64_t)a.lda, 64, BK, &ma);               // [K,M], M inner
  if (!ok) return cudaErrorInvalidValue;
  if (a.transB) ok = get_map(a.B, (uint64_t)a.K, (uint64_t)a.N, (uint64_t)a.ldb, BK, BN, &mb);      // [N,K], K inner
  else ok = get_map(a.B, (uint64_t)a.N, (uint64_t)a.K, (uint64_t)a.ldb, 64, BK, &mb);               // [K,N], N inner
  if (!ok) return cudaErrorInvalidValue;
  constexpr size_t smem = (size_t)STAGES * (BM * BK * 2 + BN * BK * 2) + 1024;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(gemm_tcgen05_kernel<BN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  int tiles = p.tiles_m * p.tiles_n;
  int grid = tiles < c.sm_count ? tiles : c.sm_count;
  gemm_tcgen05_kernel<BN><<<grid, NUM_THREADS, smem, c.stream>>>(ma, mb, p);
  GP_LAUNCH_CHECK(c);
}

template <int BN>
static cudaError_t launch_pair(const Ctx &c, const GemmArgs &a) {
  using Cfg = PairCfg<BN>;
  Params p{};
  p.M = a.M; p.N = a.N; p.K = a.K;
  p.a_mn_major = a.transA ? 1 : 0;
  p.b_mn_major = a.transB ? 0 : 1;
  p.C = a.C; p.ldc = a.ldc; p.bias = a.bias; p.resid = a.resid; p.mask = (const bf16 *)a.mask; p.ldmask = a.ldmask;
  p.flags = a.flags;
  p.colpart = a.colsum_scratch;
  p.tiles_m = (a.M + 255) / 256;
  p.tiles_n = (a.N + BN - 1) / BN;
  CUtensorMap ma, mb;
  bool ok;
  if (!a.transA) ok = get_map(a.A, (uint64_t)a.K, (uint64_t)a.M, (uint64_t)a.lda, BK, 128, &ma);    // [M,K], K inner
  else ok = get_map(a.A, (uint64_t)a.M, (uint64_t)a.K, (uint64_t)a.lda, 64, BK, &ma);               // [K,M], M inner
  if (!ok) return cudaErrorInvalidValue;
  if (a.transB) ok = get_map(a.B, (uint64_t)a.K, (uint64_t)a.N, (uint64_t)a.ldb, BK, Cfg::BNH, &mb); // [N,K], K inner
  else ok = get_map(a.B, (uint64_t)a.N, (uint64_t)a.K, (uint64_t)a.ldb, 64, BK, &mb);               // [K,N], N inner
  if (!ok) return cudaErrorInvalidValue;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(gemm_tcgen05_pair_kernel<BN>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)Cfg::SMEM);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  int tiles = p.tiles_m * p.tiles_n;
  int pairs = c.sm_count / 2;
  int grid = 2 * (tiles < pairs ? tiles : pairs);
  gemm_tcgen05_pair_kernel<BN><<<grid, NUM_THREADS, Cfg::SMEM, c.stream>>>(ma, mb, p);
  GP_LAUNCH_CHECK(c);
}

}  // namespace tc

bool gemm_tc_supported(int dt, const GemmArgs &a) {
  if (dt != GP_BF16) return false;
  if (a.M <= 0 || a.N <= 0 || a.K <= 0) return false;
  auto al16 = [](const void *p) { return ((uintptr_t)p & 15) == 0; };
  if (!al16(a.A) || !al16(a.B) || !al16(a.C)) return false;
  if (a.lda % 8 || a.ldb % 8) return false;
  // extents of the contiguous dimensions must keep TMA strides 16-byte multiples (ld % 8) and the
  // vectorised epilogue aligned
  if (a.ldc % 8 || a.N % 8) return false;
  if ((a.flags & EPI_MASK) && (a.ldmask % 8 || !al16(a.mask))) return false;
  if ((a.flags & EPI_BIAS) && !al16(a.bias)) return false;
  if ((a.flags & EPI_RESID) && !al16(a.resid)) return false;
  return true;
}

cudaError_t gemm_tc(const Ctx &c, const GemmArgs &a) {
  // CTA pairs (256 x 256 tiles) for everything big enough to give each pair real work
  static const int force = getenv("GPIPE_GEMM_KERNEL") ? atoi(getenv("GPIPE_GEMM_KERNEL")) : 0;   // 1: 1-CTA, 2: pair
  if (force != 1 && ((a.M >= 256 && a.N >= 256) || force == 2)) return tc::launch_pair<256>(c, a);
  // BN = 256 when that still gives every SM a tile, else 128 (less wave quantisation)
  int tiles256 = ((a.M + tc::BM - 1) / tc::BM) * ((a.N + 255) / 256);
  if (tiles256 >= c.sm_count && a.N >= 256) return tc::launch<256>(c, a);
  return tc::launch<128>(c, a);
}

}  // namespace gp

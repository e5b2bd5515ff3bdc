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

#include <mutex>
#include <unordered_map>

#include "common.cuh"

namespace gp {

namespace tc {

constexpr int BM = 128, BK = 64, STAGES = 4;
constexpr int NUM_THREADS = 256;
constexpr int EPI_WARP0 = 4;

// ------------------------------------------------------------------------------------------
// PTX wrappers
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ uint32_t mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {
  }
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(dst), "l"((uint64_t)map), "r"(bar), "r"(c0), "r"(c1)
      : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap *map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"((uint64_t)map) : "memory");
}
__device__ __forceinline__ void tcgen05_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tcgen05_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tcgen05_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accum) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accum)
      : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t *r) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
        "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
        "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Shared-memory matrix descriptor (sm_100 format): start address, leading / stride byte offsets
// (all >> 4), version 1, 128-byte swizzle.
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((addr >> 4) & 0x3FFF);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;      // descriptor version (Blackwell)
  d |= (uint64_t)2 << 61;      // SWIZZLE_128B
  return d;
}

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
        const int col0 = n0 + c * 32;
        const bool active = row_ok && col0 < p.N;
        const bool full = col0 + 32 <= p.N;
        float v[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]);
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
        if (p.flags & EPI_COLSUM) {
          // column sums over this warp's 32 rows: transpose-reduce across lanes (31 shuffles);
          // afterwards lane j holds the sum of column col0 + j
          if (!active) {
#pragma unroll
            for (int j = 0; j < 32; ++j) v[j] = 0.f;
          }
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
  // BN = 256 when that still gives every SM a tile, else 128 (less wave quantisation)
  int tiles256 = ((a.M + tc::BM - 1) / tc::BM) * ((a.N + 255) / 256);
  if (tiles256 >= c.sm_count && a.N >= 256) return tc::launch<256>(c, a);
  return tc::launch<128>(c, a);
}

}  // namespace gp

// attention_mma.cu - flash-style attention forward / backward on tensor cores (bf16 operands, fp32
// accumulation, warp-level online softmax; K5/K6 of DESIGN.md).
//
// One CTA = 4 warps = 64 query rows (forward, dq) or 64 key rows (dk/dv) of one (sequence, head);
// each warp owns 16 rows and keeps its S / P / dS tiles in registers (never in HBM).  The head's
// K and V (or Q and dO) are staged once in shared memory with an XOR swizzle (conflict-free
// ldmatrix).  Scores use mma.sync.m16n8k16 (the legacy warp-level tensor path: attention is 1-2 %
// of the step's FLOPs; the tcgen05 path is reserved for the GEMMs - DESIGN.md "What differs").
// The backward pass is two deterministic kernels (no atomics): dq per query block, dk/dv per key
// block, both recomputing P = exp(S - lse) from the saved log-sum-exp.
#include <math.h>

#include "common.cuh"

namespace gp {
namespace fa {

constexpr int BLK = 64;          // rows per CTA and keys per inner step
constexpr int NWARP = 4;

template <int DH>
struct Tile {
  static constexpr int CH = DH / 8;        // 16-byte chunks per row
  static constexpr int ROWB = DH * 2;
  __device__ static __forceinline__ uint32_t addr(uint32_t base, int r, int c) {
    int sw = DH >= 64 ? (r & 7) : ((r >> 1) & 3);
    return base + (uint32_t)(r * ROWB) + (uint32_t)(((c ^ sw) & (CH - 1)) << 4);
  }
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src, bool valid) {
  int sz = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
  asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
}
__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma16816(float *c, const uint32_t *a, uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t *>(&v);
}

// copy rows [row0, row0+n_rows) x DH of a [*, ld] bf16 matrix into a swizzled tile; rows >= row_limit
// are zero-filled
template <int DH>
__device__ __forceinline__ void load_tile(uint32_t dst, const bf16 *src, int64_t ld, int row0, int n_rows,
                                          int row_limit) {
  constexpr int CH = Tile<DH>::CH;
  for (int i = threadIdx.x; i < n_rows * CH; i += blockDim.x) {
    int r = i / CH, c = i - r * CH;
    bool ok = row0 + r < row_limit;
    const bf16 *p = src + (int64_t)(ok ? row0 + r : 0) * ld + c * 8;
    cp_async16(Tile<DH>::addr(dst, r, c), p, ok);
  }
}

// A fragments (16 rows x DH) of a tile, rows row0..row0+15
template <int DH>
__device__ __forceinline__ void load_a_frags(uint32_t tile, int row0, uint32_t (*f)[4]) {
  int lane = threadIdx.x & 31;
#pragma unroll
  for (int ks = 0; ks < DH / 16; ++ks)
    ldsm_x4(Tile<DH>::addr(tile, row0 + (lane & 15), ks * 2 + (lane >> 4)), f[ks][0], f[ks][1], f[ks][2], f[ks][3]);
}

// acc[nt][4] += A(16 x DH) * B^T where B is stored [n][DH] (rows n0..n0+63): scores / dP style products
template <int DH>
__device__ __forceinline__ void mma_a_bT(float (*acc)[4], const uint32_t (*af)[4], uint32_t tile, int n0) {
  int lane = threadIdx.x & 31;
#pragma unroll
  for (int ks = 0; ks < DH / 16; ++ks) {
#pragma unroll
    for (int np = 0; np < 4; ++np) {
      uint32_t b0, b1, b2, b3;
      ldsm_x4(Tile<DH>::addr(tile, n0 + np * 16 + (lane & 7) + ((lane >> 4) << 3), ks * 2 + ((lane >> 3) & 1)), b0, b1, b2, b3);
      mma16816(acc[2 * np], af[ks], b0, b1);
      mma16816(acc[2 * np + 1], af[ks], b2, b3);
    }
  }
}

// acc[nt][4] (16 x DH) += P(16 x 64, bf16 A fragments pf[4][4]) * B where B is stored [k][DH], rows k0..k0+63
template <int DH>
__device__ __forceinline__ void mma_p_b(float (*acc)[4], const uint32_t (*pf)[4], uint32_t tile, int k0) {
  int lane = threadIdx.x & 31;
#pragma unroll
  for (int kk = 0; kk < 4; ++kk) {
#pragma unroll
    for (int np = 0; np < DH / 16; ++np) {
      uint32_t b0, b1, b2, b3;
      ldsm_x4_t(Tile<DH>::addr(tile, k0 + kk * 16 + (lane & 7) + (((lane >> 3) & 1) << 3), np * 2 + (lane >> 4)), b0, b1, b2, b3);
      mma16816(acc[2 * np], pf[kk], b0, b1);
      mma16816(acc[2 * np + 1], pf[kk], b2, b3);
    }
  }
}

__device__ __forceinline__ void acc_to_a_frags(const float (*acc)[4], uint32_t (*pf)[4]) {
#pragma unroll
  for (int kk = 0; kk < 4; ++kk) {
    pf[kk][0] = pack_bf16(acc[2 * kk][0], acc[2 * kk][1]);
    pf[kk][1] = pack_bf16(acc[2 * kk][2], acc[2 * kk][3]);
    pf[kk][2] = pack_bf16(acc[2 * kk + 1][0], acc[2 * kk + 1][1]);
    pf[kk][3] = pack_bf16(acc[2 * kk + 1][2], acc[2 * kk + 1][3]);
  }
}

constexpr float LOG2E = 1.4426950408889634f;

// ---------------------------------------------------------------------------------------------
// forward
// ---------------------------------------------------------------------------------------------
template <int DH>
__global__ void __launch_bounds__(NWARP * 32)
attn_fwd_mma_kernel(const bf16 *__restrict__ qkv, bf16 *__restrict__ o, float *__restrict__ lse, int S, int A,
                    int causal, float scale) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int da = A * DH, seq = blockIdx.y / A, h = blockIdx.y % A;
  const int q0 = blockIdx.x * BLK;
  const int nk = causal ? min(S, q0 + BLK) : S;              // keys this block needs
  const int nkb = (nk + BLK - 1) / BLK;
  const uint32_t Qs = smem_u32(smem), Ks = Qs + BLK * Tile<DH>::ROWB, Vs = Ks + nkb * BLK * Tile<DH>::ROWB;
  const bf16 *base = qkv + (int64_t)seq * S * 3 * da + h * DH;
  load_tile<DH>(Qs, base, 3 * da, q0, BLK, S);
  load_tile<DH>(Ks, base + da, 3 * da, 0, nkb * BLK, nk);
  load_tile<DH>(Vs, base + 2 * da, 3 * da, 0, nkb * BLK, nk);
  cp_async_wait_all();
  __syncthreads();

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  uint32_t qf[DH / 16][4];
  load_a_frags<DH>(Qs, warp * 16, qf);
  const int r0 = q0 + warp * 16 + g, r1 = r0 + 8;
  const float sl2 = scale * LOG2E;
  float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
  float acc_o[DH / 8][4];
#pragma unroll
  for (int i = 0; i < DH / 8; ++i) acc_o[i][0] = acc_o[i][1] = acc_o[i][2] = acc_o[i][3] = 0.f;

  const int kb_end = causal ? min(nkb, (q0 + warp * 16 + 15) / BLK + 1) : nkb;
  for (int kb = 0; kb < kb_end; ++kb) {
    float s[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i) s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f;
    mma_a_bT<DH>(s, qf, Ks, kb * BLK);
    const bool need_mask = (kb * BLK + BLK > nk) || (causal && kb * BLK + BLK - 1 > q0 + warp * 16);
    if (need_mask) {
#pragma unroll
      for (int nt = 0; nt < 8; ++nt)
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          int key = kb * BLK + nt * 8 + 2 * t + (e & 1);
          int row = (e & 2) ? r1 : r0;
          if (key >= nk || (causal && key > row)) s[nt][e] = -INFINITY;
        }
    }
    float mx0 = m0, mx1 = m1;
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) {
      mx0 = fmaxf(mx0, fmaxf(s[nt][0], s[nt][1]));
      mx1 = fmaxf(mx1, fmaxf(s[nt][2], s[nt][3]));
    }
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
    // rows past the end of the sequence can be fully masked in the causal case: keep them finite
    const float ms0 = mx0 == -INFINITY ? 0.f : mx0 * sl2, ms1 = mx1 == -INFINITY ? 0.f : mx1 * sl2;
    const float c0 = exp2f(m0 == -INFINITY ? -INFINITY : m0 * sl2 - ms0);
    const float c1 = exp2f(m1 == -INFINITY ? -INFINITY : m1 * sl2 - ms1);
    m0 = mx0; m1 = mx1;
    float ps0 = 0.f, ps1 = 0.f;
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) {
      s[nt][0] = exp2f(s[nt][0] * sl2 - ms0); s[nt][1] = exp2f(s[nt][1] * sl2 - ms0);
      s[nt][2] = exp2f(s[nt][2] * sl2 - ms1); s[nt][3] = exp2f(s[nt][3] * sl2 - ms1);
      ps0 += s[nt][0] + s[nt][1];
      ps1 += s[nt][2] + s[nt][3];
    }
    l0 = l0 * c0 + ps0;
    l1 = l1 * c1 + ps1;
#pragma unroll
    for (int i = 0; i < DH / 8; ++i) {
      acc_o[i][0] *= c0; acc_o[i][1] *= c0; acc_o[i][2] *= c1; acc_o[i][3] *= c1;
    }
    uint32_t pf[4][4];
    acc_to_a_frags(s, pf);
    mma_p_b<DH>(acc_o, pf, Vs, kb * BLK);
  }
  l0 += __shfl_xor_sync(0xffffffffu, l0, 1); l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
  l1 += __shfl_xor_sync(0xffffffffu, l1, 1); l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
  const float i0 = 1.f / l0, i1 = 1.f / l1;
  if (r0 < S) {
    bf16 *orow = o + ((int64_t)seq * S + r0) * da + h * DH;
#pragma unroll
    for (int nt = 0; nt < DH / 8; ++nt)
      *reinterpret_cast<uint32_t *>(orow + nt * 8 + 2 * t) = pack_bf16(acc_o[nt][0] * i0, acc_o[nt][1] * i0);
    if (t == 0) lse[((int64_t)seq * A + h) * S + r0] = m0 * scale + logf(l0);
  }
  if (r1 < S) {
    bf16 *orow = o + ((int64_t)seq * S + r1) * da + h * DH;
#pragma unroll
    for (int nt = 0; nt < DH / 8; ++nt)
      *reinterpret_cast<uint32_t *>(orow + nt * 8 + 2 * t) = pack_bf16(acc_o[nt][2] * i1, acc_o[nt][3] * i1);
    if (t == 0) lse[((int64_t)seq * A + h) * S + r1] = m1 * scale + logf(l1);
  }
}

// ---------------------------------------------------------------------------------------------
// backward, part 1: D = rowsum(dO * O) and dq, one CTA per 64 query rows
// ---------------------------------------------------------------------------------------------
template <int DH>
__global__ void __launch_bounds__(NWARP * 32)
attn_bwd_dq_mma_kernel(const bf16 *__restrict__ qkv, const bf16 *__restrict__ o, const bf16 *__restrict__ d_o,
                       const float *__restrict__ lse, bf16 *__restrict__ dqkv, float *__restrict__ dvec, int S,
                       int A, int causal, float scale) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ float Dsm[BLK];
  const int da = A * DH, seq = blockIdx.y / A, h = blockIdx.y % A;
  const int q0 = blockIdx.x * BLK;
  const int nk = causal ? min(S, q0 + BLK) : S;
  const int nkb = (nk + BLK - 1) / BLK;
  const uint32_t Qs = smem_u32(smem), dOs = Qs + BLK * Tile<DH>::ROWB, Ks = dOs + BLK * Tile<DH>::ROWB,
                 Vs = Ks + nkb * BLK * Tile<DH>::ROWB;
  const bf16 *base = qkv + (int64_t)seq * S * 3 * da + h * DH;
  const bf16 *dobase = d_o + (int64_t)seq * S * da + h * DH;
  const bf16 *obase = o + (int64_t)seq * S * da + h * DH;
  load_tile<DH>(Qs, base, 3 * da, q0, BLK, S);
  load_tile<DH>(dOs, dobase, da, q0, BLK, S);
  load_tile<DH>(Ks, base + da, 3 * da, 0, nkb * BLK, nk);
  load_tile<DH>(Vs, base + 2 * da, 3 * da, 0, nkb * BLK, nk);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int64_t sbase = ((int64_t)seq * A + h) * S;
  // D_i = sum_c dO[i,c] * O[i,c]: two lanes per row, every load of the warp's 16 rows in flight at once
  {
    const int rr = lane >> 1, hf = lane & 1;
    const int row = q0 + warp * 16 + rr;
    float acc = 0.f;
    if (row < S) {
      const uint4 *pa = reinterpret_cast<const uint4 *>(dobase + (int64_t)row * da + hf * (DH / 2));
      const uint4 *pb = reinterpret_cast<const uint4 *>(obase + (int64_t)row * da + hf * (DH / 2));
      uint4 ua[DH / 16], ub[DH / 16];
#pragma unroll
      for (int i = 0; i < DH / 16; ++i) { ua[i] = __ldg(pa + i); ub[i] = __ldg(pb + i); }
#pragma unroll
      for (int i = 0; i < DH / 16; ++i) {
        const __nv_bfloat162 *ha = reinterpret_cast<const __nv_bfloat162 *>(&ua[i]);
        const __nv_bfloat162 *hb = reinterpret_cast<const __nv_bfloat162 *>(&ub[i]);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          float2 a = __bfloat1622float2(ha[e]), b = __bfloat1622float2(hb[e]);
          acc += a.x * b.x + a.y * b.y;
        }
      }
    }
    acc += __shfl_xor_sync(0xffffffffu, acc, 1);
    if (hf == 0) {
      Dsm[warp * 16 + rr] = acc;
      if (row < S) dvec[sbase + row] = acc;
    }
  }
  cp_async_wait_all();
  __syncthreads();

  uint32_t qf[DH / 16][4], dof[DH / 16][4];
  load_a_frags<DH>(Qs, warp * 16, qf);
  load_a_frags<DH>(dOs, warp * 16, dof);
  const int r0 = q0 + warp * 16 + g, r1 = r0 + 8;
  const float sl2 = scale * LOG2E;
  const float L0 = (r0 < S ? lse[sbase + r0] : 0.f) * LOG2E, L1 = (r1 < S ? lse[sbase + r1] : 0.f) * LOG2E;
  const float D0 = Dsm[warp * 16 + g], D1 = Dsm[warp * 16 + g + 8];
  float acc_dq[DH / 8][4];
#pragma unroll
  for (int i = 0; i < DH / 8; ++i) acc_dq[i][0] = acc_dq[i][1] = acc_dq[i][2] = acc_dq[i][3] = 0.f;
  const int kb_end = causal ? min(nkb, (q0 + warp * 16 + 15) / BLK + 1) : nkb;
  for (int kb = 0; kb < kb_end; ++kb) {
    float s[8][4], dp[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f;
      dp[i][0] = dp[i][1] = dp[i][2] = dp[i][3] = 0.f;
    }
    mma_a_bT<DH>(s, qf, Ks, kb * BLK);
    mma_a_bT<DH>(dp, dof, Vs, kb * BLK);
#pragma unroll
    for (int nt = 0; nt < 8; ++nt)
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        int key = kb * BLK + nt * 8 + 2 * t + (e & 1);
        int row = (e & 2) ? r1 : r0;
        float p = (key >= nk || (causal && key > row)) ? 0.f : exp2f(s[nt][e] * sl2 - ((e & 2) ? L1 : L0));
        s[nt][e] = p * (dp[nt][e] - ((e & 2) ? D1 : D0));           // dS
      }
    uint32_t pf[4][4];
    acc_to_a_frags(s, pf);
    mma_p_b<DH>(acc_dq, pf, Ks, kb * BLK);
  }
  if (r0 < S) {
    bf16 *row = dqkv + ((int64_t)seq * S + r0) * 3 * da + h * DH;
#pragma unroll
    for (int nt = 0; nt < DH / 8; ++nt)
      *reinterpret_cast<uint32_t *>(row + nt * 8 + 2 * t) = pack_bf16(acc_dq[nt][0] * scale, acc_dq[nt][1] * scale);
  }
  if (r1 < S) {
    bf16 *row = dqkv + ((int64_t)seq * S + r1) * 3 * da + h * DH;
#pragma unroll
    for (int nt = 0; nt < DH / 8; ++nt)
      *reinterpret_cast<uint32_t *>(row + nt * 8 + 2 * t) = pack_bf16(acc_dq[nt][2] * scale, acc_dq[nt][3] * scale);
  }
}

// ---------------------------------------------------------------------------------------------
// backward, part 2: dk, dv, one CTA per 64 key rows; works on the transposed score tile
// S^T[key, query] = K Q^T so that P^T and dS^T are directly the A operands of dV += P^T dO, dK += dS^T Q
// ---------------------------------------------------------------------------------------------
template <int DH>
__global__ void __launch_bounds__(NWARP * 32)
attn_bwd_dkv_mma_kernel(const bf16 *__restrict__ qkv, const bf16 *__restrict__ d_o, const float *__restrict__ lse,
                        const float *__restrict__ dvec, bf16 *__restrict__ dqkv, int S, int A, int causal,
                        float scale) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int da = A * DH, seq = blockIdx.y / A, h = blockIdx.y % A;
  const int j0 = blockIdx.x * BLK;
  const int ib0 = causal ? j0 / BLK : 0;                    // first query block that can see these keys
  const int nqb = (S + BLK - 1) / BLK - ib0;
  const uint32_t Ks = smem_u32(smem), Vs = Ks + BLK * Tile<DH>::ROWB, Qs = Vs + BLK * Tile<DH>::ROWB,
                 dOs = Qs + nqb * BLK * Tile<DH>::ROWB;
  float *Ls = reinterpret_cast<float *>(smem + (size_t)(2 * BLK + 2 * nqb * BLK) * Tile<DH>::ROWB);
  float *Ds = Ls + nqb * BLK;
  const bf16 *base = qkv + (int64_t)seq * S * 3 * da + h * DH;
  const bf16 *dobase = d_o + (int64_t)seq * S * da + h * DH;
  load_tile<DH>(Ks, base + da, 3 * da, j0, BLK, S);
  load_tile<DH>(Vs, base + 2 * da, 3 * da, j0, BLK, S);
  load_tile<DH>(Qs, base, 3 * da, ib0 * BLK, nqb * BLK, S);
  load_tile<DH>(dOs, dobase, da, ib0 * BLK, nqb * BLK, S);
  const int64_t sbase = ((int64_t)seq * A + h) * S;
  for (int i = threadIdx.x; i < nqb * BLK; i += blockDim.x) {
    int q = ib0 * BLK + i;
    Ls[i] = q < S ? lse[sbase + q] * LOG2E : 0.f;
    Ds[i] = q < S ? dvec[sbase + q] : 0.f;
  }
  cp_async_wait_all();
  __syncthreads();

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  uint32_t kf[DH / 16][4], vf[DH / 16][4];
  load_a_frags<DH>(Ks, warp * 16, kf);
  load_a_frags<DH>(Vs, warp * 16, vf);
  const int k0 = j0 + warp * 16 + g, k1 = k0 + 8;
  const float sl2 = scale * LOG2E;
  float acc_dk[DH / 8][4], acc_dv[DH / 8][4];
#pragma unroll
  for (int i = 0; i < DH / 8; ++i) {
    acc_dk[i][0] = acc_dk[i][1] = acc_dk[i][2] = acc_dk[i][3] = 0.f;
    acc_dv[i][0] = acc_dv[i][1] = acc_dv[i][2] = acc_dv[i][3] = 0.f;
  }
  for (int ib = 0; ib < nqb; ++ib) {
    float s[8][4], dp[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f;
      dp[i][0] = dp[i][1] = dp[i][2] = dp[i][3] = 0.f;
    }
    mma_a_bT<DH>(s, kf, Qs, ib * BLK);          // S^T = K Q^T
    mma_a_bT<DH>(dp, vf, dOs, ib * BLK);        // dP^T = V dO^T
    uint32_t pf[4][4], dsf[4][4];
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) {
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        int qi = ib * BLK + nt * 8 + 2 * t + (e & 1);          // index into Ls / Ds
        int q = ib0 * BLK + qi;
        int key = (e & 2) ? k1 : k0;
        float p = (q >= S || (causal && q < key)) ? 0.f : exp2f(s[nt][e] * sl2 - Ls[qi]);
        s[nt][e] = p;
        dp[nt][e] = p * (dp[nt][e] - Ds[qi]);
      }
    }
    acc_to_a_frags(s, pf);
    acc_to_a_frags(dp, dsf);
    mma_p_b<DH>(acc_dv, pf, dOs, ib * BLK);     // dV += P^T dO
    mma_p_b<DH>(acc_dk, dsf, Qs, ib * BLK);     // dK += dS^T Q
  }
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    int key = half ? k1 : k0;
    if (key < S) {
      bf16 *dk = dqkv + ((int64_t)seq * S + key) * 3 * da + da + h * DH;
      bf16 *dv = dk + da;
#pragma unroll
      for (int nt = 0; nt < DH / 8; ++nt) {
        *reinterpret_cast<uint32_t *>(dk + nt * 8 + 2 * t) =
            pack_bf16(acc_dk[nt][2 * half] * scale, acc_dk[nt][2 * half + 1] * scale);
        *reinterpret_cast<uint32_t *>(dv + nt * 8 + 2 * t) = pack_bf16(acc_dv[nt][2 * half], acc_dv[nt][2 * half + 1]);
      }
    }
  }
}

template <typename K>
static cudaError_t set_smem(K kernel, size_t bytes) {
  if (bytes > 227 * 1024) return cudaErrorInvalidValue;
  if (bytes > 48 * 1024) return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  return cudaSuccess;
}

template <int DH>
static cudaError_t fwd(const Ctx &c, const bf16 *qkv, bf16 *o, float *lse, int n_seq, int S, int A, int causal) {
  int nb = (S + BLK - 1) / BLK;
  size_t smem = (size_t)(BLK + 2 * nb * BLK) * DH * 2;
  cudaError_t e = set_smem(attn_fwd_mma_kernel<DH>, smem);
  if (e != cudaSuccess) return e;
  dim3 grid(nb, n_seq * A);
  attn_fwd_mma_kernel<DH><<<grid, NWARP * 32, smem, c.stream>>>(qkv, o, lse, S, A, causal, 1.f / sqrtf((float)DH));
  GP_LAUNCH_CHECK(c);
}

template <int DH>
static cudaError_t bwd(const Ctx &c, const bf16 *qkv, const bf16 *o, const bf16 *d_o, const float *lse, bf16 *dqkv,
                       float *dvec, int n_seq, int S, int A, int causal) {
  int nb = (S + BLK - 1) / BLK;
  float scale = 1.f / sqrtf((float)DH);
  size_t s1 = (size_t)(2 * BLK + 2 * nb * BLK) * DH * 2;
  size_t s2 = (size_t)(2 * BLK + 2 * nb * BLK) * DH * 2 + (size_t)2 * nb * BLK * 4;
  cudaError_t e = set_smem(attn_bwd_dq_mma_kernel<DH>, s1);
  if (e != cudaSuccess) return e;
  e = set_smem(attn_bwd_dkv_mma_kernel<DH>, s2);
  if (e != cudaSuccess) return e;
  dim3 grid(nb, n_seq * A);
  attn_bwd_dq_mma_kernel<DH><<<grid, NWARP * 32, s1, c.stream>>>(qkv, o, d_o, lse, dqkv, dvec, S, A, causal, scale);
  if (c.launches) ++*c.launches;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  attn_bwd_dkv_mma_kernel<DH><<<grid, NWARP * 32, s2, c.stream>>>(qkv, d_o, lse, dvec, dqkv, S, A, causal, scale);
  GP_LAUNCH_CHECK(c);
}

}  // namespace fa

// bf16, d_head 32 or 64, whole head resident in shared memory, 16-byte aligned rows
bool attn_mma_supported(int dt, int S, int A, int dh) {
  if (dt != GP_BF16 || (dh != 32 && dh != 64)) return false;
  int nb = (S + fa::BLK - 1) / fa::BLK;
  size_t s2 = (size_t)(2 * fa::BLK + 2 * nb * fa::BLK) * dh * 2 + (size_t)2 * nb * fa::BLK * 4;
  return s2 <= 200 * 1024 && (A * dh) % 8 == 0;
}

cudaError_t attn_fwd_mma(const Ctx &c, const void *qkv, void *o, float *lse, int n_seq, int S, int A, int dh, int causal) {
  if (n_seq == 0) return cudaSuccess;
  if (dh == 64) return fa::fwd<64>(c, (const bf16 *)qkv, (bf16 *)o, lse, n_seq, S, A, causal);
  return fa::fwd<32>(c, (const bf16 *)qkv, (bf16 *)o, lse, n_seq, S, A, causal);
}

cudaError_t attn_bwd_mma(const Ctx &c, const void *qkv, const void *o, const void *d_o, const float *lse, void *dqkv,
                         float *dvec, int n_seq, int S, int A, int dh, int causal) {
  if (n_seq == 0) return cudaSuccess;
  if (dh == 64)
    return fa::bwd<64>(c, (const bf16 *)qkv, (const bf16 *)o, (const bf16 *)d_o, lse, (bf16 *)dqkv, dvec, n_seq, S, A, causal);
  return fa::bwd<32>(c, (const bf16 *)qkv, (const bf16 *)o, (const bf16 *)d_o, lse, (bf16 *)dqkv, dvec, n_seq, S, A, causal);
}

}  // namespace gp

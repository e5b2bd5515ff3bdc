// gemm_simt.cu - fp32-FMA GEMM (no tensor cores, TF32 off) for the fp32 parity configuration and
// for shapes the tcgen05 kernel does not take (ragged / unaligned).  64x64x16 tiles, 256 threads,
// 4x4 outputs per thread, any transposition via index arithmetic, bounds-checked edges.
// The same fused epilogue as the tensor-core kernel (ops.h): +bias, ReLU, bit-packed ReLU mask
// in / out, +residual, fp32 accumulate.  Bound: ALU (fp32 FMA); only correctness matters for this path.
#include "common.cuh"

namespace gp {

constexpr int SG_BM = 64, SG_BN = 64, SG_BK = 16;

template <typename T>
__global__ void __launch_bounds__(256)
gemm_simt_kernel(GemmArgs g) {
  __shared__ float As[SG_BK][SG_BM + 4];
  __shared__ float Bs[SG_BK][SG_BN + 4];
  const T *A = (const T *)g.A;
  const T *B = (const T *)g.B;
  int tid = threadIdx.x;
  int m0 = blockIdx.y * SG_BM, n0 = blockIdx.x * SG_BN;
  int ty = tid >> 4, tx = tid & 15;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

  for (int k0 = 0; k0 < g.K; k0 += SG_BK) {
    // ---- A tile: As[k][m] ----
    if (!g.transA) {                    // global [M,K], k contiguous: threads run along k
      int kk = tid & 15, mm = tid >> 4;
#pragma unroll
      for (int p = 0; p < 4; ++p) {
        int m = m0 + mm + 16 * p, k = k0 + kk;
        As[kk][mm + 16 * p] = (m < g.M && k < g.K) ? to_f<T>(A[(int64_t)m * g.lda + k]) : 0.f;
      }
    } else {                            // global [K,M], m contiguous: threads run along m
      int mm = tid & 63, kk = tid >> 6;
#pragma unroll
      for (int p = 0; p < 4; ++p) {
        int m = m0 + mm, k = k0 + kk + 4 * p;
        As[kk + 4 * p][mm] = (m < g.M && k < g.K) ? to_f<T>(A[(int64_t)k * g.lda + m]) : 0.f;
      }
    }
    // ---- B tile: Bs[k][n] ----
    if (!g.transB) {                    // global [K,N], n contiguous
      int nn = tid & 63, kk = tid >> 6;
#pragma unroll
      for (int p = 0; p < 4; ++p) {
        int n = n0 + nn, k = k0 + kk + 4 * p;
        Bs[kk + 4 * p][nn] = (n < g.N && k < g.K) ? to_f<T>(B[(int64_t)k * g.ldb + n]) : 0.f;
      }
    } else {                            // global [N,K], k contiguous
      int kk = tid & 15, nn = tid >> 4;
#pragma unroll
      for (int p = 0; p < 4; ++p) {
        int n = n0 + nn + 16 * p, k = k0 + kk;
        Bs[kk][nn + 16 * p] = (n < g.N && k < g.K) ? to_f<T>(B[(int64_t)n * g.ldb + k]) : 0.f;
      }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < SG_BK; ++k) {
      float4 a = *reinterpret_cast<const float4 *>(&As[k][ty * 4]);
      float4 b = *reinterpret_cast<const float4 *>(&Bs[k][tx * 4]);
      float av[4] = {a.x, a.y, a.z, a.w}, bv[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
    }
    __syncthreads();
  }

  const uint32_t *maskbits = (const uint32_t *)g.mask;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    int m = m0 + ty * 4 + i;
    uint32_t nib = 0;                                 // [stored value > 0] of this thread's 4 columns
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int n = n0 + tx * 4 + j;
      if (m >= g.M || n >= g.N) continue;
      float v = acc[i][j];
      if (g.flags & EPI_BIAS) v += g.bias[n];
      if (g.flags & EPI_RELU) v = fmaxf(v, 0.f);
      if (g.flags & EPI_MASK) v = ((maskbits[(int64_t)m * g.ldmask + (n >> 5)] >> (n & 31)) & 1u) ? v : 0.f;
      if (g.flags & EPI_RESID) v += g.resid[(int64_t)m * g.ldc + n];
      int64_t ci = (int64_t)m * g.ldc + n;
      if (g.flags & EPI_ACCUM) {
        float *C = (float *)g.C;
        C[ci] += v;
      } else if (g.flags & EPI_OUT_F32) {
        ((float *)g.C)[ci] = v;
      } else {
        T s = from_f<T>(v);
        ((T *)g.C)[ci] = s;
        v = to_f<T>(s);
      }
      nib |= (v > 0.f ? 1u : 0u) << j;
    }
    if (g.flags & EPI_BITS_OUT) {
      // the 8 threads tx & ~7 .. tx | 7 of a row hold one 32-bit word (consecutive lanes of a warp)
      uint32_t w = nib << (4 * (tx & 7));
      w |= __shfl_xor_sync(0xffffffffu, w, 1);
      w |= __shfl_xor_sync(0xffffffffu, w, 2);
      w |= __shfl_xor_sync(0xffffffffu, w, 4);
      int n_word = n0 + (tx & ~7) * 4;
      if ((tx & 7) == 0 && m < g.M && n_word < g.N) ((uint32_t *)g.mask)[(int64_t)m * g.ldmask + (n_word >> 5)] = w;
    }
  }
}

cudaError_t gemm_simt(const Ctx &c, int dt, const GemmArgs &a) {
  if (a.M == 0 || a.N == 0) return cudaSuccess;
  dim3 grid((a.N + SG_BN - 1) / SG_BN, (a.M + SG_BM - 1) / SG_BM);
  if (dt == GP_BF16) gemm_simt_kernel<bf16><<<grid, 256, 0, c.stream>>>(a);
  else gemm_simt_kernel<float><<<grid, 256, 0, c.stream>>>(a);
  GP_LAUNCH_CHECK(c);
}

}  // namespace gp

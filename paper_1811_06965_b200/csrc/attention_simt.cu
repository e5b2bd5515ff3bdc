// attention_simt.cu - flash-style attention with warp-level online softmax, fp32-FMA version.
// One warp owns one query row (forward, dq) or one key row (dk/dv); the head's K/V (or Q/dO)
// live in shared memory as fp32 with a padded row stride (dh+1) so both the lane-per-row and the
// lane-per-column access patterns are bank-conflict free.  Scores are never written to HBM; the
// forward saves the log-sum-exp per row, the backward recomputes p = exp(s - lse)
// (SURVEY 8(a) a7, a16).  Used by the fp32 parity path and as the reference for the tensor-core
// attention kernels.  Deterministic: no atomics.
#include <math.h>

#include "common.cuh"

namespace gp {

constexpr int AT_WARPS = 8;
constexpr int AT_ROWS = 64;       // rows of the sequence handled by one block

template <typename T>
__device__ __forceinline__ void load_head_rows(float *dst, const T *src, int64_t ld, int n_rows,
                                               int dh) {
  // dst[r*(dh+1) + c] = src[r*ld + c]
  for (int i = threadIdx.x; i < n_rows * dh; i += blockDim.x) {
    int r = i / dh, c = i - r * dh;
    dst[r * (dh + 1) + c] = to_f<T>(src[(int64_t)r * ld + c]);
  }
}

template <typename T, int DH>
__global__ void __launch_bounds__(AT_WARPS * 32)
attn_fwd_simt_kernel(const T *__restrict__ qkv, T *__restrict__ o, float *__restrict__ lse, int S,
                     int A, int causal, float scale) {
  constexpr int NU = (DH + 31) / 32;
  extern __shared__ float sm[];
  int da = A * DH;
  int seq = blockIdx.x / A, h = blockIdx.x % A;
  int r0 = blockIdx.y * AT_ROWS;
  int r1 = min(S, r0 + AT_ROWS);
  int nk_block = causal ? r1 : S;                   // keys this block can need
  float *Ks = sm, *Vs = sm + (size_t)S * (DH + 1), *qs = Vs + (size_t)S * (DH + 1);
  const T *base = qkv + (int64_t)seq * S * 3 * da + h * DH;
  load_head_rows<T>(Ks, base + da, 3 * da, nk_block, DH);
  load_head_rows<T>(Vs, base + 2 * da, 3 * da, nk_block, DH);
  __syncthreads();
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  float *q = qs + w * DH;
  for (int i = r0 + w; i < r1; i += AT_WARPS) {
    __syncwarp();
    for (int c = lane; c < DH; c += 32) q[c] = to_f<T>(base[(int64_t)i * 3 * da + c]) * scale;
    __syncwarp();
    int nk = causal ? i + 1 : S;
    float m = -INFINITY, l = 0.f, acc[NU];
#pragma unroll
    for (int u = 0; u < NU; ++u) acc[u] = 0.f;
    for (int jb = 0; jb < nk; jb += 32) {
      int j = jb + lane;
      float s = -INFINITY;
      if (j < nk) {
        s = 0.f;
        const float *kr = Ks + j * (DH + 1);
#pragma unroll 8
        for (int c = 0; c < DH; ++c) s = fmaf(q[c], kr[c], s);
      }
      float mnew = fmaxf(m, warp_max(s));
      float p = j < nk ? expf(s - mnew) : 0.f;
      float corr = expf(m - mnew);
      l = l * corr + warp_sum(p);
#pragma unroll
      for (int u = 0; u < NU; ++u) acc[u] *= corr;
      int jn = min(32, nk - jb);
      for (int jj = 0; jj < jn; ++jj) {
        float pj = __shfl_sync(0xffffffffu, p, jj);
        const float *vr = Vs + (jb + jj) * (DH + 1);
#pragma unroll
        for (int u = 0; u < NU; ++u) {
          int c = lane + 32 * u;
          if (c < DH) acc[u] = fmaf(pj, vr[c], acc[u]);
        }
      }
      m = mnew;
    }
    float inv = 1.f / l;
    T *orow = o + ((int64_t)seq * S + i) * da + h * DH;
#pragma unroll
    for (int u = 0; u < NU; ++u) {
      int c = lane + 32 * u;
      if (c < DH) orow[c] = from_f<T>(acc[u] * inv);
    }
    if (lane == 0) lse[((int64_t)seq * A + h) * S + i] = m + logf(l);
  }
}

// dq and the D = rowsum(dO * O) pre-pass, one warp per query row
template <typename T, int DH>
__global__ void __launch_bounds__(AT_WARPS * 32)
attn_bwd_dq_simt_kernel(const T *__restrict__ qkv, const T *__restrict__ o, const T *__restrict__ d_o,
                        const float *__restrict__ lse, T *__restrict__ dqkv, float *__restrict__ dvec,
                        int S, int A, int causal, float scale) {
  constexpr int NU = (DH + 31) / 32;
  extern __shared__ float sm[];
  int da = A * DH;
  int seq = blockIdx.x / A, h = blockIdx.x % A;
  int r0 = blockIdx.y * AT_ROWS;
  int r1 = min(S, r0 + AT_ROWS);
  int nk_block = causal ? r1 : S;
  float *Ks = sm, *Vs = sm + (size_t)S * (DH + 1), *qs = Vs + (size_t)S * (DH + 1);
  float *dos = qs + AT_WARPS * DH;
  const T *base = qkv + (int64_t)seq * S * 3 * da + h * DH;
  load_head_rows<T>(Ks, base + da, 3 * da, nk_block, DH);
  load_head_rows<T>(Vs, base + 2 * da, 3 * da, nk_block, DH);
  __syncthreads();
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  float *q = qs + w * DH, *dor = dos + w * DH;
  for (int i = r0 + w; i < r1; i += AT_WARPS) {
    __syncwarp();
    const T *orow = o + ((int64_t)seq * S + i) * da + h * DH;
    const T *dorow = d_o + ((int64_t)seq * S + i) * da + h * DH;
    float dsum = 0.f;
    for (int c = lane; c < DH; c += 32) {
      q[c] = to_f<T>(base[(int64_t)i * 3 * da + c]) * scale;
      float dv = to_f<T>(dorow[c]);
      dor[c] = dv;
      dsum += dv * to_f<T>(orow[c]);
    }
    float D = warp_sum(dsum);
    __syncwarp();
    int64_t sidx = ((int64_t)seq * A + h) * S + i;
    float L = lse[sidx];
    if (lane == 0) dvec[sidx] = D;
    int nk = causal ? i + 1 : S;
    float acc[NU];
#pragma unroll
    for (int u = 0; u < NU; ++u) acc[u] = 0.f;
    for (int jb = 0; jb < nk; jb += 32) {
      int j = jb + lane;
      float ds = 0.f;
      if (j < nk) {
        float s = 0.f, dp = 0.f;
        const float *kr = Ks + j * (DH + 1), *vr = Vs + j * (DH + 1);
#pragma unroll 8
        for (int c = 0; c < DH; ++c) {
          s = fmaf(q[c], kr[c], s);
          dp = fmaf(dor[c], vr[c], dp);
        }
        ds = expf(s - L) * (dp - D);
      }
      int jn = min(32, nk - jb);
      for (int jj = 0; jj < jn; ++jj) {
        float dj = __shfl_sync(0xffffffffu, ds, jj);
        const float *kr = Ks + (jb + jj) * (DH + 1);
#pragma unroll
        for (int u = 0; u < NU; ++u) {
          int c = lane + 32 * u;
          if (c < DH) acc[u] = fmaf(dj, kr[c], acc[u]);
        }
      }
    }
    T *dq = dqkv + ((int64_t)seq * S + i) * 3 * da + h * DH;
#pragma unroll
    for (int u = 0; u < NU; ++u) {
      int c = lane + 32 * u;
      if (c < DH) dq[c] = from_f<T>(acc[u] * scale);
    }
  }
}

// dk, dv: one warp per key row; Q and dO of the head in shared memory
template <typename T, int DH>
__global__ void __launch_bounds__(AT_WARPS * 32)
attn_bwd_dkv_simt_kernel(const T *__restrict__ qkv, const T *__restrict__ d_o,
                         const float *__restrict__ lse, const float *__restrict__ dvec,
                         T *__restrict__ dqkv, int S, int A, int causal, float scale) {
  constexpr int NU = (DH + 31) / 32;
  extern __shared__ float sm[];
  int da = A * DH;
  int seq = blockIdx.x / A, h = blockIdx.x % A;
  int r0 = blockIdx.y * AT_ROWS;
  int r1 = min(S, r0 + AT_ROWS);
  int i_lo = causal ? r0 : 0;                        // queries that can see these keys
  float *Qs = sm, *dOs = sm + (size_t)S * (DH + 1), *ks = dOs + (size_t)S * (DH + 1);
  float *vs = ks + AT_WARPS * DH, *Ls = vs + AT_WARPS * DH, *Ds = Ls + S;
  const T *base = qkv + (int64_t)seq * S * 3 * da + h * DH;
  const T *dobase = d_o + (int64_t)seq * S * da + h * DH;
  load_head_rows<T>(Qs + (size_t)i_lo * (DH + 1), base + (int64_t)i_lo * 3 * da, 3 * da, S - i_lo, DH);
  load_head_rows<T>(dOs + (size_t)i_lo * (DH + 1), dobase + (int64_t)i_lo * da, da, S - i_lo, DH);
  for (int i = i_lo + threadIdx.x; i < S; i += blockDim.x) {
    int64_t sidx = ((int64_t)seq * A + h) * S + i;
    Ls[i] = lse[sidx];
    Ds[i] = dvec[sidx];
  }
  __syncthreads();
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  float *kk = ks + w * DH, *vv = vs + w * DH;
  for (int j = r0 + w; j < r1; j += AT_WARPS) {
    __syncwarp();
    for (int c = lane; c < DH; c += 32) {
      kk[c] = to_f<T>(base[(int64_t)j * 3 * da + da + c]) * scale;
      vv[c] = to_f<T>(base[(int64_t)j * 3 * da + 2 * da + c]);
    }
    __syncwarp();
    float adk[NU], adv[NU];
#pragma unroll
    for (int u = 0; u < NU; ++u) adk[u] = adv[u] = 0.f;
    int ib0 = causal ? (j / 32) * 32 : 0;
    for (int ib = ib0; ib < S; ib += 32) {
      int i = ib + lane;
      float p = 0.f, ds = 0.f;
      if (i < S && (!causal || i >= j)) {
        float s = 0.f, dp = 0.f;
        const float *qr = Qs + i * (DH + 1), *dr = dOs + i * (DH + 1);
#pragma unroll 8
        for (int c = 0; c < DH; ++c) {
          s = fmaf(qr[c], kk[c], s);
          dp = fmaf(dr[c], vv[c], dp);
        }
        p = expf(s - Ls[i]);
        ds = p * (dp - Ds[i]);
      }
      int in = min(32, S - ib);
      for (int ii = 0; ii < in; ++ii) {
        float pi = __shfl_sync(0xffffffffu, p, ii);
        float di = __shfl_sync(0xffffffffu, ds, ii);
        const float *qr = Qs + (ib + ii) * (DH + 1), *dr = dOs + (ib + ii) * (DH + 1);
#pragma unroll
        for (int u = 0; u < NU; ++u) {
          int c = lane + 32 * u;
          if (c < DH) {
            adv[u] = fmaf(pi, dr[c], adv[u]);
            adk[u] = fmaf(di, qr[c], adk[u]);
          }
        }
      }
    }
    T *dk = dqkv + ((int64_t)seq * S + j) * 3 * da + da + h * DH;
    T *dv = dk + da;
#pragma unroll
    for (int u = 0; u < NU; ++u) {
      int c = lane + 32 * u;
      if (c < DH) {
        dk[c] = from_f<T>(adk[u] * scale);
        dv[c] = from_f<T>(adv[u]);
      }
    }
  }
}

static size_t attn_smem_fwd(int S, int dh) { return ((size_t)2 * S * (dh + 1) + AT_WARPS * dh) * 4; }
static size_t attn_smem_dq(int S, int dh) { return ((size_t)2 * S * (dh + 1) + 2 * AT_WARPS * dh) * 4; }
static size_t attn_smem_dkv(int S, int dh) {
  return ((size_t)2 * S * (dh + 1) + 2 * AT_WARPS * dh + 2 * S) * 4;
}

template <typename K>
static cudaError_t set_smem(K kernel, size_t bytes) {
  if (bytes > 227 * 1024) return cudaErrorInvalidValue;
  if (bytes > 48 * 1024)
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  return cudaSuccess;
}

template <typename T, int DH>
static cudaError_t attn_fwd_simt_t(const Ctx &c, const T *qkv, T *o, float *lse, int n_seq, int S,
                                   int A, int causal) {
  size_t smem = attn_smem_fwd(S, DH);
  cudaError_t e = set_smem(attn_fwd_simt_kernel<T, DH>, smem);
  if (e != cudaSuccess) return e;
  dim3 grid(n_seq * A, (S + AT_ROWS - 1) / AT_ROWS);
  attn_fwd_simt_kernel<T, DH><<<grid, AT_WARPS * 32, smem, c.stream>>>(qkv, o, lse, S, A, causal,
                                                                       1.f / sqrtf((float)DH));
  GP_LAUNCH_CHECK(c);
}

template <typename T, int DH>
static cudaError_t attn_bwd_simt_t(const Ctx &c, const T *qkv, const T *o, const T *d_o,
                                   const float *lse, T *dqkv, float *dvec, int n_seq, int S, int A,
                                   int causal) {
  float scale = 1.f / sqrtf((float)DH);
  dim3 grid(n_seq * A, (S + AT_ROWS - 1) / AT_ROWS);
  size_t s1 = attn_smem_dq(S, DH), s2 = attn_smem_dkv(S, DH);
  cudaError_t e = set_smem(attn_bwd_dq_simt_kernel<T, DH>, s1);
  if (e != cudaSuccess) return e;
  e = set_smem(attn_bwd_dkv_simt_kernel<T, DH>, s2);
  if (e != cudaSuccess) return e;
  attn_bwd_dq_simt_kernel<T, DH><<<grid, AT_WARPS * 32, s1, c.stream>>>(qkv, o, d_o, lse, dqkv, dvec,
                                                                        S, A, causal, scale);
  if (c.launches) ++*c.launches;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  attn_bwd_dkv_simt_kernel<T, DH><<<grid, AT_WARPS * 32, s2, c.stream>>>(qkv, d_o, lse, dvec, dqkv, S,
                                                                         A, causal, scale);
  GP_LAUNCH_CHECK(c);
}

#define GP_DH_SWITCH(dh, CALL)                 \
  switch (dh) {                                \
    case 16: { constexpr int DH = 16; CALL; }  \
    case 32: { constexpr int DH = 32; CALL; }  \
    case 64: { constexpr int DH = 64; CALL; }  \
    case 128: { constexpr int DH = 128; CALL; }\
    default: return cudaErrorInvalidValue;     \
  }

cudaError_t attn_fwd_simt(const Ctx &c, int dt, const void *qkv, void *o, float *lse, int n_seq,
                          int S, int A, int dh, int causal) {
  if (n_seq == 0) return cudaSuccess;
  if (dt == GP_BF16) {
    GP_DH_SWITCH(dh, return (attn_fwd_simt_t<bf16, DH>(c, (const bf16 *)qkv, (bf16 *)o, lse, n_seq, S, A, causal)));
  } else {
    GP_DH_SWITCH(dh, return (attn_fwd_simt_t<float, DH>(c, (const float *)qkv, (float *)o, lse, n_seq, S, A, causal)));
  }
}

cudaError_t attn_bwd_simt(const Ctx &c, int dt, const void *qkv, const void *o, const void *d_o,
                          const float *lse, void *dqkv, float *dvec, int n_seq, int S, int A, int dh,
                          int causal) {
  if (n_seq == 0) return cudaSuccess;
  if (dt == GP_BF16) {
    GP_DH_SWITCH(dh, return (attn_bwd_simt_t<bf16, DH>(c, (const bf16 *)qkv, (const bf16 *)o, (const bf16 *)d_o, lse, (bf16 *)dqkv, dvec, n_seq, S, A, causal)));
  } else {
    GP_DH_SWITCH(dh, return (attn_bwd_simt_t<float, DH>(c, (const float *)qkv, (const float *)o, (const float *)d_o, lse, (float *)dqkv, dvec, n_seq, S, A, causal)));
  }
}

}  // namespace gp

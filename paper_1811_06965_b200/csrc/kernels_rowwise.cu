// kernels_rowwise.cu - HBM-bound kernels of the hot path: embedding, fused pre-LayerNorm,
// LayerNorm backward (+ residual-gradient add, + lp operand copy, + dgamma/dbeta partials),
// bias-gradient column sums.  One warp owns one token row; the row lives in registers.
// Roofline: HBM; algorithmic bytes per token are listed there.
#include "common.cuh"

namespace gp {

// ---------------------------------------------------------------------------------------------
// embedding: x0[t,:] = E[tok[t],:] + PE[t mod S,:]          (reading A6)
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void embed_fwd_kernel(const int32_t *__restrict__ tok, const T *__restrict__ emb,
                                 const float *__restrict__ pe, float *__restrict__ x,
                                 int64_t n_tok, int S, int d4) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_tok * d4) return;
  int64_t t = i / d4;
  int c = (int)(i - t * d4) * 4;
  int d = d4 * 4;
  float4 e = load4(emb + (int64_t)tok[t] * d + c);
  float4 p = load4(pe + (int64_t)(t % S) * d + c);
  store4(x + t * d + c, make_float4(e.x + p.x, e.y + p.y, e.z + p.z, e.w + p.w));
}

__global__ void embed_bwd_kernel(const int32_t *__restrict__ tok, const float *__restrict__ dx,
                                 float *__restrict__ gemb, int64_t n_tok, int d) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_tok * d) return;
  int64_t t = i / d;
  int c = (int)(i - t * d);
  atomicAdd(gemb + (int64_t)tok[t] * d + c, dx[i]);      // dE[tok] += dx0 (order-free, A13)
}

// PE[t,2i] = sin(t / 10000^(2i/d)), PE[t,2i+1] = cos(...), evaluated in double, stored fp32
__global__ void positional_kernel(float *pe, int S, int d) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= S * d) return;
  int t = i / d, j = i % d;
  int i2 = j - (j & 1);
  double ang = (double)t / pow(10000.0, (double)i2 / (double)d);
  pe[i] = (float)((j & 1) ? cos(ang) : sin(ang));
}

cudaError_t embed_fwd(const Ctx &c, int dt, const int32_t *tok, const void *emb, const float *pe,
                      float *x, int64_t n_tok, int S, int d) {
  int64_t n = n_tok * (d / 4);
  if (n == 0) return cudaSuccess;
  unsigned grid = (unsigned)((n + 255) / 256);
  if (dt == GP_BF16)
    embed_fwd_kernel<bf16><<<grid, 256, 0, c.stream>>>(tok, (const bf16 *)emb, pe, x, n_tok, S, d / 4);
  else
    embed_fwd_kernel<float><<<grid, 256, 0, c.stream>>>(tok, (const float *)emb, pe, x, n_tok, S, d / 4);
  GP_LAUNCH_CHECK(c);
}

cudaError_t embed_bwd(const Ctx &c, const int32_t *tok, const float *dx, float *gemb,
                      int64_t n_tok, int d) {
  int64_t n = n_tok * d;
  if (n == 0) return cudaSuccess;
  embed_bwd_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(tok, dx, gemb, n_tok, d);
  GP_LAUNCH_CHECK(c);
}

cudaError_t positional_table(const Ctx &c, float *pe, int S, int d) {
  positional_kernel<<<(S * d + 255) / 256, 256, 0, c.stream>>>(pe, S, d);
  GP_LAUNCH_CHECK(c);
}

// ---------------------------------------------------------------------------------------------
// LayerNorm forward: one warp per row, row in registers (NV float4 per lane), two-pass variance
// ---------------------------------------------------------------------------------------------
template <typename T, int NV>
__global__ void __launch_bounds__(128)
ln_fwd_kernel(const float *__restrict__ x, const float *__restrict__ gamma,
              const float *__restrict__ beta, T *__restrict__ y, float *__restrict__ mean,
              float *__restrict__ rstd, int64_t n_tok, int d, float eps) {
  int lane = threadIdx.x & 31;
  int64_t row = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
  if (row >= n_tok) return;
  int d4 = d >> 2;
  const float *xr = x + row * d;
  float4 v[NV];
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int j = lane + 32 * i;
    v[i] = j < d4 ? load4(xr + 4 * j) : make_float4(0.f, 0.f, 0.f, 0.f);
    s += (v[i].x + v[i].y) + (v[i].z + v[i].w);
  }
  float mu = warp_sum(s) / (float)d;
  float q = 0.f;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int j = lane + 32 * i;
    if (j < d4) {
      float a = v[i].x - mu, b = v[i].y - mu, c2 = v[i].z - mu, e = v[i].w - mu;
      q += (a * a + b * b) + (c2 * c2 + e * e);
    }
  }
  float rs = rsqrtf(warp_sum(q) / (float)d + eps);
  if (lane == 0) {
    mean[row] = mu;
    rstd[row] = rs;
  }
  T *yr = y + row * d;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int j = lane + 32 * i;
    if (j < d4) {
      float4 g = load4(gamma + 4 * j), b = load4(beta + 4 * j);
      float4 o;
      o.x = (v[i].x - mu) * rs * g.x + b.x;
      o.y = (v[i].y - mu) * rs * g.y + b.y;
      o.z = (v[i].z - mu) * rs * g.z + b.z;
      o.w = (v[i].w - mu) * rs * g.w + b.w;
      store4(yr + 4 * j, o);
    }
  }
}

template <typename T>
static cudaError_t ln_fwd_t(const Ctx &c, const float *x, const float *gamma, const float *beta,
                            T *y, float *mean, float *rstd, int64_t n_tok, int d, float eps) {
  if (n_tok == 0) return cudaSuccess;
  unsigned grid = (unsigned)((n_tok + 3) / 4);
  int nv = (d / 4 + 31) / 32;
  if (nv <= 1)
    ln_fwd_kernel<T, 1><<<grid, 128, 0, c.stream>>>(x, gamma, beta, y, mean, rstd, n_tok, d, eps);
  else if (nv <= 8)
    ln_fwd_kernel<T, 8><<<grid, 128, 0, c.stream>>>(x, gamma, beta, y, mean, rstd, n_tok, d, eps);
  else if (nv <= 16)
    ln_fwd_kernel<T, 16><<<grid, 128, 0, c.stream>>>(x, gamma, beta, y, mean, rstd, n_tok, d, eps);
  else
    return cudaErrorInvalidValue;
  GP_LAUNCH_CHECK(c);
}

cudaError_t ln_fwd(const Ctx &c, int dt, const float *x, const float *gamma, const float *beta,
                   void *y, float *mean, float *rstd, int64_t n_tok, int d, float eps) {
  return dt == GP_BF16 ? ln_fwd_t<bf16>(c, x, gamma, beta, (bf16 *)y, mean, rstd, n_tok, d, eps)
                       : ln_fwd_t<float>(c, x, gamma, beta, (float *)y, mean, rstd, n_tok, d, eps);
}

// ---------------------------------------------------------------------------------------------
// LayerNorm backward.  dxhat = dy*gamma; dx = (dxhat - mean(dxhat) - xhat*mean(dxhat*xhat))*rstd
// dx_out = dres_in + dx (residual adds gradients); optional lp copy (the next GEMM's operand).
// dgamma/dbeta: each warp accumulates its rows in registers; per-block partials are written to
// `partials` [gridDim.x, 2, d] and summed by ln_bwd_reduce_kernel in a fixed order.
// ---------------------------------------------------------------------------------------------
template <typename T, int NV>
__global__ void __launch_bounds__(128)
ln_bwd_kernel(const T *__restrict__ dy, const float *__restrict__ x, const float *__restrict__ mean,
              const float *__restrict__ rstd, const float *__restrict__ gamma,
              const float *__restrict__ dres_in, float *__restrict__ dx_out,
              T *__restrict__ dx_out_lp, float *__restrict__ partials, int64_t n_tok, int d) {
  extern __shared__ float sm[];       // [4 warps][2][d]
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int d4 = d >> 2;
  float4 g[NV], ag[NV], ab[NV];
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int j = lane + 32 * i;
    g[i] = j < d4 ? load4(gamma + 4 * j) : make_float4(0.f, 0.f, 0.f, 0.f);
    ag[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    ab[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  for (int64_t row = (int64_t)blockIdx.x * 4 + w; row < n_tok; row += (int64_t)gridDim.x * 4) {
    float mu = mean[row], rs = rstd[row];
    float4 xh[NV], dh[NV];
    float s1 = 0.f, s2 = 0.f;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      int j = lane + 32 * i;
      if (j < d4) {
        float4 xv = load4(x + row * d + 4 * j);
        float4 dv = load4(dy + row * d + 4 * j);
        xh[i] = make_float4((xv.x - mu) * rs, (xv.y - mu) * rs, (xv.z - mu) * rs, (xv.w - mu) * rs);
        ag[i].x += dv.x * xh[i].x; ag[i].y += dv.y * xh[i].y;
        ag[i].z += dv.z * xh[i].z; ag[i].w += dv.w * xh[i].w;
        ab[i].x += dv.x; ab[i].y += dv.y; ab[i].z += dv.z; ab[i].w += dv.w;
        dh[i] = make_float4(dv.x * g[i].x, dv.y * g[i].y, dv.z * g[i].z, dv.w * g[i].w);
        s1 += (dh[i].x + dh[i].y) + (dh[i].z + dh[i].w);
        s2 += (dh[i].x * xh[i].x + dh[i].y * xh[i].y) + (dh[i].z * xh[i].z + dh[i].w * xh[i].w);
      } else {
        xh[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        dh[i] = xh[i];
      }
    }
    float m1 = warp_sum(s1) / (float)d, m2 = warp_sum(s2) / (float)d;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      int j = lane + 32 * i;
      if (j < d4) {
        float4 o;
        o.x = (dh[i].x - m1 - xh[i].x * m2) * rs;
        o.y = (dh[i].y - m1 - xh[i].y * m2) * rs;
        o.z = (dh[i].z - m1 - xh[i].z * m2) * rs;
        o.w = (dh[i].w - m1 - xh[i].w * m2) * rs;
        if (dres_in) {
          float4 r = load4(dres_in + row * d + 4 * j);
          o.x += r.x; o.y += r.y; o.z += r.z; o.w += r.w;
        }
        store4(dx_out + row * d + 4 * j, o);
        if (dx_out_lp) store4(dx_out_lp + row * d + 4 * j, o);
      }
    }
  }
  // cross-warp reduction of the dgamma/dbeta partials, fixed order w = 0..3
  float *mine = sm + (size_t)w * 2 * d;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int j = lane + 32 * i;
    if (j < d4) {
      store4(mine + 4 * j, ag[i]);
      store4(mine + d + 4 * j, ab[i]);
    }
  }
  __syncthreads();
  float *out = partials + (size_t)blockIdx.x * 2 * d;
  for (int i = threadIdx.x; i < 2 * d; i += blockDim.x)
    out[i] = (sm[i] + sm[2 * d + i]) + (sm[4 * d + i] + sm[6 * d + i]);
}

__global__ void ln_bwd_reduce_kernel(const float *__restrict__ partials, int n_part, int d,
                                     float *__restrict__ dgamma, float *__restrict__ dbeta) {
  // one warp per 32 columns; each lane sums a strided subset of the partial rows, fixed order
  __shared__ float red[8][33];
  int col = blockIdx.x * 32 + (threadIdx.x & 31);
  int which = blockIdx.y;
  int ry = threadIdx.x >> 5;                      // 8 row groups
  float s = 0.f;
  if (col < d)
    for (int r = ry; r < n_part; r += 8) s += partials[((size_t)r * 2 + which) * d + col];
  red[ry][threadIdx.x & 31] = s;
  __syncthreads();
  if (ry == 0 && col < d) {
    float t = 0.f;
#pragma unroll
    for (int r = 0; r < 8; ++r) t += red[r][threadIdx.x & 31];
    float *dst = which == 0 ? dgamma : dbeta;
    dst[col] += t;
  }
}

int ln_bwd_partial_rows(int sm_count) { return sm_count * 2; }

template <typename T>
static cudaError_t ln_bwd_t(const Ctx &c, const T *dy, const float *x, const float *mean,
                            const float *rstd, const float *gamma, const float *dres_in,
                            float *dx_out, T *dx_out_lp, float *partials, float *dgamma,
                            float *dbeta, int64_t n_tok, int d) {
  if (n_tok == 0) return cudaSuccess;
  int64_t want = (n_tok + 3) / 4;
  int grid = (int)(want < ln_bwd_partial_rows(c.sm_count) ? want : ln_bwd_partial_rows(c.sm_count));
  size_t smem = (size_t)4 * 2 * d * sizeof(float);
  int nv = (d / 4 + 31) / 32;
#define GP_LNB(NV_)                                                                               \
  do {                                                                                            \
    if (smem > 48 * 1024)                                                                         \
      cudaFuncSetAttribute(ln_bwd_kernel<T, NV_>, cudaFuncAttributeMaxDynamicSharedMemorySize,    \
                           (int)smem);                                                            \
    ln_bwd_kernel<T, NV_><<<grid, 128, smem, c.stream>>>(dy, x, mean, rstd, gamma, dres_in,       \
                                                         dx_out, dx_out_lp, partials, n_tok, d);  \
  } while (0)
  if (nv <= 1) GP_LNB(1);
  else if (nv <= 8) GP_LNB(8);
  else if (nv <= 16) GP_LNB(16);
  else return cudaErrorInvalidValue;
#undef GP_LNB
  if (c.launches) ++*c.launches;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  dim3 rg((d + 31) / 32, 2);
  ln_bwd_reduce_kernel<<<rg, 256, 0, c.stream>>>(partials, grid, d, dgamma, dbeta);
  GP_LAUNCH_CHECK(c);
}

cudaError_t ln_bwd(const Ctx &c, int dt, const void *dy, const float *x, const float *mean,
                   const float *rstd, const float *gamma, const float *dres_in, float *dx_out,
                   void *dx_out_lp, float *partials, float *dgamma, float *dbeta, int64_t n_tok,
                   int d) {
  return dt == GP_BF16
             ? ln_bwd_t<bf16>(c, (const bf16 *)dy, x, mean, rstd, gamma, dres_in, dx_out,
                              (bf16 *)dx_out_lp, partials, dgamma, dbeta, n_tok, d)
             : ln_bwd_t<float>(c, (const float *)dy, x, mean, rstd, gamma, dres_in, dx_out,
                               (float *)dx_out_lp, partials, dgamma, dbeta, n_tok, d);
}

// ---------------------------------------------------------------------------------------------
// bias gradient: out[n] += sum_t dy[t,n].  Block = 8 warps x 64 columns; warp w takes rows
// w, w+8, ...; lanes take two adjacent columns.  Fixed summation order (deterministic).
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256)
colsum_kernel(const T *__restrict__ dy, int64_t ld, float *__restrict__ out, int64_t n_tok, int n) {
  __shared__ float red[8][64];
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int col = blockIdx.x * 64 + lane * 2;
  float a = 0.f, b = 0.f;
  if (col + 1 < n) {
    for (int64_t r = w; r < n_tok; r += 8) {
      const T *p = dy + r * ld + col;
      a += to_f<T>(p[0]);
      b += to_f<T>(p[1]);
    }
  } else if (col < n) {
    for (int64_t r = w; r < n_tok; r += 8) a += to_f<T>(dy[r * ld + col]);
  }
  red[w][lane * 2] = a;
  red[w][lane * 2 + 1] = b;
  __syncthreads();
  if (threadIdx.x < 64) {
    int cidx = blockIdx.x * 64 + threadIdx.x;
    if (cidx < n) {
      float t = 0.f;
#pragma unroll
      for (int r = 0; r < 8; ++r) t += red[r][threadIdx.x];
      out[cidx] += t;
    }
  }
}

cudaError_t colsum_accum(const Ctx &c, int dt, const void *dy, int64_t ld, float *out,
                         int64_t n_tok, int n) {
  if (n == 0) return cudaSuccess;
  unsigned grid = (unsigned)((n + 63) / 64);
  if (dt == GP_BF16)
    colsum_kernel<bf16><<<grid, 256, 0, c.stream>>>((const bf16 *)dy, ld, out, n_tok, n);
  else
    colsum_kernel<float><<<grid, 256, 0, c.stream>>>((const float *)dy, ld, out, n_tok, n);
  GP_LAUNCH_CHECK(c);
}

template <typename T>
__global__ void cast_kernel(const float *__restrict__ src, T *__restrict__ dst, int64_t n4) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n4) store4(dst + 4 * i, load4(src + 4 * i));
}

cudaError_t cast_to_lp(const Ctx &c, int dt, const float *src, void *dst, int64_t n) {
  if (n == 0) return cudaSuccess;
  int64_t n4 = n / 4;                 // callers pass multiples of 4 (d % 4 == 0)
  unsigned grid = (unsigned)((n4 + 255) / 256);
  if (dt == GP_BF16) cast_kernel<bf16><<<grid, 256, 0, c.stream>>>(src, (bf16 *)dst, n4);
  else cast_kernel<float><<<grid, 256, 0, c.stream>>>(src, (float *)dst, n4);
  GP_LAUNCH_CHECK(c);
}

}  // namespace gp

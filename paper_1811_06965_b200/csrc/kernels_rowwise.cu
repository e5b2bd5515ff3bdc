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

// dE[tok[t]] += dx0[t], without atomics and in a fixed order: warp w of the grid owns the vocabulary rows v
// with v mod W == w (W = warps in the grid), scans all token ids 32 at a time and adds the rows of the
// tokens it owns in ascending t.  One owner per row + program order within a lane = a deterministic
// sum whatever the multiplicity of an id (the atomicAdd version was the last order-dependent kernel).
__global__ void __launch_bounds__(256)
embed_bwd_kernel(const int32_t *__restrict__ tok, const float *__restrict__ dx, float *__restrict__ gemb,
                 int64_t n_tok, int d) {
  const int lane = threadIdx.x & 31;
  const unsigned W = gridDim.x * (blockDim.x >> 5), w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int d4 = d >> 2;
  for (int64_t base = 0; base < n_tok; base += 32) {
    const int64_t t = base + lane;
    const int id = t < n_tok ? tok[t] : -1;
    unsigned mine = __ballot_sync(0xffffffffu, id >= 0 && (unsigned)id % W == w);
    while (mine) {
      const int src = __ffs(mine) - 1;
      mine &= mine - 1;
      const int v = __shfl_sync(0xffffffffu, id, src);
      const float *row = dx + (base + src) * d;
      float *dst = gemb + (int64_t)v * d;
      for (int j = lane; j < d4; j += 32) {
        float4 a = load4(dst + 4 * j), b = load4(row + 4 * j);
        store4(dst + 4 * j, make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w));
      }
    }
  }
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
  if (n_tok == 0 || d == 0) return cudaSuccess;
  if (d % 4) return cudaErrorInvalidValue;
  // ~one owned token per warp at T_mb = 2048; never more warps than tokens
  int64_t blocks = (n_tok + 7) / 8;
  if (blocks > 2 * (int64_t)c.sm_count) blocks = 2 * (int64_t)c.sm_count;
  embed_bwd_kernel<<<(unsigned)blocks, 256, 0, c.stream>>>(tok, dx, gemb, n_tok, d);
  GP_LAUNCH_CHECK(c);
}

cudaError_t positional_table(const Ctx &c, float *pe, int S, int d) {
  positional_kernel<<<(S * d + 255) / 256, 256, 0, c.stream>>>(pe, S, d);
  GP_LAUNCH_CHECK(c);
}

// ---------------------------------------------------------------------------------------------
// LayerNorm forward: one warp per row, row in registers (NV float4 per lane), two-pass variance.
// Fused residual: when resid_out != NULL the kernel also writes resid_out = x + resid_bias, the
// value the branch's output GEMM then accumulates into (x' = x + branch(LN(x)) + b, SURVEY 8(a)
// a5/a8, a9/a11): the GEMM epilogue becomes a TMA reduce-add and never reads x into the SM.
// ---------------------------------------------------------------------------------------------
template <typename T, int NV>
__global__ void __launch_bounds__(128)
ln_fwd_kernel(const float *__restrict__ x, const float *__restrict__ gamma,
              const float *__restrict__ beta, T *__restrict__ y, float *__restrict__ mean,
              float *__restrict__ rstd, const float *__restrict__ resid_bias, float *__restrict__ resid_out,
              int64_t n_tok, int d, float eps) {
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
      if (resid_out) {
        float4 rb = load4(resid_bias + 4 * j);
        store4(resid_out + row * d + 4 * j, make_float4(v[i].x + rb.x, v[i].y + rb.y, v[i].z + rb.z, v[i].w + rb.w));
      }
    }
  }
}

template <typename T>
static cudaError_t ln_fwd_t(const Ctx &c, const float *x, const float *gamma, const float *beta,
                            T *y, float *mean, float *rstd, const float *resid_bias, float *resid_out,
                            int64_t n_tok, int d, float eps) {
  if (n_tok == 0) return cudaSuccess;
  unsigned grid = (unsigned)((n_tok + 3) / 4);
  int nv = (d / 4 + 31) / 32;
  if (nv <= 1)
    ln_fwd_kernel<T, 1><<<grid, 128, 0, c.stream>>>(x, gamma, beta, y, mean, rstd, resid_bias, resid_out, n_tok, d, eps);
  else if (nv <= 8)
    ln_fwd_kernel<T, 8><<<grid, 128, 0, c.stream>>>(x, gamma, beta, y, mean, rstd, resid_bias, resid_out, n_tok, d, eps);
  else if (nv <= 16)
    ln_fwd_kernel<T, 16><<<grid, 128, 0, c.stream>>>(x, gamma, beta, y, mean, rstd, resid_bias, resid_out, n_tok, d, eps);
  else
    return cudaErrorInvalidValue;
  GP_LAUNCH_CHECK(c);
}

cudaError_t ln_fwd(const Ctx &c, int dt, const float *x, const float *gamma, const float *beta,
                   void *y, float *mean, float *rstd, const float *resid_bias, float *resid_out,
                   int64_t n_tok, int d, float eps) {
  if (resid_out && !resid_bias) return cudaErrorInvalidValue;
  return dt == GP_BF16 ? ln_fwd_t<bf16>(c, x, gamma, beta, (bf16 *)y, mean, rstd, resid_bias, resid_out, n_tok, d, eps)
                       : ln_fwd_t<float>(c, x, gamma, beta, (float *)y, mean, rstd, resid_bias, resid_out, n_tok, d, eps);
}

// ---------------------------------------------------------------------------------------------
// LayerNorm backward.  dxhat = dy*gamma; dx = (dxhat - mean(dxhat) - xhat*mean(dxhat*xhat))*rstd
// dx_out = dres_in + dx (residual adds gradients); optional lp copy (the next GEMM's operand).
// Fused reductions over the token axis, all in a fixed order (deterministic):
//   dgamma += sum_t dy*xhat, dbeta += sum_t dy, and optionally colsum_out += sum_t dx_out (the bias
//   gradient of the linear layer whose output gradient dx_out is: db_2 / db_o).
// One warp per row, WARPS rows per block pass, every load of a row (x, dy, incoming residual
// gradient) in flight at once: the kernel is one DRAM round trip deep.  Each warp leaves its row's
// three contribution vectors in its own shared-memory slot; the block sums the slots column-wise
// (thread t owns columns t, t + blockDim, ...), keeps the running sums in registers across passes
// and writes one partial row [3][d] per block; a second small kernel sums the partial rows.
// ---------------------------------------------------------------------------------------------
template <typename T, int NV, int WARPS>
__global__ void __launch_bounds__(WARPS * 32, 1)
ln_bwd_kernel(const T *__restrict__ dy, const float *__restrict__ x, const float *__restrict__ mean,
              const float *__restrict__ rstd, const float *__restrict__ gamma,
              const float *__restrict__ dres_in, float *__restrict__ dx_out,
              T *__restrict__ dx_out_lp, float *__restrict__ partials, int64_t n_tok, int d, int want_colsum) {
  extern __shared__ __align__(16) float red[];       // [WARPS][3][d]
  constexpr int NT = WARPS * 32;
  constexpr int NACC = (3 * 128 * NV + NT - 1) / NT; // columns of [3][d] per thread (d <= 128*NV)
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int d4 = d >> 2;
  float *slot = red + (size_t)w * 3 * d;
  float acc[NACC];
#pragma unroll
  for (int j = 0; j < NACC; ++j) acc[j] = 0.f;
  for (int64_t base = (int64_t)blockIdx.x * WARPS; base < n_tok; base += (int64_t)gridDim.x * WARPS) {
    const int64_t row = base + w;
    if (row < n_tok) {
      float4 xh[NV], dh[NV], dr[NV];
#pragma unroll
      for (int i = 0; i < NV; ++i) {
        const int j = lane + 32 * i;
        if (j < d4) {
          xh[i] = load4(x + row * d + 4 * j);
          dh[i] = load4(dy + row * d + 4 * j);
          dr[i] = dres_in ? load4(dres_in + row * d + 4 * j) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
      }
      const float mu = mean[row], rs = rstd[row];
      float s1 = 0.f, s2 = 0.f;
#pragma unroll
      for (int i = 0; i < NV; ++i) {
        const int j = lane + 32 * i;
        if (j < d4) {
          const float4 gv = load4(gamma + 4 * j);
          xh[i] = make_float4((xh[i].x - mu) * rs, (xh[i].y - mu) * rs, (xh[i].z - mu) * rs, (xh[i].w - mu) * rs);
          *reinterpret_cast<float4 *>(slot + 4 * j) =
              make_float4(dh[i].x * xh[i].x, dh[i].y * xh[i].y, dh[i].z * xh[i].z, dh[i].w * xh[i].w);
          *reinterpret_cast<float4 *>(slot + d + 4 * j) = dh[i];
          dh[i] = make_float4(dh[i].x * gv.x, dh[i].y * gv.y, dh[i].z * gv.z, dh[i].w * gv.w);
          s1 += (dh[i].x + dh[i].y) + (dh[i].z + dh[i].w);
          s2 += (dh[i].x * xh[i].x + dh[i].y * xh[i].y) + (dh[i].z * xh[i].z + dh[i].w * xh[i].w);
        }
      }
      const float m1 = warp_sum(s1) / (float)d, m2 = warp_sum(s2) / (float)d;
#pragma unroll
      for (int i = 0; i < NV; ++i) {
        const int j = lane + 32 * i;
        if (j < d4) {
          float4 o;
          o.x = (dh[i].x - m1 - xh[i].x * m2) * rs + dr[i].x;
          o.y = (dh[i].y - m1 - xh[i].y * m2) * rs + dr[i].y;
          o.z = (dh[i].z - m1 - xh[i].z * m2) * rs + dr[i].z;
          o.w = (dh[i].w - m1 - xh[i].w * m2) * rs + dr[i].w;
          store4(dx_out + row * d + 4 * j, o);
          if (dx_out_lp) {
            store4(dx_out_lp + row * d + 4 * j, o);
            if (want_colsum)                                           // sum what the GEMMs will read
              o = make_float4(to_f<T>(from_f<T>(o.x)), to_f<T>(from_f<T>(o.y)), to_f<T>(from_f<T>(o.z)),
                              to_f<T>(from_f<T>(o.w)));
          }
          *reinterpret_cast<float4 *>(slot + 2 * d + 4 * j) = o;
        }
      }
    } else {
      for (int j = lane; j < 3 * d4; j += 32) *reinterpret_cast<float4 *>(slot + 4 * j) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < NACC; ++j) {
      const int idx = threadIdx.x + NT * j;
      if (idx < 3 * d) {
        float t = 0.f;
#pragma unroll
        for (int r = 0; r < WARPS; ++r) t += red[(size_t)r * 3 * d + idx];      // rows in order
        acc[j] += t;
      }
    }
    __syncthreads();
  }
  float *out = partials + (size_t)blockIdx.x * 3 * d;
#pragma unroll
  for (int j = 0; j < NACC; ++j) {
    const int idx = threadIdx.x + NT * j;
    if (idx < 3 * d) out[idx] = acc[j];
  }
}

// dst[which][col] += sum_r partials[r][which][col]; block = 32 row-lanes x 32 columns
__global__ void __launch_bounds__(1024)
ln_bwd_reduce_kernel(const float *__restrict__ partials, int n_part, int d, float *__restrict__ dgamma,
                     float *__restrict__ dbeta, float *__restrict__ colsum_out) {
  __shared__ float red[32][33];
  int which = blockIdx.y;
  float *dst = which == 0 ? dgamma : (which == 1 ? dbeta : colsum_out);
  if (!dst) return;
  const int cx = threadIdx.x & 31, ry = threadIdx.x >> 5;
  const int col = blockIdx.x * 32 + cx;
  float s = 0.f;
  if (col < d)
    for (int r = ry; r < n_part; r += 32) s += partials[((size_t)r * 3 + which) * d + col];
  red[ry][cx] = s;
  __syncthreads();
  if (ry == 0 && col < d) {
    float t = 0.f;
#pragma unroll
    for (int r = 0; r < 32; ++r) t += red[r][cx];
    dst[col] += t;
  }
}

// one partial row per block, at most one block per SM and never more than the memory plan provides for (148)
int ln_bwd_partial_rows(int sm_count) { return sm_count < 148 ? sm_count : 148; }

template <typename T, int NV, int WARPS>
static cudaError_t ln_bwd_launch(const Ctx &c, const T *dy, const float *x, const float *mean, const float *rstd,
                                 const float *gamma, const float *dres_in, float *dx_out, T *dx_out_lp,
                                 float *partials, int64_t n_tok, int d, int want_colsum, int *grid_out) {
  int64_t want = (n_tok + WARPS - 1) / WARPS;
  int grid = (int)(want < ln_bwd_partial_rows(c.sm_count) ? want : ln_bwd_partial_rows(c.sm_count));
  size_t smem = (size_t)WARPS * 3 * d * sizeof(float);
  auto kern = ln_bwd_kernel<T, NV, WARPS>;
  if (smem > 48 * 1024) {                                  // once per device, for the widest row this instantiation takes
    cudaError_t e = ensure_dyn_smem<ln_bwd_kernel<T, NV, WARPS>>((size_t)WARPS * 3 * 128 * NV * sizeof(float), c.device);
    if (e != cudaSuccess) return e;
  }
  kern<<<grid, WARPS * 32, smem, c.stream>>>(dy, x, mean, rstd, gamma, dres_in, dx_out, dx_out_lp, partials, n_tok, d,
                                             want_colsum);
  *grid_out = grid;
  return cudaGetLastError();
}

template <typename T>
static cudaError_t ln_bwd_t(const Ctx &c, const T *dy, const float *x, const float *mean,
                            const float *rstd, const float *gamma, const float *dres_in,
                            float *dx_out, T *dx_out_lp, float *partials, float *dgamma,
                            float *dbeta, float *colsum_out, int64_t n_tok, int d) {
  if (n_tok == 0) return cudaSuccess;
  const int nv = (d / 4 + 31) / 32;
  const int wc = colsum_out != nullptr;
  int grid = 0;
  cudaError_t e;
  if (nv <= 1) e = ln_bwd_launch<T, 1, 16>(c, dy, x, mean, rstd, gamma, dres_in, dx_out, dx_out_lp, partials, n_tok, d, wc, &grid);
  else if (nv <= 8) e = ln_bwd_launch<T, 8, 16>(c, dy, x, mean, rstd, gamma, dres_in, dx_out, dx_out_lp, partials, n_tok, d, wc, &grid);
  else if (nv <= 16) e = ln_bwd_launch<T, 16, 8>(c, dy, x, mean, rstd, gamma, dres_in, dx_out, dx_out_lp, partials, n_tok, d, wc, &grid);
  else return cudaErrorInvalidValue;
  if (c.launches) ++*c.launches;
  if (e != cudaSuccess) return e;
  dim3 rg((d + 31) / 32, colsum_out ? 3 : 2);
  ln_bwd_reduce_kernel<<<rg, 1024, 0, c.stream>>>(partials, grid, d, dgamma, dbeta, colsum_out);
  GP_LAUNCH_CHECK(c);
}

cudaError_t ln_bwd(const Ctx &c, int dt, const void *dy, const float *x, const float *mean,
                   const float *rstd, const float *gamma, const float *dres_in, float *dx_out,
                   void *dx_out_lp, float *partials, float *dgamma, float *dbeta, float *colsum_out,
                   int64_t n_tok, int d) {
  return dt == GP_BF16
             ? ln_bwd_t<bf16>(c, (const bf16 *)dy, x, mean, rstd, gamma, dres_in, dx_out,
                              (bf16 *)dx_out_lp, partials, dgamma, dbeta, colsum_out, n_tok, d)
             : ln_bwd_t<float>(c, (const float *)dy, x, mean, rstd, gamma, dres_in, dx_out,
                               (float *)dx_out_lp, partials, dgamma, dbeta, colsum_out, n_tok, d);
}

// ---------------------------------------------------------------------------------------------
// bias gradient: out[n] += sum_t dy[t,n], two deterministic stages.  Stage 1: block = 16 row-lanes
// x 16 column groups of 8 (16-byte loads), grid (n/128, R slabs) -> partial [R][n].  Stage 2 sums
// the R partial rows.  Fixed summation order.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256)
colsum_stage1_kernel(const T *__restrict__ dy, int64_t ld, float *__restrict__ partial, int64_t n_tok, int n,
                     int rows_per_slab) {
  __shared__ float red[16][129];
  int cg = threadIdx.x & 15, rl = threadIdx.x >> 4;
  int col = blockIdx.x * 128 + cg * 8;
  int64_t r0 = (int64_t)blockIdx.y * rows_per_slab;
  int64_t r1 = r0 + rows_per_slab < n_tok ? r0 + rows_per_slab : n_tok;
  float acc[8];
#pragma unroll
  for (int e = 0; e < 8; ++e) acc[e] = 0.f;
  if (col + 8 <= n && (ld % 8) == 0 && sizeof(T) == 2) {
    for (int64_t r = r0 + rl; r < r1; r += 16) {
      uint4 u = *reinterpret_cast<const uint4 *>(dy + r * ld + col);
      const __nv_bfloat162 *h = reinterpret_cast<const __nv_bfloat162 *>(&u);
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        float2 f = __bfloat1622float2(h[q]);
        acc[2 * q] += f.x;
        acc[2 * q + 1] += f.y;
      }
    }
  } else {
    for (int64_t r = r0 + rl; r < r1; r += 16)
#pragma unroll
      for (int e = 0; e < 8; ++e)
        if (col + e < n) acc[e] += to_f<T>(dy[r * ld + col + e]);
  }
#pragma unroll
  for (int e = 0; e < 8; ++e) red[rl][cg * 8 + e] = acc[e];
  __syncthreads();
  if (threadIdx.x < 128) {
    int cidx = blockIdx.x * 128 + threadIdx.x;
    if (cidx < n) {
      float t = 0.f;
#pragma unroll
      for (int r = 0; r < 16; ++r) t += red[r][threadIdx.x];
      partial[(size_t)blockIdx.y * n + cidx] = t;
    }
  }
}

__global__ void __launch_bounds__(256)
colsum_stage2_kernel(const float *__restrict__ partial, int R, int n, int64_t ld, float *__restrict__ out) {
  int col = blockIdx.x * 256 + threadIdx.x;
  if (col >= n) return;
  float t = 0.f;
  for (int r = 0; r < R; ++r) t += partial[(size_t)r * ld + col];
  out[col] += t;
}

int colsum_scratch_rows(int64_t n_tok) {
  int64_t r = (n_tok + 127) / 128;
  return (int)(r < 1 ? 1 : (r > 32 ? 32 : r));
}

cudaError_t colsum_reduce_partials(const Ctx &c, const float *partial, int R, int n, int64_t ld, float *out) {
  if (n == 0) return cudaSuccess;
  colsum_stage2_kernel<<<(n + 255) / 256, 256, 0, c.stream>>>(partial, R, n, ld, out);
  GP_LAUNCH_CHECK(c);
}

cudaError_t colsum_accum(const Ctx &c, int dt, const void *dy, int64_t ld, float *out, float *scratch,
                         int64_t n_tok, int n) {
  if (n == 0 || n_tok == 0) return cudaSuccess;
  int R = colsum_scratch_rows(n_tok);
  int rows_per_slab = (int)((n_tok + R - 1) / R);
  dim3 grid((n + 127) / 128, R);
  if (dt == GP_BF16)
    colsum_stage1_kernel<bf16><<<grid, 256, 0, c.stream>>>((const bf16 *)dy, ld, scratch, n_tok, n, rows_per_slab);
  else
    colsum_stage1_kernel<float><<<grid, 256, 0, c.stream>>>((const float *)dy, ld, scratch, n_tok, n, rows_per_slab);
  if (c.launches) ++*c.launches;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  return colsum_reduce_partials(c, scratch, R, n, n, out);
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

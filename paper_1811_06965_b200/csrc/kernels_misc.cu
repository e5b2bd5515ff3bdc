// kernels_misc.cu - fused softmax cross-entropy over the vocabulary, loss reduction, SGD apply,
// device-side parameter initialisation (Philox-4x32-10 + Box-Muller) and dtype conversions.
#include "common.cuh"

namespace gp {

// ---------------------------------------------------------------------------------------------
// Fused softmax cross-entropy (reading A8): one block per token row.
//   rowloss[t] = (log sum_v exp(z_v - max) + max - z_label) * inv_T
//   z_v <- (exp(z_v - max)/sum - [v == label]) * inv_T            (in place: logits -> dlogits)
// Logit clipping ("we clip the logit predictions (softmax pre-activations) whenever their magnitude
// exceeds a certain value"; reading B5): with clip > 0 the softmax sees z = min(max(logit, -clip), clip) and the
// gradient is zero wherever the clamp is active (|logit| > clip); clip == 0 turns it off.
// The row is read once from HBM and kept on the SM - vectors of 8 (bf16) / 4 (fp32) elements, VR per thread in
// registers and VS more in shared memory - when it fits (up to 8192 vectors), so HBM traffic is one read + one
// write of the row; longer rows fall back to three passes over global memory (L2-resident row).
// ---------------------------------------------------------------------------------------------
template <typename T> struct VecIO;       // 16-byte vectors kept packed in registers
template <> struct VecIO<float> {
  static constexpr int W = 4;
  __device__ static void unpack(const uint4 &u, float *v) {
    v[0] = __uint_as_float(u.x); v[1] = __uint_as_float(u.y);
    v[2] = __uint_as_float(u.z); v[3] = __uint_as_float(u.w);
  }
  __device__ static uint4 pack(const float *v) {
    return make_uint4(__float_as_uint(v[0]), __float_as_uint(v[1]), __float_as_uint(v[2]),
                      __float_as_uint(v[3]));
  }
  __device__ static float vmax(const uint4 &u) {
    return fmaxf(fmaxf(__uint_as_float(u.x), __uint_as_float(u.y)), fmaxf(__uint_as_float(u.z), __uint_as_float(u.w)));
  }
};
template <> struct VecIO<bf16> {
  static constexpr int W = 8;
  __device__ static void unpack(const uint4 &u, float *v) {
    const __nv_bfloat162 *h = reinterpret_cast<const __nv_bfloat162 *>(&u);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      float2 f = __bfloat1622float2(h[i]);
      v[2 * i] = f.x;
      v[2 * i + 1] = f.y;
    }
  }
  __device__ static uint4 pack(const float *v) {
    uint4 u;
    __nv_bfloat162 *h = reinterpret_cast<__nv_bfloat162 *>(&u);
#pragma unroll
    for (int i = 0; i < 4; ++i) h[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]);
    return u;
  }
  __device__ static float vmax(const uint4 &u) {           // the maximum is exact in any format: packed bf16 max
    const __nv_bfloat162 *h = reinterpret_cast<const __nv_bfloat162 *>(&u);
    const __nv_bfloat162 m = __hmax2(__hmax2(h[0], h[1]), __hmax2(h[2], h[3]));
    return fmaxf(__low2float(m), __high2float(m));
  }
};

// 2^x on the special-function unit, one instruction (relative error 2^-22; results below 2^-126 flush to zero)
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// Instruction budget (the row pass is issue-bound before it is HBM-bound: 131 M elements per config-5 micro-batch):
// packed max in pass 1; per element one subtract, one multiply / FMA and one ex2 in passes 2 and 3 - the factors
// 1/sum and 1/T go into the exponent of pass 3 (p / T = 2^((z - max) log2 e - log2 sum + log2 (1/T))); the label's
// "- 1/T" is applied to its one vector; the clamp exists only in the CLIP instantiation.
// Residency: a row of V = 64000 bf16 is 125 KB - as registers alone it takes a whole SM's register file, and then an SM
// works on ONE row at a time with nothing to overlap its load, its two block-wide reductions and its store with.  So
// a block is NT <= 512 threads and keeps VR vectors per thread in registers and VS more in shared memory (thread-
// private slots, conflict-free): two blocks = two rows in flight per SM.
template <typename T, int NT, int VR, int VS, bool CLIP>
__global__ void __launch_bounds__(NT, NT == 512 ? 2 : 1)
softmax_ce_reg_kernel(T *__restrict__ logits, const int32_t *__restrict__ labels,
                      float *__restrict__ rowloss, int V, float inv_T, float clip) {
  const float hi = CLIP ? clip : INFINITY, lo = -hi;
  constexpr int W = VecIO<T>::W;
  constexpr float L2E = 1.4426950408889634f;
  extern __shared__ uint4 spill[];          // [VS][NT]
  __shared__ float red[33];
  int64_t row = blockIdx.x;
  uint4 *z = reinterpret_cast<uint4 *>(logits + row * (int64_t)V);
  int nvec = V / W;
  uint4 raw[VR];
  float mx = -INFINITY;
#pragma unroll
  for (int i = 0; i < VR + VS; ++i) {
    int j = threadIdx.x + i * NT;
    if (j < nvec) {
      const uint4 u = z[j];
      if (i < VR) raw[i < VR ? i : 0] = u;
      else spill[(i - VR) * NT + threadIdx.x] = u;
      mx = fmaxf(mx, VecIO<T>::vmax(u));
    }
  }
  mx = block_max(mx, red);
  if (CLIP) mx = fmaxf(fminf(mx, hi), lo);   // max of the clamped row (the clamp is monotone)
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < VR + VS; ++i) {
    int j = threadIdx.x + i * NT;
    if (j < nvec) {
      float v[W];
      VecIO<T>::unpack(i < VR ? raw[i < VR ? i : 0] : spill[(i - VR) * NT + threadIdx.x], v);
#pragma unroll
      for (int e = 0; e < W; ++e) {
        const float x = CLIP ? fminf(fmaxf(v[e], lo), hi) : v[e];
        s += ex2_approx((x - mx) * L2E);
      }
    }
  }
  s = block_sum(s, red);
  const int lab = labels[row];
  const int jl = lab / W, el = lab - jl * W;
  if (threadIdx.x == 0) {
    const float zl = to_f<T>(logits[row * (int64_t)V + lab]);
    rowloss[row] = (logf(s) + mx - (CLIP ? fminf(fmaxf(zl, lo), hi) : zl)) * inv_T;
  }
  const float c = log2f(inv_T) - log2f(s);
  __syncthreads();                       // z[lab] read before anyone overwrites it
#pragma unroll
  for (int i = 0; i < VR + VS; ++i) {
    int j = threadIdx.x + i * NT;
    if (j < nvec) {
      const uint4 u = i < VR ? raw[i < VR ? i : 0] : spill[(i - VR) * NT + threadIdx.x];
      float v[W];
      VecIO<T>::unpack(u, v);
#pragma unroll
      for (int e = 0; e < W; ++e) {
        const float x = CLIP ? fminf(fmaxf(v[e], lo), hi) : v[e];
        const float p = ex2_approx(fmaf(x - mx, L2E, c));
        v[e] = (!CLIP || (v[e] >= lo && v[e] <= hi)) ? p : 0.f;
      }
      if (j == jl) {                       // the label's element: (p - 1) / T, or zero under an active clamp
        if constexpr (CLIP) {
          float r[W];
          VecIO<T>::unpack(u, r);
#pragma unroll
          for (int e = 0; e < W; ++e)
            if (e == el && r[e] >= lo && r[e] <= hi) v[e] -= inv_T;
        } else {
#pragma unroll
          for (int e = 0; e < W; ++e)
            if (e == el) v[e] -= inv_T;
        }
      }
      z[j] = VecIO<T>::pack(v);
    }
  }
}

template <typename T>
__global__ void __launch_bounds__(1024)
softmax_ce_3pass_kernel(T *__restrict__ logits, const int32_t *__restrict__ labels,
                        float *__restrict__ rowloss, int V, float inv_T, float clip) {
  const float hi = clip > 0.f ? clip : INFINITY, lo = -hi;
  __shared__ float red[33];
  int64_t row = blockIdx.x;
  T *z = logits + row * (int64_t)V;
  float mx = -INFINITY;
  for (int j = threadIdx.x; j < V; j += blockDim.x) mx = fmaxf(mx, to_f<T>(z[j]));
  mx = fmaxf(fminf(block_max(mx, red), hi), lo);
  float s = 0.f;
  for (int j = threadIdx.x; j < V; j += blockDim.x) s += expf(fminf(fmaxf(to_f<T>(z[j]), lo), hi) - mx);
  s = block_sum(s, red);
  int lab = labels[row];
  float inv = 1.f / s;
  if (threadIdx.x == 0) rowloss[row] = (logf(s) + mx - fminf(fmaxf(to_f<T>(z[lab]), lo), hi)) * inv_T;
  __syncthreads();
  for (int j = threadIdx.x; j < V; j += blockDim.x) {
    const float zj = to_f<T>(z[j]);
    float p = expf(fminf(fmaxf(zj, lo), hi) - mx) * inv;
    if (j == lab) p -= 1.f;
    z[j] = from_f<T>((zj >= lo && zj <= hi) ? p * inv_T : 0.f);
  }
}

template <typename T>
static cudaError_t softmax_ce_t(const Ctx &c, T *logits, const int32_t *labels, float *rowloss,
                                int64_t n_tok, int V, float inv_T, float clip) {
  if (n_tok == 0) return cudaSuccess;
  constexpr int W = VecIO<T>::W;
  unsigned grid = (unsigned)n_tok;
  int nvec = V / W;
  bool vec_ok = (V % W == 0);
  const bool cl = clip > 0.f;
  if (vec_ok && nvec <= 256) {
    if (cl) softmax_ce_reg_kernel<T, 256, 1, 0, true><<<grid, 256, 0, c.stream>>>(logits, labels, rowloss, V, inv_T, clip);
    else softmax_ce_reg_kernel<T, 256, 1, 0, false><<<grid, 256, 0, c.stream>>>(logits, labels, rowloss, V, inv_T, clip);
  } else if (vec_ok && nvec <= 512 * 8) {
    if (cl) softmax_ce_reg_kernel<T, 512, 8, 0, true><<<grid, 512, 0, c.stream>>>(logits, labels, rowloss, V, inv_T, clip);
    else softmax_ce_reg_kernel<T, 512, 8, 0, false><<<grid, 512, 0, c.stream>>>(logits, labels, rowloss, V, inv_T, clip);
  } else if (vec_ok && nvec <= 512 * 16) {
    constexpr size_t smem = (size_t)8 * 512 * sizeof(uint4);            // 64 KB: two blocks per SM
    cudaError_t e = cl ? ensure_dyn_smem<softmax_ce_reg_kernel<T, 512, 8, 8, true>>(smem, c.device)
                       : ensure_dyn_smem<softmax_ce_reg_kernel<T, 512, 8, 8, false>>(smem, c.device);
    if (e != cudaSuccess) return e;
    if (cl) softmax_ce_reg_kernel<T, 512, 8, 8, true><<<grid, 512, smem, c.stream>>>(logits, labels, rowloss, V, inv_T, clip);
    else softmax_ce_reg_kernel<T, 512, 8, 8, false><<<grid, 512, smem, c.stream>>>(logits, labels, rowloss, V, inv_T, clip);
  } else
    softmax_ce_3pass_kernel<T><<<grid, 1024, 0, c.stream>>>(logits, labels, rowloss, V, inv_T, clip);
  GP_LAUNCH_CHECK(c);
}

cudaError_t softmax_ce(const Ctx &c, int dt, void *logits, const int32_t *labels, float *rowloss,
                       int64_t n_tok, int V, float inv_T, float clip) {
  return dt == GP_BF16 ? softmax_ce_t<bf16>(c, (bf16 *)logits, labels, rowloss, n_tok, V, inv_T, clip)
                       : softmax_ce_t<float>(c, (float *)logits, labels, rowloss, n_tok, V, inv_T, clip);
}

// single block, fixed order: loss = sum_t rowloss[t]
__global__ void __launch_bounds__(1024)
loss_reduce_kernel(const float *__restrict__ rowloss, float *__restrict__ loss, int64_t n) {
  __shared__ float red[33];
  float s = 0.f;
  for (int64_t i = threadIdx.x; i < n; i += blockDim.x) s += rowloss[i];
  s = block_sum(s, red);
  if (threadIdx.x == 0) *loss = s;
}

cudaError_t loss_reduce(const Ctx &c, const float *rowloss, float *loss, int64_t n_tok) {
  loss_reduce_kernel<<<1, 1024, 0, c.stream>>>(rowloss, loss, n_tok);
  GP_LAUNCH_CHECK(c);
}

// ---------------------------------------------------------------------------------------------
// SGD apply: master -= lr*g; working copy = RNE(master); g = 0.  One pass.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256)
sgd_kernel(float *__restrict__ master, float *__restrict__ grad, T *__restrict__ w_lp, int64_t n4,
           float lr) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4;
       i += (int64_t)gridDim.x * blockDim.x) {
    float4 m = load4(master + 4 * i), g = load4(grad + 4 * i);
    m.x -= lr * g.x; m.y -= lr * g.y; m.z -= lr * g.z; m.w -= lr * g.w;
    store4(master + 4 * i, m);
    if (w_lp) store4(w_lp + 4 * i, m);
    store4(grad + 4 * i, make_float4(0.f, 0.f, 0.f, 0.f));
  }
}

cudaError_t sgd_apply(const Ctx &c, int dt, float *master, float *grad, void *w_lp, int64_t n,
                      float lr) {
  if (n == 0) return cudaSuccess;
  int64_t n4 = n / 4;
  int64_t want = (n4 + 255) / 256;
  unsigned grid = (unsigned)(want < (int64_t)c.sm_count * 16 ? want : (int64_t)c.sm_count * 16);
  if (dt == GP_BF16) sgd_kernel<bf16><<<grid, 256, 0, c.stream>>>(master, grad, (bf16 *)w_lp, n4, lr);
  else sgd_kernel<float><<<grid, 256, 0, c.stream>>>(master, grad, (float *)nullptr, n4, lr);
  GP_LAUNCH_CHECK(c);
}

// ---------------------------------------------------------------------------------------------
// RMSProp apply ("12 bytes [per parameter] since we applied RMSProp": weight +
// gradient + one fp32 slot).  ms = rho*ms + (1-rho)*g^2; master -= lr * g / (sqrt(ms) + eps); working copy =
// RNE(master); g = 0 (reading A20).  One pass: 26 B / parameter in bf16 mode (g r+w, ms r+w, master r+w, lp w).
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256)
rmsprop_kernel(float *__restrict__ master, float *__restrict__ grad, float *__restrict__ ms, T *__restrict__ w_lp,
               int64_t n4, float lr, float rho, float eps) {
  const float om = 1.f - rho;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4;
       i += (int64_t)gridDim.x * blockDim.x) {
    float4 m = load4(master + 4 * i), g = load4(grad + 4 * i), v = load4(ms + 4 * i);
    v.x = rho * v.x + om * g.x * g.x; v.y = rho * v.y + om * g.y * g.y;
    v.z = rho * v.z + om * g.z * g.z; v.w = rho * v.w + om * g.w * g.w;
    m.x -= lr * g.x / (sqrtf(v.x) + eps); m.y -= lr * g.y / (sqrtf(v.y) + eps);
    m.z -= lr * g.z / (sqrtf(v.z) + eps); m.w -= lr * g.w / (sqrtf(v.w) + eps);
    store4(ms + 4 * i, v);
    store4(master + 4 * i, m);
    if (w_lp) store4(w_lp + 4 * i, m);
    store4(grad + 4 * i, make_float4(0.f, 0.f, 0.f, 0.f));
  }
}

cudaError_t rmsprop_apply(const Ctx &c, int dt, float *master, float *grad, float *ms, void *w_lp, int64_t n,
                          float lr, float rho, float eps) {
  if (n == 0) return cudaSuccess;
  int64_t n4 = n / 4;
  int64_t want = (n4 + 255) / 256;
  unsigned grid = (unsigned)(want < (int64_t)c.sm_count * 16 ? want : (int64_t)c.sm_count * 16);
  if (dt == GP_BF16) rmsprop_kernel<bf16><<<grid, 256, 0, c.stream>>>(master, grad, ms, (bf16 *)w_lp, n4, lr, rho, eps);
  else rmsprop_kernel<float><<<grid, 256, 0, c.stream>>>(master, grad, ms, (float *)nullptr, n4, lr, rho, eps);
  GP_LAUNCH_CHECK(c);
}

// ---------------------------------------------------------------------------------------------
// Data-parallel replicas: gradient reduction fused with the apply ("scale ... using
// data parallelism": R replicas of the pipeline hold identical parameters and take different mini-batches).
// Replica r owns the contiguous shard [lo, hi) of the flat parameter range.  One kernel per replica, launched after
// every replica's gpipe_step has finished:
//   g   = scale * (grad_0[i] + grad_1[i] + ... + grad_{R-1}[i])       peer loads over NVLink, summed in rank order
//   grad_p[i] = 0 for every p                                         (nobody but the owner reads shard elements)
//   SGD:      m = master_r[i] - lr g
//   RMSProp:  ms_r[i] = rho ms_r[i] + (1 - rho) g^2 ;  m = master_r[i] - lr g / (sqrt(ms_r[i]) + eps)
//   master_p[i] = m, working copy_p[i] = RNE(m) for every p           peer stores: the all-gather of the update
// i.e. reduce-scatter + optimizer + all-gather in one pass over the shard, no staging buffers, no collective
// library call; every replica ends with bit-identical parameters (one owner computes each element, in a fixed
// order).  The kernel waits on no other replica: ordering between replicas is the host's (a barrier before - all
// gradients final - and after - all parameters updated), so R launches may also run back to back on ONE device
// (how the single-GPU tests emulate R ranks).  Roofline: NVLink for R > 1 ((R-1)/R of 4 B read + 10 B written per
// parameter cross the links), HBM for R = 1.
// ---------------------------------------------------------------------------------------------
template <typename T, bool RMS>
__global__ void __launch_bounds__(256)
dp_apply_kernel(DpPeers P, int world, int self, int64_t lo4, int64_t hi4, float lr, float gscale, float rho, float eps) {
  const float om = 1.f - rho;
  for (int64_t i = lo4 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < hi4; i += (int64_t)gridDim.x * blockDim.x) {
    float4 g = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int p = 0; p < world; ++p) {                       // rank order: the sum is the same whoever computes it
      const float4 q = load4(P.grad[p] + 4 * i);
      g.x += q.x; g.y += q.y; g.z += q.z; g.w += q.w;
    }
    g.x *= gscale; g.y *= gscale; g.z *= gscale; g.w *= gscale;
    float4 m = load4(P.master[self] + 4 * i);
    if (RMS) {
      float4 v = load4(P.slot + 4 * i);
      v.x = rho * v.x + om * g.x * g.x; v.y = rho * v.y + om * g.y * g.y;
      v.z = rho * v.z + om * g.z * g.z; v.w = rho * v.w + om * g.w * g.w;
      m.x -= lr * g.x / (sqrtf(v.x) + eps); m.y -= lr * g.y / (sqrtf(v.y) + eps);
      m.z -= lr * g.z / (sqrtf(v.z) + eps); m.w -= lr * g.w / (sqrtf(v.w) + eps);
      store4(P.slot + 4 * i, v);
    } else {
      m.x -= lr * g.x; m.y -= lr * g.y; m.z -= lr * g.z; m.w -= lr * g.w;
    }
    for (int p = 0; p < world; ++p) {
      store4(P.grad[p] + 4 * i, make_float4(0.f, 0.f, 0.f, 0.f));
      store4(P.master[p] + 4 * i, m);
      if (P.wlp[p]) store4(reinterpret_cast<T *>(P.wlp[p]) + 4 * i, m);
    }
  }
}

// the shard of replica `rank`: 64-element aligned cuts of [0, n) (every tensor starts on a 64-element boundary)
void dp_shard(int64_t n, int rank, int world, int64_t *lo, int64_t *hi) {
  const int64_t blocks = (n + 63) / 64, per = (blocks + world - 1) / world;
  int64_t a = (int64_t)rank * per * 64, b = (int64_t)(rank + 1) * per * 64;
  *lo = a < n ? a : n;
  *hi = b < n ? b : n;
}

cudaError_t dp_apply(const Ctx &c, int dt, const DpPeers &P, int world, int self, int64_t n, float lr, float gscale,
                     int rms, float rho, float eps) {
  if (world < 1 || world > DpPeers::kMax || self < 0 || self >= world) return cudaErrorInvalidValue;
  int64_t lo, hi;
  dp_shard(n, self, world, &lo, &hi);
  if (hi <= lo) return cudaSuccess;
  const int64_t lo4 = lo / 4, hi4 = hi / 4, n4 = hi4 - lo4;
  int64_t want = (n4 + 255) / 256;
  unsigned grid = (unsigned)(want < (int64_t)c.sm_count * 16 ? want : (int64_t)c.sm_count * 16);
  if (dt == GP_BF16) {
    if (rms) dp_apply_kernel<bf16, true><<<grid, 256, 0, c.stream>>>(P, world, self, lo4, hi4, lr, gscale, rho, eps);
    else dp_apply_kernel<bf16, false><<<grid, 256, 0, c.stream>>>(P, world, self, lo4, hi4, lr, gscale, rho, eps);
  } else {
    if (rms) dp_apply_kernel<float, true><<<grid, 256, 0, c.stream>>>(P, world, self, lo4, hi4, lr, gscale, rho, eps);
    else dp_apply_kernel<float, false><<<grid, 256, 0, c.stream>>>(P, world, self, lo4, hi4, lr, gscale, rho, eps);
  }
  GP_LAUNCH_CHECK(c);
}

// ---------------------------------------------------------------------------------------------
// Philox-4x32-10 counter RNG + Box-Muller; element i uses counter (i/4, stream_id), lane i%4
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox_round(uint32_t &c0, uint32_t &c1, uint32_t &c2, uint32_t &c3,
                                             uint32_t k0, uint32_t k1) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
  uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
  uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
  c0 = n0; c1 = n1; c2 = n2; c3 = n3;
}

template <typename T>
__global__ void __launch_bounds__(256)
init_normal_kernel(float *__restrict__ master, T *__restrict__ w_lp, int64_t n4, uint64_t seed,
                   uint64_t stream_id, float mean, float std) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4;
       i += (int64_t)gridDim.x * blockDim.x) {
    uint32_t c0 = (uint32_t)i, c1 = (uint32_t)((uint64_t)i >> 32);
    uint32_t c2 = (uint32_t)stream_id, c3 = (uint32_t)(stream_id >> 32);
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
      philox_round(c0, c1, c2, c3, k0, k1);
      k0 += 0x9E3779B9u;
      k1 += 0xBB67AE85u;
    }
    const float two32 = 2.3283064365386963e-10f;
    float u0 = ((float)c0 + 0.5f) * two32, u1 = ((float)c1 + 0.5f) * two32;
    float u2 = ((float)c2 + 0.5f) * two32, u3 = ((float)c3 + 0.5f) * two32;
    u0 = fminf(fmaxf(u0, 1e-12f), 1.f);
    u2 = fminf(fmaxf(u2, 1e-12f), 1.f);
    float r0 = sqrtf(-2.f * logf(u0)), r1 = sqrtf(-2.f * logf(u2));
    float s0, c0f, s1, c1f;
    sincospif(2.f * u1, &s0, &c0f);
    sincospif(2.f * u3, &s1, &c1f);
    float4 v = make_float4(mean + std * r0 * c0f, mean + std * r0 * s0, mean + std * r1 * c1f,
                           mean + std * r1 * s1);
    if (w_lp) {                      // bf16 mode: master = the RNE-rounded draw (reading A12)
      store4(w_lp + 4 * i, v);
      v = load4(w_lp + 4 * i);
    }
    store4(master + 4 * i, v);
  }
}

cudaError_t init_normal(const Ctx &c, int dt, float *master, void *w_lp, int64_t n, uint64_t seed,
                        uint64_t stream_id, float mean, float std) {
  if (n == 0) return cudaSuccess;
  int64_t n4 = n / 4;
  int64_t want = (n4 + 255) / 256;
  unsigned grid = (unsigned)(want < (int64_t)c.sm_count * 16 ? want : (int64_t)c.sm_count * 16);
  if (dt == GP_BF16)
    init_normal_kernel<bf16><<<grid, 256, 0, c.stream>>>(master, (bf16 *)w_lp, n4, seed, stream_id, mean, std);
  else
    init_normal_kernel<float><<<grid, 256, 0, c.stream>>>(master, (float *)nullptr, n4, seed, stream_id, mean, std);
  GP_LAUNCH_CHECK(c);
}

__global__ void fill_kernel(float *p, int64_t n, float v) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x)
    p[i] = v;
}
cudaError_t fill_f32(const Ctx &c, float *p, int64_t n, float v) {
  if (n == 0) return cudaSuccess;
  int64_t want = (n + 255) / 256;
  unsigned grid = (unsigned)(want < (int64_t)c.sm_count * 16 ? want : (int64_t)c.sm_count * 16);
  fill_kernel<<<grid, 256, 0, c.stream>>>(p, n, v);
  GP_LAUNCH_CHECK(c);
}

// master (fp32) -> lp working copy; round_master != 0 also writes the rounded value back
template <typename T>
__global__ void master_to_lp_kernel(float *__restrict__ master, T *__restrict__ w_lp, int64_t n,
                                    int round_master) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x) {
    T v = from_f<T>(master[i]);
    w_lp[i] = v;
    if (round_master) master[i] = to_f<T>(v);
  }
}
cudaError_t master_to_lp(const Ctx &c, int dt, float *master, void *w_lp, int64_t n, int round_master) {
  if (n == 0 || dt != GP_BF16) return cudaSuccess;
  int64_t want = (n + 255) / 256;
  unsigned grid = (unsigned)(want < (int64_t)c.sm_count * 16 ? want : (int64_t)c.sm_count * 16);
  master_to_lp_kernel<bf16><<<grid, 256, 0, c.stream>>>(master, (bf16 *)w_lp, n, round_master);
  GP_LAUNCH_CHECK(c);
}

template <typename T>
__global__ void lp_to_f32_kernel(const T *__restrict__ src, float *__restrict__ dst, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x)
    dst[i] = to_f<T>(src[i]);
}
cudaError_t lp_to_f32(const Ctx &c, int dt, const void *src, float *dst, int64_t n) {
  if (n == 0) return cudaSuccess;
  int64_t want = (n + 255) / 256;
  unsigned grid = (unsigned)(want < (int64_t)c.sm_count * 16 ? want : (int64_t)c.sm_count * 16);
  if (dt == GP_BF16) lp_to_f32_kernel<bf16><<<grid, 256, 0, c.stream>>>((const bf16 *)src, dst, n);
  else lp_to_f32_kernel<float><<<grid, 256, 0, c.stream>>>((const float *)src, dst, n);
  GP_LAUNCH_CHECK(c);
}

__global__ void check_ids_kernel(const int32_t *__restrict__ ids, int64_t n, int V, int *flag) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x)
    if (ids[i] < 0 || ids[i] >= V) *flag = 1;
}
cudaError_t check_ids(const Ctx &c, const int32_t *ids, int64_t n, int V, int *flag) {
  if (n == 0) return cudaSuccess;
  int64_t want = (n + 255) / 256;
  unsigned grid = (unsigned)(want < (int64_t)c.sm_count * 4 ? want : (int64_t)c.sm_count * 4);
  check_ids_kernel<<<grid, 256, 0, c.stream>>>(ids, n, V, flag);
  GP_LAUNCH_CHECK(c);
}

}  // namespace gp

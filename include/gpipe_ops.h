/* gpipe_ops.h - C ABI of the individual sm_100a kernels of the GPipe hot path, exported so that
 * each one can be checked against the oracle's corresponding operator on identical inputs
 * ("teacher-forced" per-kernel parity) and timed in isolation against its roofline.
 * gpipe_step (gpipe.h) is built from exactly these launchers.
 *
 * All data pointers are DEVICE pointers; `stream` is a cudaStream_t (0 = default stream).
 * `dtype` is GPIPE_DTYPE_FP32 or GPIPE_DTYPE_BF16 and selects the storage type of "lp" tensors
 * (tensor-core operands: activations, activation gradients, weight matrices); residual stream,
 * statistics, biases/gains, losses and parameter gradients are always fp32.  Calls are
 * asynchronous on `stream`; status 0 / negative as in gpipe.h (message via gpipe_last_error).
 * Layer math per BASELINE.json north_star and DESIGN.md readings A2-A8 (the paper cites [15]
 * for the layer).
 */
#ifndef GPIPE_OPS_H_
#define GPIPE_OPS_H_
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#pragma GCC visibility push(default)   /* the library is built with -fvisibility=hidden */
#endif

/* epilogue flags of gpipe_op_gemm */
#define GPIPE_EPI_BIAS    1   /* + bias[n]            (fp32 [N])                                  */
#define GPIPE_EPI_RELU    2   /* max(v, 0)                                                        */
#define GPIPE_EPI_MASK    4   /* v * maskbit[m,n]: mask is a bit-packed uint32 [M, ldmask] array, bit
                                 (n % 32) of word n / 32 (ReLU backward); ldmask >= ceil(N / 32)      */
#define GPIPE_EPI_RESID   8   /* + resid[m,n]         (fp32 [M, ldc], may alias C)                */
#define GPIPE_EPI_ACCUM  16   /* C (fp32) += v        (wgrad accumulation across micro-batches)   */
#define GPIPE_EPI_OUT_F32 32  /* C is fp32, else lp                                               */
#define GPIPE_EPI_COLSUM 64   /* colsum_out[n] += sum_m C[m,n] of the stored values (bias gradient
                                 of the layer below, fused into the dgrad GEMM); lp output only   */
#define GPIPE_EPI_BITS_OUT 128 /* mask (layout of GPIPE_EPI_MASK) is an OUTPUT: bit = [stored C > 0]
                                 (the FFN1 epilogue records the ReLU pattern in 1 bit per unit
                                 instead of having backward re-read h)                             */

/* C[M,N] = epilogue(op(A)[M,K] op(B)[K,N]), fp32 accumulation.  transA = 0: A stored [M,K]
 * row-major, 1: stored [K,M]; transB = 0: B stored [K,N], 1: stored [N,K].  backend: 0 = auto
 * (tcgen05 tensor cores for bf16 - a bf16 problem the tensor-core kernel cannot take, i.e. an
 * unaligned base / row pitch or N % 32 != 0 with a ReLU pattern, fails with GPIPE_EINVAL; the SIMT
 * kernel for fp32), 1 = fp32-FMA SIMT kernel,
 * 2 = tcgen05 or fail with GPIPE_EINVAL, 3 = tcgen05 with 256 x 256 CTA-pair tiles only, 4 = tcgen05 with
 * 256 x 512 CTA-pair tiles (N >= 512; flags 0, ACCUM | OUT_F32 or BIAS | RELU | BITS_OUT) or fail with
 * GPIPE_EINVAL; backends 0 and 2 pick the tile from the shape (results are bitwise the same).  colsum_out fp32 [N] / colsum_scratch fp32
 * [gpipe_op_colsum_scratch_floats(M, N)] are only read with GPIPE_EPI_COLSUM.
 * workspace (device, may be NULL): gpipe_op_gemm_workspace_bytes(M, N, K) bytes that were ZERO before
 * their first use and are only ever used by launches on one stream at a time; with it, shapes
 * with few output tiles and a long K are split along K over all SMs and reduced in a fixed order
 * (deterministic); without it they are not split. */
int64_t gpipe_op_gemm_workspace_bytes(int M, int N, int K);
int gpipe_op_gemm(void *stream, int dtype, int M, int N, int K, const void *A, int64_t lda, int transA,
                  const void *B, int64_t ldb, int transB, void *C, int64_t ldc, const float *bias,
                  const float *resid, void *mask, int64_t ldmask, float *colsum_out,
                  float *colsum_scratch, void *workspace, int64_t workspace_bytes, int flags, int backend);

/* y = LayerNorm(x) * gamma + beta over the last axis (biased variance); y lp [n_tok,d]; x fp32.
 * Fused residual: if resid_out != NULL (fp32 [n_tok,d], device, caller-owned)
 * the kernel also writes resid_out = x + resid_bias (fp32 [d], required then) - the buffer the branch's
 * output GEMM accumulates into with GPIPE_EPI_ACCUM, giving x' = x + branch(y) + bias. */
int gpipe_op_ln_fwd(void *stream, int dtype, const float *x, const float *gamma, const float *beta,
                    void *y, float *mean, float *rstd, const float *resid_bias, float *resid_out,
                    int64_t n_tok, int d, float eps);
/* dx_out = (dres_in ? dres_in : 0) + LN'(dy); dx_out_lp optional lp copy; dgamma/dbeta += ;
 * colsum_out (optional, fp32 [d]) += sum_t dx_out[t,:] (the lp copy's values when there is one).
 * partials: fp32 scratch of gpipe_op_ln_bwd_scratch_floats(d) floats. */
int64_t gpipe_op_ln_bwd_scratch_floats(int d);
int gpipe_op_ln_bwd(void *stream, int dtype, const void *dy, const float *x, const float *mean,
                    const float *rstd, const float *gamma, const float *dres_in, float *dx_out,
                    void *dx_out_lp, float *partials, float *dgamma, float *dbeta, float *colsum_out,
                    int64_t n_tok, int d);

/* qkv lp [n_seq*S, 3*A*dh] (q|k|v blocks); o lp [n_seq*S, A*dh]; lse fp32 [n_seq, A, S].
 * backend: 0 = auto (bf16: tcgen05 when d_head = 64 and S <= 256, else mma.sync; fp32: SIMT), 1 = SIMT,
 * 2 = legacy mma.sync kernels (bf16, d_head 32 / 64; GPIPE_ENOTIMPL-style CUDA error otherwise). */
int gpipe_op_attn_fwd(void *stream, int dtype, const void *qkv, void *o, float *lse, int n_seq, int S,
                      int A, int dh, int causal, int backend);
/* colpart (optional; bf16, d_head 64, S <= 256, backend 0 only - GPIPE_ECUDA/invalid value otherwise): fp32
 * [n_seq, 3*A*dh], row s = the column sums of the dqkv rows of sequence s as stored (the per-sequence partials of the
 * bias gradient db_qkv), fused into the kernel's store path. */
int gpipe_op_attn_bwd(void *stream, int dtype, const void *qkv, const void *o, const void *d_o,
                      const float *lse, void *dqkv, float *dvec, int n_seq, int S, int A, int dh,
                      int causal, int backend, float *colpart);

/* in place logits -> dlogits = (softmax - onehot) * inv_T; rowloss[t] = CE_t * inv_T.
 * clip > 0 ("we clip the logit predictions (softmax pre-activations) whenever their magnitude exceeds a
 * certain value"; reading B5): the softmax and the loss see clamp(logit, -clip, clip) and dlogits is 0
 * wherever |logit| > clip; clip == 0: no clipping. */
int gpipe_op_softmax_ce(void *stream, int dtype, void *logits, const int32_t *labels, float *rowloss,
                        int64_t n_tok, int V, float inv_T, float clip);
/* out[n] += sum_t dy[t,n]; scratch: fp32 [gpipe_op_colsum_scratch_floats(n_tok, n)] */
int64_t gpipe_op_colsum_scratch_floats(int64_t n_tok, int n);
int gpipe_op_colsum(void *stream, int dtype, const void *dy, int64_t ld, float *out, float *scratch,
                    int64_t n_tok, int n);
/* The same column sums for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): out[n] += sum_t dy[t,n] with the kernels' scratch in a file-scope
 * __device__ array inside the library (2 MiB, held by every GPU that loads the library until the process exits)
 * instead of a caller-owned buffer.  Same kernels, same summation order: results are bitwise those of gpipe_op_colsum.
 * dy: device, dtype elements [n_tok, ld]; out: device fp32 [n], accumulated into; both caller-owned.  n <=
 * GPIPE_COLSUM_STATIC_MAX_N, wider inputs return GPIPE_EINVAL (message names the limit).  The call allocates nothing
 * (no cudaMalloc / cudaFree / allocating library routine) and runs on the current device.  All calls share the one
 * array per device: calls that overlap on the GPU (different streams) race - serialise them, or use gpipe_op_colsum
 * with one scratch buffer per stream.  Nothing in the array has to be cleared between calls. */
#define GPIPE_COLSUM_STATIC_MAX_N 16384
int gpipe_op_colsum_static(void *stream, int dtype, const void *dy, int64_t ld, float *out, int64_t n_tok, int n);
/* x[t,:] = emb[tok[t],:] + pe[t mod S,:];  gemb[tok[t],:] += dx[t,:] */
int gpipe_op_embed_fwd(void *stream, int dtype, const int32_t *tok, const void *emb, const float *pe,
                       float *x, int64_t n_tok, int S, int d);
int gpipe_op_embed_bwd(void *stream, const int32_t *tok, const float *dx, float *gemb, int64_t n_tok, int d);
int gpipe_op_positional(void *stream, float *pe, int S, int d);
/* master -= lr*grad; w_lp = RNE(master) (bf16 mode, may be NULL); grad = 0.  n multiple of 4. */
/* The fused data-parallel apply of gpipe_dp_apply_sgd on raw arrays: replica `rank` of `world`
 * sums grad[0..world)[i] over its shard gpipe_dp_shard(n, rank, world) in rank order, times grad_scale, clears them,
 * updates master[rank][i] and stores the result (and its RNE-bf16 copy when w_lp != NULL) into every replica.
 * master / grad / w_lp: HOST arrays of `world` DEVICE pointers (n fp32 / n fp32 / n bf16 elements each). */
int gpipe_op_dp_apply_sgd(void *stream, int dtype, int world, int rank, float *const *master, float *const *grad,
                          void *const *w_lp, int64_t n, float lr, float grad_scale);
/* ms = rho*ms + (1-rho)*grad^2; master -= lr*grad/(sqrt(ms)+eps); w_lp = RNE(master) (may be NULL); grad = 0. */
int gpipe_op_rmsprop(void *stream, int dtype, float *master, float *grad, float *ms, void *w_lp, int64_t n, float lr,
                     float rho, float eps);
int gpipe_op_sgd(void *stream, int dtype, float *master, float *grad, void *w_lp, int64_t n, float lr);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif
#ifdef __cplusplus
}
#endif
#endif

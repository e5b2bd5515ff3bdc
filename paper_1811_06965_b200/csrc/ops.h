// ops.h - internal launcher interface between the engine (scheduler, planner) and the sm_100a
// kernels.  Plain pointers + sizes; every launcher enqueues on ctx.stream and returns the CUDA
// status of the launch.  `dt` selects the storage type of tensor-core operands ("lp" tensors):
// GP_F32 -> float (SIMT FMA path, TF32 off), GP_BF16 -> __nv_bfloat16.  The residual stream,
// LayerNorm statistics, biases, gains, losses and all gradients of parameters are always fp32.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gp {

enum { GP_F32 = 0, GP_BF16 = 1 };

struct Ctx {
  cudaStream_t stream;
  int64_t *launches;   // host counter, incremented once per kernel launch
  int sm_count;
  int gemm_backend;    // 0 = auto (tcgen05 for bf16, SIMT for fp32), 1 = force SIMT, 2 = tcgen05 or fail,
                       // 3 = tcgen05 with 256 x 256 pair tiles or fail, 4 = tcgen05 with 256 x 512 pair tiles or fail
  int device;          // CUDA device ordinal the stream belongs to (per-device function attributes)
  int streams = 1;     // streams that share the GPU with this launch (the cells of a pipeline on this device):
                       // with >= 8 the GEMMs take 256 x 512 pair tiles wherever they can (gemm_tcgen05.cu)
};

inline size_t lp_size(int dt) { return dt == GP_BF16 ? 2 : 4; }

// ---- GEMM ---------------------------------------------------------------------------------
// C[M,N] = epilogue( op(A)[M,K] * op(B)[K,N] ), fp32 accumulation.
//   transA == 0: A stored [M,K] row-major (lda >= K);  transA == 1: A stored [K,M] (lda >= M)
//   transB == 0: B stored [K,N] row-major (ldb >= N);  transB == 1: B stored [N,K] (ldb >= K)
// Epilogue, in this order: +bias[n]; relu; *maskbit[m,n]; +resid[m,n]; +C_old[m,n]; store; bits out.
enum {
  EPI_BIAS = 1,       // bias: fp32 [N]
  EPI_RELU = 2,
  EPI_MASK = 4,       // mask: bit-packed uint32 [M, ldmask] (bit n%32 of word n/32); keeps v where the bit
                      // is set, else 0 (ReLU backward); ldmask >= ceil(N/32)
  EPI_RESID = 8,      // resid: fp32 [M, ldc]  (may alias C)
  EPI_ACCUM = 16,     // C is fp32 and is read-modify-written: C += v   (wgrad accumulation)
  EPI_OUT_F32 = 32,   // C is fp32 (else lp)
  EPI_COLSUM = 64,    // colsum_out[n] += sum_m C[m,n] (of the stored, rounded values); needs colsum_scratch
  EPI_BITS_OUT = 128  // mask (same layout as EPI_MASK) is WRITTEN: bit = [stored value > 0]
};
struct GemmArgs {
  int M, N, K;
  const void *A; int64_t lda; int transA;
  const void *B; int64_t ldb; int transB;
  void *C; int64_t ldc;
  const float *bias;
  const float *resid;
  void *mask; int64_t ldmask;      // uint32 words, ldmask in words
  int flags;
  float *colsum_out;       // EPI_COLSUM: fp32 [N], accumulated into
  float *colsum_scratch;   // EPI_COLSUM: fp32 [ceil(M/128), N]
  void *ws; size_t ws_bytes;   // split-K workspace (gemm_splitk_ws_bytes), counters zeroed once; NULL: never split
};
cudaError_t gemm(const Ctx &c, int dt, const GemmArgs &a);
size_t gemm_splitk_ws_bytes(int M, int N, int K, int sm_count);
// true when the tcgen05 kernel handles this problem (bf16, aligned shapes)
bool gemm_tc_supported(int dt, const GemmArgs &a);

// ---- embedding ------------------------------------------------------------------------------
cudaError_t embed_fwd(const Ctx &c, int dt, const int32_t *tok, const void *emb, const float *pe,
                      float *x, int64_t n_tok, int S, int d);
cudaError_t embed_bwd(const Ctx &c, const int32_t *tok, const float *dx, float *gemb,
                      int64_t n_tok, int d);
cudaError_t positional_table(const Ctx &c, float *pe, int S, int d);

// ---- LayerNorm ------------------------------------------------------------------------------
// y = (x - mean) * rstd * gamma + beta, biased variance; y is lp, stats fp32 [n_tok].
// resid_out (optional, fp32 [n_tok, d]) = x + resid_bias[d]: the residual-initialised output the
// branch's last GEMM accumulates into (EPI_ACCUM).
cudaError_t ln_fwd(const Ctx &c, int dt, const float *x, const float *gamma, const float *beta,
                   void *y, float *mean, float *rstd, const float *resid_bias, float *resid_out,
                   int64_t n_tok, int d, float eps);
// dx_out = (dres_in ? dres_in : 0) + LN'(dy);  dx_out_lp (optional) = lp copy of dx_out.
// partials: fp32 [ln_bwd_partial_rows(), 3, d] scratch; then dgamma += sum, dbeta += sum and,
// if colsum_out != NULL, colsum_out[n] += sum_t dx_out[t,n] (the lp copy's values when there is one).
int ln_bwd_partial_rows(int sm_count);
cudaError_t ln_bwd(const Ctx &c, int dt, const void *dy, const float *x, const float *mean,
                   const float *rstd, const float *gamma, const float *dres_in, float *dx_out,
                   void *dx_out_lp, float *partials, float *dgamma, float *dbeta, float *colsum_out,
                   int64_t n_tok, int d);

// ---- bias gradient ----------------------------------------------------------------------------
// out[n] += sum_t dy[t, n]; dy is lp [n_tok, ld]; scratch: fp32 [colsum_scratch_rows(n_tok), n]
int colsum_scratch_rows(int64_t n_tok);
cudaError_t colsum_accum(const Ctx &c, int dt, const void *dy, int64_t ld, float *out, float *scratch,
                         int64_t n_tok, int n);
// out[n] += sum_r partial[r * ld + n], r = 0 .. R-1 in order
cudaError_t colsum_reduce_partials(const Ctx &c, const float *partial, int R, int n, int64_t ld, float *out);
// fp32 -> lp copy (the operand copy of a residual gradient)
cudaError_t cast_to_lp(const Ctx &c, int dt, const float *src, void *dst, int64_t n);

// ---- attention --------------------------------------------------------------------------------
// qkv: lp [n_seq*S, 3*da] (q | k | v column blocks, head h at columns h*dh);  o: lp [n_seq*S, da]
// lse: fp32 [n_seq, A, S] natural-log-sum-exp of the scaled, masked scores.
cudaError_t attn_fwd(const Ctx &c, int dt, const void *qkv, void *o, float *lse, int n_seq, int S,
                     int A, int dh, int causal);
// dqkv: lp [n_seq*S, 3*da];  dvec: fp32 scratch [n_seq, A, S]
// colpart (optional, only where attn_bwd_fuses_colsum() is true): fp32 [n_seq, 3*da], row s = sum over the tokens of
// sequence s of the stored dqkv rows - the per-sequence partials of the bias gradient db_qkv (colsum_reduce_partials
// adds them up), fused into the kernel's store path instead of a separate pass over dqkv.
bool attn_bwd_fuses_colsum(int dt, int S, int A, int dh);
cudaError_t attn_bwd(const Ctx &c, int dt, const void *qkv, const void *o, const void *d_o,
                     const float *lse, void *dqkv, float *dvec, int n_seq, int S, int A, int dh,
                     int causal, float *colpart = nullptr);

// ---- watchdog -------------------------------------------------------------------------------------
// The tcgen05 kernels bound every mbarrier wait (tcgen05.cuh); a wait that times out records where it
// was in a block of mapped host memory and traps.  watchdog_init() allocates that block once per
// process and hands it to the kernels; watchdog_describe() returns "" or a one-line diagnosis.
cudaError_t watchdog_init();
const char *watchdog_describe();

// ---- softmax cross-entropy ----------------------------------------------------------------------
// In place: logits lp [n_tok, V] -> dlogits = (softmax - onehot) * inv_T; rowloss[t] =
// (logsumexp - logit[label]) * inv_T.  Then loss_reduce sums rowloss into *loss (fp32, overwritten).
// clip > 0: the softmax sees the logits clamped to [-clip, clip] and dlogits is 0 where the clamp is active
// (reading B5); clip == 0: off.
cudaError_t softmax_ce(const Ctx &c, int dt, void *logits, const int32_t *labels, float *rowloss,
                       int64_t n_tok, int V, float inv_T, float clip = 0.f);
cudaError_t loss_reduce(const Ctx &c, const float *rowloss, float *loss, int64_t n_tok);

// ---- parameters ---------------------------------------------------------------------------------
cudaError_t sgd_apply(const Ctx &c, int dt, float *master, float *grad, void *w_lp, int64_t n,
                      float lr);
cudaError_t rmsprop_apply(const Ctx &c, int dt, float *master, float *grad, float *ms, void *w_lp, int64_t n,
                          float lr, float rho, float eps);
// data-parallel replicas: fused gradient reduce + apply + all-gather of the update over peer-mapped pointers
struct DpPeers {
  static constexpr int kMax = 16;
  float *master[kMax];       // replica p's fp32 master array (addressable from this device)
  float *grad[kMax];         // replica p's fp32 gradient array
  void *wlp[kMax];           // replica p's bf16 working copy (NULL in fp32 mode)
  float *slot;               // this replica's RMSProp slot (NULL for SGD)
};
void dp_shard(int64_t n, int rank, int world, int64_t *lo, int64_t *hi);
cudaError_t dp_apply(const Ctx &c, int dt, const DpPeers &P, int world, int self, int64_t n, float lr, float gscale,
                     int rms, float rho, float eps);
cudaError_t init_normal(const Ctx &c, int dt, float *master, void *w_lp, int64_t n, uint64_t seed,
                        uint64_t stream_id, float mean, float std);
cudaError_t fill_f32(const Ctx &c, float *p, int64_t n, float v);
cudaError_t master_to_lp(const Ctx &c, int dt, float *master, void *w_lp, int64_t n, int round_master);
cudaError_t lp_to_f32(const Ctx &c, int dt, const void *src, float *dst, int64_t n);
cudaError_t check_ids(const Ctx &c, const int32_t *ids, int64_t n, int V, int *flag);

}  // namespace gp

/* gpipe.h - C ABI of the B200-native GPipe hot path (libgpipe_b200.so).
 *
 * What the library computes (citations: /root/reference/PAPER.md line numbers, arXiv 1811.06965):
 *   A model is "a sequence of L layers" partitioned into K consecutive cells (2.1;
 *   the user specifies "(i) the number of model partitions K, (ii) the number of micro-batches
 *   M, and (iii) the sequence and definitions of L layers").  Every mini-batch of
 *   N sequences is divided into M equal micro-batches which are pipelined through the K cells;
 *   the backward pass of each micro-batch uses the same parameters as its forward pass;
 *   gradients of all M micro-batches are accumulated and applied once per mini-batch
 *   (2.2).  With re-materialization each cell stores only its boundary (input)
 *   activation and recomputes its forward F_k just before its backward (2.3); the
 *   recompute does not wait for the upstream gradient.
 *   The layers are pre-LayerNorm self-attention + ReLU-FFN Transformer layers
 *   (BASELINE.json north_star; readings A2-A8), the loss is the token-mean softmax
 *   cross-entropy of the whole mini-batch.
 *
 * On one GPU the K cells are K CUDA streams with event dependencies F(k,m) <- F(k-1,m),
 * B(k,m) <- B(k+1,m) (Fig. 2c).  All arithmetic runs in the library's own
 * sm_100a kernels.  There is no CPU fallback: every call fails with GPIPE_ECUDA if no device
 * is usable.
 *
 * Conventions
 *   - Status: 0 = success, negative = error; gpipe_last_error() returns a thread-local,
 *     NUL-terminated message for the last failing call on this thread.  Nothing aborts or
 *     throws across this boundary.
 *   - "host" / "device" is stated per pointer.  All matrices are row-major, y = x * W.
 *   - The library never allocates device memory: the caller passes one arena and K streams
 *     (PyTorch supplies both in the Python binding).  The arena must stay alive and untouched
 *     until gpipe_destroy.
 *   - Canonical tensor order (index i of gpipe_tensor_info / get / set):
 *       emb [V,d];
 *       per layer l: ln1_g [1,d], ln1_b [1,d], w_qkv [d,3*da] (column blocks q|k|v, head h owns
 *       columns h*d_head.. of each block), b_qkv [1,3*da], w_o [da,d], b_o [1,d], ln2_g, ln2_b,
 *       w_1 [d,H], b_1 [1,H], w_2 [H,d], b_2 [1,d];
 *       lnf_g [1,d], lnf_b [1,d], w_out [d,V].     (da = n_heads * d_head)
 */
#ifndef GPIPE_H_
#define GPIPE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#pragma GCC visibility push(default)   /* the library is built with -fvisibility=hidden */
#endif

#define GPIPE_OK        0
#define GPIPE_EINVAL   -1   /* bad argument / unsupported shape; message says which            */
#define GPIPE_ECUDA    -2   /* CUDA runtime/driver error; message carries the CUDA error string */
#define GPIPE_ENOMEM   -3   /* arena too small; message carries the needed byte count           */
#define GPIPE_ENOTIMPL -4

#define GPIPE_DTYPE_FP32 0  /* fp32 storage and arithmetic everywhere, TF32 off (SIMT FMA)      */
#define GPIPE_DTYPE_BF16 1  /* bf16 weights/activations as tensor-core operands, fp32 residual
                               stream, fp32 accumulation, fp32 master weights and gradients      */

/* peak-HBM categories (index into by_category[]) */
#define GPIPE_CAT_WEIGHTS   0   /* working copy of the parameters (bf16 in bf16 mode, else fp32) */
#define GPIPE_CAT_MASTERS   1   /* fp32 master copy (bf16 mode only)                             */
#define GPIPE_CAT_GRADS     2   /* fp32 gradient accumulators                                    */
#define GPIPE_CAT_BOUNDARY  3   /* K*M cell-boundary activations + boundary-gradient ring        */
#define GPIPE_CAT_INTERIOR  4   /* per-cell interior workspaces (x M when remat is off)          */
#define GPIPE_CAT_HEAD      5   /* logits / dlogits workspace, loss partials                     */
#define GPIPE_CAT_MISC      6   /* token ids, positional table, reduction scratch                */
#define GPIPE_CAT_BWD       7   /* backward-pass scratch of a cell (activation gradients)        */
#define GPIPE_NUM_CATS      8

typedef struct gpipe gpipe_t;   /* opaque handle, owned by the library */

/* "the sequence and definitions of L layers": n_layers identical Transformer
 * layers that differ only in their attention mask. */
typedef struct {
  int32_t n_layers;     /* L >= 0                                                              */
  int32_t d_model;      /* d, multiple of 4 (bf16 mode: multiple of 64)                        */
  int32_t d_ffn;        /* H, multiple of 4 (bf16 mode: multiple of 32)                        */
  int32_t n_heads;      /* A                                                                   */
  int32_t d_head;       /* 0 -> d_model / n_heads.  Supported: 16, 32, 64, 128                 */
  int32_t vocab;        /* V                                                                   */
  int32_t seq_len;      /* S, every sequence has exactly S tokens (dense batches)              */
  int32_t dtype;        /* GPIPE_DTYPE_*                                                       */
  const uint8_t *causal;/* host, [n_layers] 0/1, read during gpipe_create only; NULL = all 1   */
  float   ln_eps;       /* 0 -> 1e-5                                                           */
} gpipe_layer_spec;

typedef struct {
  void   *arena;        /* device, >= gpipe_plan_bytes(), 1024-byte aligned                    */
  size_t  arena_bytes;
  void *const *streams; /* host array of n_streams cudaStream_t, one per cell (n_streams >= K).
                         * n_streams >= 2K: streams[K + k] is cell k's second stream - the weight-gradient
                         * GEMMs of B(k,m) run there, beside the cell's dgrad / LayerNorm / attention chain
                         * (same kernels, same accumulation order: bitwise the same gradients)          */
  int32_t n_streams;
} gpipe_env;

/* One scheduled task of a traced step (gpipe_trace): kind 'F' forward, 'R' re-materialization
 * replay, 'B' backward; start/end in milliseconds since the step's first enqueue (CUDA events
 * on the cell's stream). */
typedef struct {
  int32_t kind, k, m, enqueue_index;
  float   start_ms, end_ms;
} gpipe_trace_event;

/* Bytes of arena that gpipe_create needs for (spec, K, M, remat) and a mini-batch of n_seqs
 * sequences (O(N + (L/K)(N/M)) activations with remat).  Host only, no CUDA. */
int gpipe_plan_bytes(const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs,
                     size_t *bytes_out);

/* gpipe_create(layer_spec, K, M, remat) of BASELINE.json.  1 <= K <= max(L,1); the first
 * L mod K cells get one more layer; M >= 1; n_seqs % M == 0 ("M equal micro-batches",
 * PAPER.md:67).  n_seqs fixes the mini-batch size the plan is built for.  Parameters start at
 * zero (LayerNorm gains too): call gpipe_init_params or gpipe_set_param. */
int gpipe_create(const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs,
                 const gpipe_env *env, gpipe_t **out);
void gpipe_destroy(gpipe_t *g);

/* ---- cell partitioning ("consecutive layers between layers i and j"; "the
 * partitioning algorithm minimizes the variance in the estimated cost of all cells") ----
 *
 * gpipe_layer_costs: the per-token FLOP estimate c_i of every layer of `spec` (forward + backward, plus the replayed
 * forward when remat != 0; SURVEY.md 8(d) formulas: causal layers count the unmasked half of the attention
 * products), the cost the embedding adds to cell 0 (0: a gather) and the cost the head (final LayerNorm, logits,
 * loss) adds to cell K-1.  Host only.  layer_cost_out: host [n_layers]; any out pointer may be NULL.
 *
 * gpipe_partition_min_variance: boundaries cell_lo_out[K+1] (host; cell k = layers [lo[k], lo[k+1]), lo[0] = 0,
 * lo[K] = L, every cell non-empty) that minimise the variance of C_k = sum of layer_cost over the cell
 * (+ first_extra for k = 0, + last_extra for k = K-1) over ALL consecutive partitions - exact (dynamic
 * program); among equal minima the one with the earliest boundaries.  Needs 1 <= K <= L, costs >= 0. Host only.
 *
 * gpipe_create_partitioned: gpipe_create with explicit boundaries cell_lo[K+1] (host, read during the call).
 * The arena need is the same as gpipe_plan_bytes reports (it does not depend on the boundaries).
 * gpipe_cell_range: the layers [*lo, *hi) cell k of a handle runs. */
int gpipe_layer_costs(const gpipe_layer_spec *spec, int remat, double *layer_cost_out, double *embed_cost,
                      double *head_cost);
int gpipe_partition_min_variance(const double *layer_cost, int L, double first_extra, double last_extra, int K,
                                 int32_t *cell_lo_out);
int gpipe_create_partitioned(const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs,
                             const gpipe_env *env, const int32_t *cell_lo, gpipe_t **out);
int gpipe_cell_range(const gpipe_t *g, int k, int32_t *lo, int32_t *hi);

/* ---- the pipeline across accelerators ("GPipe places the k-th cell on the k-th
 * accelerator", "only needs to pass activation tensors at the partition boundaries") ----
 * gpipe_create_pipeline builds the same engine with ONE arena, ONE stream and ONE device PER CELL: cell k's
 * parameters, gradient accumulators, optimizer slots, boundary slots, interior workspaces and scratch live in
 * cells[k].arena on device cells[k].device, and its tasks F(k,m), R(k,m), B(k,m) run on cells[k].stream.  The only
 * tensors that move between arenas are the boundary activation ([T_mb, d] fp32, forward) and its gradient (fp32 +
 * the bf16 operand copy, backward): cudaMemcpyPeerAsync on the producing cell's stream, ordered with the consumer
 * by the same events as the single-device schedule (cudaStreamWaitEvent works across devices of one process).
 * Token ids go to cell 0's device, labels to cell K-1's.  The schedule, the kernels and therefore every result
 * are those of gpipe_create (bitwise, except the FFN2 bias gradient of each cell's last layer, which the owning
 * cell now sums itself).  All devices must be visible to THIS process; the call enables peer access between
 * neighbouring cells' devices.  Cells may share a device (cells[k].device all equal): the same code path on one
 * GPU - how the single-GPU tests cover it; flags & GPIPE_PIPE_STAGED then forces the staged boundary copies that
 * different devices always use.  One handle = one host thread driving K devices; the step is enqueued eagerly
 * (no CUDA graph) when the devices differ.  gpipe_plan_bytes_pipeline: bytes each cell's arena needs (host only;
 * cell_lo may be NULL for the equal split).  Optimizer slots: gpipe_attach_optimizer_slots_cell per cell
 * (gpipe_cell_param_count(k) * 4 bytes on that cell's device). */
typedef struct {
  int32_t device;       /* CUDA device ordinal of this cell                                    */
  void   *arena;        /* device memory ON THAT DEVICE, >= gpipe_plan_bytes_pipeline()[k], 1024-byte aligned */
  size_t  arena_bytes;
  void   *stream;       /* cudaStream_t created on that device                                 */
} gpipe_cell_env;
#define GPIPE_PIPE_STAGED 1
int gpipe_plan_bytes_pipeline(const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs,
                              const int32_t *cell_lo, size_t *bytes_out /* [K] */);
int gpipe_create_pipeline(const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs,
                          const gpipe_cell_env *cells /* [K] */, const int32_t *cell_lo, int flags, gpipe_t **out);
int gpipe_attach_optimizer_slots_cell(gpipe_t *g, int k, void *slots_dev, size_t bytes);
int gpipe_cell_param_count(const gpipe_t *g, int k, int64_t *n_out);

/* ---- the encoder-decoder Transformer T(L,H,A) on the same schedule ----
 * PAPER.md:160 (footnote 1): "T(L,H,A) is a Transformer model with L encoder layers and L decoder layers, a
 * feed-forward hidden dimension of H and A attention heads.  The model dimension is fixed to 1024"; PAPER.md:174:
 * "we clip the logit predictions (softmax pre-activations) whenever their magnitude exceeds a certain value" and "we
 * scale down the initialization of all transformer feed-forward layers by the number of layers".
 * The model is still ONE sequence of layers enc_0 .. enc_{n_enc-1}, dec_0 .. dec_{n_dec-1} cut into K cells of
 * consecutive layers; M micro-batches, boundary-only storage and replay are unchanged.  What crosses a
 * cell boundary is a PAIR (x, aux): in the encoder x is the source stream and aux the target embedding; the cell
 * holding dec_0 forms the memory LN_e(x_src), and from there x is the target stream and aux the memory.
 * Readings (B1-B6): an encoder layer is the layer of gpipe_layer_spec without mask; a decoder layer
 * is causal self-attention, then cross-attention (pre-LN on the target stream; queries from it, keys / values from
 * the memory, no mask), then the ReLU FFN; one embedding table for source and target ids, untied w_out; source
 * and target both have seq_len tokens.
 * Canonical tensor order: emb; per layer l = 0 .. n_enc+n_dec-1: [lne_g, lne_b in front of layer n_enc;] ln1_g,
 * ln1_b, w_qkv, b_qkv, w_o, b_o, [decoder layers: lnx_g, lnx_b, w_q [d,da], b_q, w_kv [d,2*da] (k|v), b_kv,
 * w_o2 [da,d], b_o2,] ln2_g, ln2_b, w_1, b_1, w_2, b_2; lnf_g, lnf_b, w_out.
 * gpipe_create_encdec: as gpipe_create; cell_lo (host, K+1 boundaries over the n_enc+n_dec layers) may be NULL for
 * the equal split; 1 <= K <= n_enc + n_dec.  gpipe_step_encdec: src, tgt, labels are HOST int32 [n_seqs, seq_len]
 * (labels[t] = the target id the decoder must predict at position t); gpipe_step_encdec_device: the same ids already
 * in HBM.  gpipe_step / gpipe_step_device on such a handle (and these on a plain handle) return GPIPE_EINVAL.
 * Every other call (apply, parameters, tracker, trace, graph, data-parallel apply) works unchanged.
 * gpipe_create_pipeline_encdec / gpipe_plan_bytes_pipeline_encdec: the same model on the pipeline handle of
 * gpipe_create_pipeline (one arena, stream and device per cell): BOTH members of the boundary pair and both of its
 * gradient travel between neighbouring cells (store and forward: every cell keeps its own copy of the target embedding
 * or of the memory and passes it on with its output). */
typedef struct {
  int32_t n_enc, n_dec; /* >= 1 each                                                           */
  int32_t d_model, d_ffn, n_heads, d_head, vocab, seq_len, dtype;   /* as gpipe_layer_spec    */
  float   ln_eps;       /* 0 -> 1e-5                                                           */
  float   logit_clip;   /* c >= 0; 0 = no clipping                                             */
} gpipe_encdec_spec;
int gpipe_plan_bytes_encdec(const gpipe_encdec_spec *spec, int K, int M, int remat, int64_t n_seqs,
                            const int32_t *cell_lo, size_t *bytes_out);
/* gpipe_layer_costs for this model ("estimated cost"): a decoder layer adds the cross-attention block's
 * projections (2 * 4 d d_a FLOPs per token) and one unmasked attention over the seq_len memory positions.  The result
 * feeds gpipe_partition_min_variance; layer_cost_out: host [n_enc + n_dec]. */
int gpipe_layer_costs_encdec(const gpipe_encdec_spec *spec, int remat, double *layer_cost_out, double *embed_cost,
                             double *head_cost);
int gpipe_create_encdec(const gpipe_encdec_spec *spec, int K, int M, int remat, int64_t n_seqs,
                        const gpipe_env *env, const int32_t *cell_lo, gpipe_t **out);
int gpipe_plan_bytes_pipeline_encdec(const gpipe_encdec_spec *spec, int K, int M, int remat, int64_t n_seqs,
                                     const int32_t *cell_lo, size_t *bytes_out /* [K] */);
int gpipe_create_pipeline_encdec(const gpipe_encdec_spec *spec, int K, int M, int remat, int64_t n_seqs,
                                 const gpipe_cell_env *cells /* [K] */, const int32_t *cell_lo, int flags, gpipe_t **out);
int gpipe_step_encdec(gpipe_t *g, const int32_t *src, const int32_t *tgt, const int32_t *labels, float *loss_out);
int gpipe_step_encdec_device(gpipe_t *g, const int32_t *src_dev, const int32_t *tgt_dev, const int32_t *labels_dev,
                             float *loss_out);

/* N(0, std) for matrices and emb, from a counter-based generator on the device (Philox-4x32-10
 * + Box-Muller); parity != 0 also draws biases / beta ~ N(0,std) and gamma = 1 + N(0,std)
 * (reading A10), parity == 0 sets gamma = 1, beta = bias = 0.  bf16 mode: the master is the
 * RNE-bf16-rounded draw (reading A12). */
int gpipe_init_params(gpipe_t *g, uint64_t seed, float std, int parity);
/* The same draw with the FFN matrices w_1, w_2 of every layer drawn at std * ffn_scale ("we scale down
 * the initialization of all transformer feed-forward layers by the number of layers": ffn_scale = 1 / n_layers). */
int gpipe_init_params_scaled(gpipe_t *g, uint64_t seed, float std, int parity, float ffn_scale);

/* gpipe_step(tokens, labels) -> loss.  tokens, labels: HOST, int32 [n_seqs, seq_len] row-major,
 * values in [0, V), read during the call only.  Runs the whole GPipe schedule (forward ticks,
 * then backward ticks with replay), ADDS d(mean loss)/dw into the fp32 gradient buffers and
 * writes the mini-batch mean loss to *loss_out (host).  Synchronous on return. */
int gpipe_step(gpipe_t *g, const int32_t *tokens, const int32_t *labels, float *loss_out);

/* Same with DEVICE-resident int32 ids (inputs already in HBM); loss still returned to host. */
int gpipe_step_device(gpipe_t *g, const int32_t *tokens_dev, const int32_t *labels_dev,
                      float *loss_out);

/* w <- w - lr * g for every parameter, once per mini-batch, then g <- 0.
 * bf16 mode updates the fp32 master and re-rounds the bf16 working copy. */
int gpipe_apply_sgd(gpipe_t *g, float lr);
int gpipe_zero_grads(gpipe_t *g);

/* RMSProp, the optimizer the paper's memory table assumes ("Each model parameter needs 12 bytes since we applied
 * RMSProp": weight + gradient + one slot).  The slot is caller-owned DEVICE memory
 * (the library never allocates): gpipe_optimizer_slot_bytes() bytes, 16-byte aligned, handed over once with
 * gpipe_attach_optimizer_slots (zeroed there; must outlive the handle).  gpipe_apply_rmsprop, once per mini-batch:
 *   ms <- rho * ms + (1 - rho) * g^2;   w <- w - lr * g / (sqrt(ms) + eps);   g <- 0        (reading A20)
 * bf16 mode updates the fp32 master and re-rounds the bf16 working copy.  0 <= rho < 1, eps > 0 (a parameter
 * whose gradient is exactly zero then stays put: 0 / (0 + eps)). */
int gpipe_optimizer_slot_bytes(const gpipe_t *g, size_t *bytes_out);
int gpipe_attach_optimizer_slots(gpipe_t *g, void *slots_dev, size_t bytes);
int gpipe_apply_rmsprop(gpipe_t *g, float lr, float rho, float eps);

/* ---- data-parallel replicas with the gradient reduction fused into the apply (PAPER.md:45:
 * GPipe "can be complemented with data parallelism to further scale training") ----
 * R replicas - one handle per GPU, created with the same spec, K, M, remat and n_seqs, started from the same
 * parameters - each run gpipe_step on their own mini-batch.  gpipe_dp_apply_* then replaces gpipe_apply_*: replica
 * `rank` owns the shard gpipe_dp_shard(n_flat, rank, world) of the flat parameter range and, in ONE kernel, sums
 * that shard's gradients over all replicas (loads through peer_arenas[p], rank order, times grad_scale - 1/R for
 * the mean over replicas, which with equal mini-batch sizes is the mean loss of the union), zeroes them in every
 * replica, applies the update to its master shard (SGD, or RMSProp with its own slot shard) and stores the new
 * master and working-copy values into every replica: reduce-scatter + optimizer + all-gather over NVLink peer
 * memory with no staging buffer and no collective call.  All replicas end with bit-identical parameters.
 *   peer_arenas: HOST array of `world` DEVICE pointers, peer_arenas[p] = the address under which THIS process
 *   reaches replica p's arena (its own arena for p == rank; a CUDA-IPC mapping - gpipe_ipc_export / gpipe_ipc_open -
 *   or, several handles in one process, the other handle's arena).  Offsets inside the arena are the same for every
 *   replica (gpipe_dp_layout reports them).
 *   Ordering: the kernel waits on no other replica.  The CALLER separates the phases: every replica's gpipe_step has
 *   returned before any replica calls gpipe_dp_apply_*, and every replica's gpipe_dp_apply_* has returned before
 *   the next gpipe_step (torch.distributed barriers in the Python binding).  Synchronous on return. */
int gpipe_dp_shard(int64_t n_flat, int rank, int world, int64_t *lo, int64_t *hi);      /* host only */
int gpipe_dp_layout(const gpipe_t *g, int64_t *n_flat, size_t *master_off, size_t *grad_off, size_t *wlp_off);
int gpipe_dp_apply_sgd(gpipe_t *g, int rank, int world, void *const *peer_arenas, float lr, float grad_scale);
int gpipe_dp_apply_rmsprop(gpipe_t *g, int rank, int world, void *const *peer_arenas, float lr, float rho, float eps,
                           float grad_scale);
/* CUDA IPC for the peer arenas: handle (64 bytes, host) of the device ALLOCATION containing dev_ptr plus dev_ptr's
 * byte offset in it; gpipe_ipc_open maps a peer's allocation into this process (returns its base; add the offset);
 * gpipe_ipc_close unmaps it. */
int gpipe_ipc_export(const void *dev_ptr, unsigned char *handle_out, size_t *offset_out);
int gpipe_ipc_open(const unsigned char *handle, void **base_out);
int gpipe_ipc_close(void *base);

int gpipe_num_tensors(const gpipe_t *g);
/* *name points into library-owned storage valid until gpipe_destroy. */
int gpipe_tensor_info(const gpipe_t *g, int i, const char **name, int64_t *rows, int64_t *cols);
/* host_out / host_in: HOST fp32 [rows*cols].  get_param returns the values the kernels use
 * (bf16 mode: the bf16 working copy widened).  set_param in bf16 mode RNE-rounds into both the
 * master and the working copy. */
int gpipe_get_param(gpipe_t *g, int i, float *host_out);
int gpipe_set_param(gpipe_t *g, int i, const float *host_in);
int gpipe_get_grad(gpipe_t *g, int i, float *host_out);

/* Exact training state, for checkpoint / resume (a step is deterministic, so save -> restore -> step reproduces an
 * uninterrupted run bit for bit).  gpipe_get_master / gpipe_set_master move the fp32 MASTER copy of tensor i with
 * no rounding (bf16 mode: set_master re-derives the bf16 working copy as RNE(master); fp32 mode: same as
 * get/set_param).  gpipe_get_optimizer_slot / gpipe_set_optimizer_slot move the RMSProp second-moment slot of
 * tensor i (GPIPE_EINVAL until gpipe_attach_optimizer_slots was called).  host_out / host_in: HOST fp32
 * [rows*cols]. */
int gpipe_get_master(gpipe_t *g, int i, float *host_out);
int gpipe_set_master(gpipe_t *g, int i, const float *host_in);
int gpipe_get_optimizer_slot(gpipe_t *g, int i, float *host_out);
int gpipe_set_optimizer_slot(gpipe_t *g, int i, const float *host_in);

/* Peak-HBM tracker: bytes the engine holds at its high-water mark, total, by category
 * (by_category[GPIPE_NUM_CATS], may be NULL) and by cell (by_cell[K], activations and scratch
 * owned by that cell; may be NULL). */
int gpipe_peak_bytes(const gpipe_t *g, size_t *total, size_t *by_category, size_t *by_cell);

/* Tasks that run.  A step runs the tasks of Fig. 2c - F(k,m), then per cell for m = M-1..0 the replay
 * R(k,m) (remat only) and B(k,m) - except work whose result is already resident or never read (readings A15,
 * A15b, A15c; results are bitwise those of running everything): with remat, R(k, M-1) for k < K-1 is elided (the cell's
 * workspace still holds the interior of F(k, M-1) when B(k, M-1) starts), every F(K-1, m) is elided (the last cell's
 * forward has no consumer but the loss, which R(K-1, m) produces again; the loss partial is taken from the replay),
 * and a replay of cells 0..K-2 skips the cell's last FFN2.  The trace shows exactly the tasks that ran.
 *
 * enable != 0: subsequent steps record one gpipe_trace_event per task.  With events_out != NULL
 * copies up to *n_events events of the last step and sets *n_events to the number written;
 * with events_out == NULL sets *n_events to the number available. */
int gpipe_trace(gpipe_t *g, int enable, gpipe_trace_event *events_out, int64_t *n_events);

/* Per-launch timing for the roofline report: with enable != 0 every kernel launch of the following
 * steps is bracketed by CUDA events on its stream and accumulated per kernel class (enabling
 * resets the counters).  gpipe_kernel_stats returns, for class cls in [0, GPIPE_NUM_KCLASSES):
 * its name, launches, summed device milliseconds, and summed ALGORITHMIC flops and bytes
 * (2MNK per GEMM; operand + output bytes once).  enable bit 1 (value 2 or 3)
 * additionally serialises all cells onto stream 0, so that each launch is timed running alone. */
#define GPIPE_NUM_KCLASSES 10
int gpipe_kernel_timing(gpipe_t *g, int enable);
int gpipe_kernel_stats(const gpipe_t *g, int cls, const char **name, int64_t *count, double *ms,
                       double *flops, double *bytes);

/* Number of kernels the library launched since gpipe_create (for bench.py's gpu_launches). */
int64_t gpipe_launch_count(const gpipe_t *g);

/* CUDA graph of the step (on by default): the first gpipe_step of a handle enqueues its ~(M K) tasks eagerly on the
 * K streams, the second captures the same fork / join DAG into a CUDA graph (the memory plan is static: every
 * pointer and TMA descriptor of a step is the same each time) and every later step is one cudaGraphLaunch - the
 * host then spends microseconds per step instead of enqueueing tens of thousands of launches.  Results are
 * bit-identical to eager enqueue (same kernels, same dependencies).  Steps with gpipe_trace or gpipe_kernel_timing
 * enabled enqueue eagerly.  gpipe_cuda_graph(g, 0) switches the graph off (and frees it), 1 on again.
 * gpipe_cuda_graph_state: 0 = eager so far, 1 = next step captures, 2 = replaying a graph, -1 = capture failed and
 * the handle stays eager (not an error). */
int gpipe_cuda_graph(gpipe_t *g, int enable);
int gpipe_cuda_graph_state(const gpipe_t *g);

/* Debug/verification taps for the per-kernel parity tests: copies a named device buffer of the
 * LAST executed (cell k, micro-batch m) task to host as fp32.  layer >= 0: "a", "qkv", "o", "c", "h", "x1",
 * "lse", and "hbits" - the bit-packed ReLU pattern [h > 0] (bit n%32 of word n/32, [T_mb, ceil(H/32)] uint32
 * words copied bit-exact into the 4-byte slots of host_out; reading A14 (iii)).  layer < 0: "y", "dlogits", "x_out". */
int gpipe_debug_read(gpipe_t *g, const char *what, int layer, float *host_out, int64_t max_elems,
                     int64_t *n_elems);

const char *gpipe_last_error(void);
const char *gpipe_version(void);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif
#ifdef __cplusplus
}
#endif
#endif /* GPIPE_H_ */

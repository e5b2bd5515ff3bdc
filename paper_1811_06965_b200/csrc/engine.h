// engine.h - host-side state of one gpipe handle: parameter inventory, memory plan (arena carving
// + peak-HBM tracker), cell workspaces, and the GPipe scheduler (K streams, events, replay).
#pragma once
#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "../../include/gpipe.h"
#include "ops.h"

namespace gp {

struct TensorInfo {
  std::string name;
  int64_t rows, cols;
  int64_t off;        // element offset into the flat master / grad / lp arrays (canonical order)
  bool matrix;        // matrices are tensor-core operands (lp working copy); vectors stay fp32
  int cell = 0;       // the cell that owns the tensor (emb: 0, final LN / w_out: K-1, layer l: its cell)
};

struct LayerParams {  // indices into Engine::tensors
  int ln1_g, ln1_b, w_qkv, b_qkv, w_o, b_o, ln2_g, ln2_b, w_1, b_1, w_2, b_2;
  // decoder layers of an encoder-decoder handle: the cross-attention block; -1 otherwise
  int lnx_g = -1, lnx_b = -1, w_q = -1, b_q = -1, w_kv = -1, b_kv = -1, w_o2 = -1, b_o2 = -1;
};

// Interior activations of one layer that the backward pass needs.
struct LayerBuf {
  void *a, *qkv, *o, *c, *h;             // lp
  uint32_t *hbits;                       // [T_mb, H/32] bit-packed ReLU pattern [h > 0] (written by FFN1's epilogue)
  float *x1, *x2;                        // fp32 residual stream (x2 unused for the cell's last layer)
  float *lse, *mean1, *rstd1, *mean2, *rstd2;
  // decoder layer: cx = LN_x(x1); qkv2 = [cx W_q + b_q | mem W_kv + b_kv] in the [q|k|v] layout of qkv, so the same
  // attention kernels serve the cross-attention; o2 its output; x1c = x1 + o2 W_o2 + b_o2
  void *cx = nullptr, *qkv2 = nullptr, *o2 = nullptr;
  float *x1c = nullptr, *lse2 = nullptr, *meanx = nullptr, *rstdx = nullptr;
};

struct Workspace {                       // one per cell (remat) or per (cell, micro-batch)
  float *x_emb = nullptr;                // cell 0: embedding output
  float *x_out = nullptr;                // last cell: x_L; other cells: replay output scratch
  std::vector<LayerBuf> layers;
  float *meanf = nullptr, *rstdf = nullptr, *rowloss = nullptr;   // head (last cell)
  void *y = nullptr, *logits = nullptr;
  // encoder-decoder: the cell that holds the first decoder layer turns the source stream into the memory
  float *aux_emb = nullptr;              // cell 0 when it also holds the transition: the target embedding
  void *mem = nullptr;                   // transition cell: LN_e(x_src) (lp), as replayed / when no later cell reads it
  float *mean_e = nullptr, *rstd_e = nullptr;
};

struct BwdScratch {                      // one per cell
  float *dx[2];                          // residual-gradient ping-pong, fp32 [T_mb, d]
  void *dx_lp[2];                        // lp operand copies (bf16 mode)
  void *dh, *dc, *d_o, *dqkv;            // lp activation gradients
  float *dvec;                           // attention D = rowsum(dO*O)
  float *ln_partials;
  float *colsum_scratch;                 // [max(T_mb/128, colsum rows), max(H, 3*da, d)]
  void *splitk_ws;                       // split-K partials + counters of this cell's GEMMs (one stream -> one user at a time)
  float *daux = nullptr;                 // encoder-decoder, transition cell: gradient of the memory (fp32, summed over the decoder layers)
  float *dtgt = nullptr;                 // ... when that cell is cell 0: gradient of the target embedding
};

struct Arena {
  char *base = nullptr;
  size_t cap = 0, used = 0;
  bool dry = true;
  size_t by_cat[GPIPE_NUM_CATS] = {0};
  std::vector<size_t> by_cell;
  void *alloc(size_t bytes, int cat, int cell);
};

// kernel classes of the per-launch timing facility (gpipe_kernel_timing / gpipe_kernel_stats)
enum KClass { KC_GEMM_FWD = 0, KC_GEMM_DGRAD, KC_GEMM_WGRAD, KC_ATTN_FWD, KC_ATTN_BWD, KC_LN_FWD, KC_LN_BWD,
              KC_CE, KC_COLSUM, KC_EMBED, KC_NUM };
struct KRec { int cls; double flops, bytes; cudaEvent_t e0, e1; };
struct KStat { int64_t count = 0; double ms = 0, flops = 0, bytes = 0; };

struct TraceRec {
  int kind, k, m, idx;
  cudaEvent_t e0, e1;
};

struct Engine {
  gpipe_layer_spec spec;
  std::vector<uint8_t> causal;
  int K = 1, M = 1, remat = 1, dt = GP_F32;
  int64_t n_seqs = 0, nb = 0, T_mb = 0, T_total = 0;   // nb = sequences per micro-batch
  int d = 0, H = 0, A = 0, dh = 0, da = 0, V = 0, S = 0;
  float eps = 1e-5f;
  // encoder-decoder T(L,H,A): layers [0, n_enc) are encoder layers, [n_enc, L) decoder
  // layers (causal self-attention + cross-attention over the encoder memory).  What crosses a cell boundary is the
  // pair (x, aux): aux = target embedding up to the transition, the memory after it.  n_dec == 0: the plain stack.
  int n_enc = 0, n_dec = 0;
  float logit_clip = 0.f;                              // > 0: logits clamped to [-c, c] before the softmax
  bool encdec() const { return n_dec > 0; }
  bool is_dec(int l) const { return n_dec > 0 && l >= n_enc; }
  int kt = 0;                                          // the cell that holds layer n_enc (the transition)
  int i_lne_g = -1, i_lne_b = -1;
  int32_t *tgt_dev = nullptr;                          // target ids (cell 0 embeds both id sequences)
  // aux_in[k][m], k = 1..K-1: the second member of cell k's input pair - the target embedding (fp32) for k <= kt, the
  // memory (lp) for k > kt.  One arena: a single buffer per micro-batch serves every cell that reads it (the hand-off
  // is a pointer, as for x).  Pipeline handle: each cell has its own copy in its own arena and forwards it to the
  // next cell with the boundary transfer (store and forward: only neighbouring devices talk).
  std::vector<std::vector<void *>> aux_in;
  std::vector<float *> dbound_aux[2];                  // [k]: gradient wrt the aux input of cell k (two-entry ring like dbound)
  std::vector<float *> dout_aux[2];                    // [k]: gradient wrt the aux OUTPUT of cell k (= dbound_aux[k+1], or its local copy)
  int sm_count = 148;                                  // of the device the handle lives on (launch geometry)
  // The memory plan must not depend on the device (gpipe_plan_bytes is host-only): scratch whose size follows the
  // launch geometry is planned for this fixed SM-count bound and the launchers clamp to what was planned.
  static constexpr int kPlanSmCount = 148;
  int device = 0;
  int gemm_backend = 0;
  int replay_full = 0;
  size_t splitk_ws_bytes = 0;

  std::vector<TensorInfo> tensors;
  std::vector<LayerParams> lp;
  int i_emb = 0, i_lnf_g = 0, i_lnf_b = 0, i_w_out = 0;
  int64_t n_flat = 0;
  float *master = nullptr, *grad = nullptr;            // single-arena mode: the whole flat range
  void *w_lp = nullptr;                                // bf16 working copy (bf16 mode), else = master

  std::vector<int> cell_lo, cell_hi;                   // layers [lo, hi) of cell k
  // Memory homes.  n_arenas == 1: one arena, one device (K streams share it).  n_arenas == K ("pipeline" handle,
  // SURVEY 8(f) f1 / PAPER.md:65 "places the k-th cell on the k-th accelerator"): cell k's parameters, gradients,
  // activations and scratch live in arena k on device cell_device[k] and run on stream k of that device; the
  // boundary activation and its gradient are the only data that cross.
  int n_arenas = 1;
  Arena arena;                                         // single-arena mode
  std::vector<Arena> parena;                           // pipeline mode: [K]
  std::vector<int> cell_device;                        // [K]
  bool multi() const { return n_arenas > 1; }
  bool multi_device = false;                           // cells on different devices (peer copies, no CUDA graph)
  int boundary_staged = 0;                             // pipeline: F_k writes its output locally, then a peer copy moves it
  Arena &ar(int k) { return multi() ? parena[k] : arena; }
  const Arena &ar(int k) const { return multi() ? parena[k] : arena; }
  std::vector<int64_t> cell_off;                       // [K+1]: cell k owns elements [cell_off[k], cell_off[k+1]) of the flat order
  std::vector<float *> cmaster, cgrad, copt;           // per-cell bases (single mode: master + cell_off[k], ...)
  std::vector<void *> cwlp;
  std::vector<float *> dout[2];                        // pipeline: local copy of the gradient wrt cell k's OUTPUT
  std::vector<void *> dout_lp[2];
  std::vector<cudaStream_t> streams;
  // Optional second stream per cell (single-arena handle with env->n_streams >= 2K): the weight-gradient GEMMs of
  // B(k, m) have no consumer inside the task, so they run beside the dgrad / LayerNorm / attention chain of the same
  // cell - what a cell's accelerator would do with them anyway when fewer than ~8 cells share the GPU.  Same kernels,
  // same accumulation order (the side stream is in-order), hence bitwise the same gradients.  side_tail[k]: the last
  // side-stream event cell k's main stream has not waited for yet (waited before the cell's next task / the join).
  std::vector<cudaStream_t> side;
  std::vector<cudaEvent_t> side_tail;
  bool side_active() const { return !side.empty() && !serial && !multi() && !trace_on; }
  std::vector<std::vector<float *>> slot;              // slot[k][m], k = 1..K-1: input of cell k
  std::vector<float *> dbound[2];                      // dbound[i][k]: gradient wrt input of cell k
  std::vector<void *> dbound_lp[2];
  std::vector<std::vector<Workspace>> ws;              // ws[k][remat ? 0 : m]
  std::vector<BwdScratch> bwd;
  int32_t *tok_dev = nullptr, *lab_dev = nullptr;
  float *pe = nullptr, *loss_parts = nullptr, *loss_dummy = nullptr;
  int *flag_dev = nullptr, *flag_dev_last = nullptr;   // id-check flags: with the tokens (cell 0) / the labels (cell K-1)
  float *host_loss = nullptr;                          // pinned
  int *host_flag = nullptr;                            // pinned

  std::vector<std::vector<cudaEvent_t>> ev_f, ev_b;    // [k][m]
  cudaEvent_t ev_in = nullptr;
  std::vector<cudaEvent_t> ev_done;                    // per stream

  // CUDA graph of one step: the K-stream fork / join DAG of run_step is captured once - the plan is
  // static, so every kernel argument and every TMA descriptor of a step is the same each time - and replayed with one
  // cudaGraphLaunch; tracing and per-launch timing enqueue eagerly.  graph_state: 0 = first step runs eagerly (sets
  // function attributes, fills the descriptor cache), 1 = capture on this step, 2 = replay, -1 = capture failed:
  // stay eager.
  int use_graph = 1;
  int graph_state = 0;
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t graph_exec = nullptr;
  int64_t graph_launches = 0;                          // kernels inside the graph (gpipe_launch_count)
  cudaError_t enqueue_step();                          // every task of a mini-batch + the loss copy, on the K streams
  void drop_graph();

  int trace_on = 0;
  std::vector<TraceRec> trace;
  std::vector<cudaEvent_t> ev_pool;
  size_t ev_pool_used = 0;
  cudaEvent_t ev_t0 = nullptr;
  int64_t launches = 0;
  int ktiming_on = 0;
  int serial = 0;                                      // debug/profiling: every cell on stream 0
  cudaStream_t st(int k) const { return streams[serial ? 0 : k]; }
  std::vector<KRec> krecs;
  float *opt_ms = nullptr;           // RMSProp second-moment slot (caller-supplied device memory, n_flat floats)
  KStat kstats[KC_NUM];
  cudaError_t resolve_kernel_timing();
  template <typename F>
  cudaError_t timed_on(cudaStream_t s, int cls, double flops, double bytes, F &&fn) {
    if (!ktiming_on) return fn();
    KRec r{cls, flops, bytes, pool_event(), pool_event()};
    if (!r.e0 || !r.e1) return pool_err;
    cudaError_t e = cudaEventRecord(r.e0, s);
    if (e != cudaSuccess) return e;
    e = fn();
    if (e != cudaSuccess) return e;
    e = cudaEventRecord(r.e1, s);
    krecs.push_back(r);
    return e;
  }
  template <typename F>
  cudaError_t timed(int k, int cls, double flops, double bytes, F &&fn) {
    return timed_on(st(k), cls, flops, bytes, static_cast<F &&>(fn));
  }

  // -- construction --
  int build_inventory(std::string &err);
  int build_plan(bool dry, std::string &err);
  // -- helpers --
  int cells_on_device(int k) const {
    if (!multi()) return K;
    int n = 0;
    for (int j = 0; j < K; ++j) n += cell_device[j] == cell_device[k];
    return n;
  }
  Ctx ctx(int k) { return Ctx{st(k), &launches, sm_count, gemm_backend, multi() ? cell_device[k] : device, cells_on_device(k)}; }
  int64_t rel(int i) const { return tensors[i].off - cell_off[tensors[i].cell]; }
  float *P(int i) const { return cmaster[tensors[i].cell] + rel(i); }  // fp32 master / vector param
  void *Wl(int i) const {                                              // bf16 working copy (bf16 mode)
    return (void *)((char *)cwlp[tensors[i].cell] + rel(i) * 2);
  }
  const void *W(int i) const {                                         // matrix operand
    return dt == GP_BF16 ? (const void *)Wl(i) : (const void *)P(i);
  }
  float *G(int i) const { return cgrad[tensors[i].cell] + rel(i); }
  float *Opt(int i) const { return copt[tensors[i].cell] + rel(i); }
  cudaError_t use(int k) const {                                       // make cell k's device current
    return multi_device ? cudaSetDevice(cell_device[k]) : cudaSuccess;
  }
  Workspace &wsp(int k, int m) { return ws[k][remat ? 0 : m]; }
  // Which of the schedule's tasks run (readings A15b / A15c).  With re-materialization the last cell's
  // forward tasks are elided (their only product, the loss, comes out of the replay again), and for every other cell
  // R(k, M-1) is: the workspace still holds F(k, M-1)'s interior when B(k, M-1) starts.
  bool forward_runs(int k) const { return !(remat && k == K - 1) || replay_full; }
  bool replay_runs(int k, int m) const { return remat && (!forward_runs(k) || m != M - 1 || replay_full); }
  // -- schedule --
  cudaError_t peer_copy(int k_dst, void *dst, int k_src, const void *src, size_t bytes, cudaStream_t s);
  cudaError_t forward_cell(int k, int m, bool replay);
  cudaError_t backward_cell(int k, int m);
  cudaError_t run_step(float *loss_out);
  cudaEvent_t pool_event();                            // nullptr (and pool_err set) when cudaEventCreate fails
  cudaError_t pool_err = cudaSuccess;
};

}  // namespace gp

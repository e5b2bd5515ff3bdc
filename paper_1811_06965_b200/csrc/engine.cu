// engine.cu - parameter inventory, memory plan / peak-HBM tracker, cell executor and the GPipe
// scheduler (PAPER.md:59-67 cells and micro-batches; :87 boundary-only storage + replay; :89 early
// replay).  Host code only: every arithmetic step is a launcher from ops.h.
#include "engine.h"

#include <stdio.h>
#include <stdlib.h>
#include <string.h>

namespace gp {

#define GP_TRY(x)                       \
  do {                                  \
    cudaError_t e__ = (x);              \
    if (e__ != cudaSuccess) return e__; \
  } while (0)

void *Arena::alloc(size_t bytes, int cat, int cell) {
  size_t a = (bytes + 1023) & ~(size_t)1023;
  size_t off = used;
  used += a;
  by_cat[cat] += a;
  if (cell >= 0 && cell < (int)by_cell.size()) by_cell[cell] += a;
  if (dry) return nullptr;
  return used <= cap ? (void *)(base + off) : nullptr;
}

// Canonical tensor list (gpipe.h); every tensor padded to a multiple of 64 elements so that the
// flat SGD / init kernels can run over one contiguous range with 16-byte vectors.
int Engine::build_inventory(std::string &err) {
  (void)err;
  tensors.clear();
  lp.clear();
  int64_t off = 0;
  auto add = [&](const std::string &name, int64_t r, int64_t c, bool matrix) {
    TensorInfo t{name, r, c, off, matrix};
    off += ((r * c + 63) / 64) * 64;
    tensors.push_back(t);
    return (int)tensors.size() - 1;
  };
  i_emb = add("emb", V, d, true);
  for (int l = 0; l < spec.n_layers; ++l) {
    std::string p = "l" + std::to_string(l) + ".";
    LayerParams q;
    if (encdec() && l == n_enc) {          // encoder output LayerNorm: in front of the first decoder layer
      i_lne_g = add("lne_g", 1, d, false);
      i_lne_b = add("lne_b", 1, d, false);
    }
    q.ln1_g = add(p + "ln1_g", 1, d, false);
    q.ln1_b = add(p + "ln1_b", 1, d, false);
    q.w_qkv = add(p + "w_qkv", d, 3 * da, true);
    q.b_qkv = add(p + "b_qkv", 1, 3 * da, false);
    q.w_o = add(p + "w_o", da, d, true);
    q.b_o = add(p + "b_o", 1, d, false);
    if (is_dec(l)) {                       // cross-attention block (canonical order of gpipe.h)
      q.lnx_g = add(p + "lnx_g", 1, d, false);
      q.lnx_b = add(p + "lnx_b", 1, d, false);
      q.w_q = add(p + "w_q", d, da, true);
      q.b_q = add(p + "b_q", 1, da, false);
      q.w_kv = add(p + "w_kv", d, 2 * da, true);
      q.b_kv = add(p + "b_kv", 1, 2 * da, false);
      q.w_o2 = add(p + "w_o2", da, d, true);
      q.b_o2 = add(p + "b_o2", 1, d, false);
    }
    q.ln2_g = add(p + "ln2_g", 1, d, false);
    q.ln2_b = add(p + "ln2_b", 1, d, false);
    q.w_1 = add(p + "w_1", d, H, true);
    q.b_1 = add(p + "b_1", 1, H, false);
    q.w_2 = add(p + "w_2", H, d, true);
    q.b_2 = add(p + "b_2", 1, d, false);
    lp.push_back(q);
  }
  i_lnf_g = add("lnf_g", 1, d, false);
  i_lnf_b = add("lnf_b", 1, d, false);
  i_w_out = add("w_out", d, V, true);
  n_flat = off;
  // owners: the canonical order is emb | layers in order | final LN, w_out and cells are consecutive layer ranges,
  // so every cell owns one contiguous range of the flat order
  tensors[i_emb].cell = 0;
  kt = 0;
  for (int k = 0; k < K; ++k)
    for (int l = cell_lo[k]; l < cell_hi[k]; ++l) {
      const LayerParams &q = lp[l];
      for (int i : {q.ln1_g, q.ln1_b, q.w_qkv, q.b_qkv, q.w_o, q.b_o, q.ln2_g, q.ln2_b, q.w_1, q.b_1, q.w_2, q.b_2,
                    q.lnx_g, q.lnx_b, q.w_q, q.b_q, q.w_kv, q.b_kv, q.w_o2, q.b_o2})
        if (i >= 0) tensors[i].cell = k;
      if (encdec() && l == n_enc) { kt = k; tensors[i_lne_g].cell = tensors[i_lne_b].cell = k; }
    }
  tensors[i_lnf_g].cell = tensors[i_lnf_b].cell = tensors[i_w_out].cell = K - 1;
  cell_off.assign(K + 1, n_flat);
  cell_off[0] = 0;
  for (int k = 1; k < K; ++k) {
    if (cell_lo[k] >= spec.n_layers) cell_off[k] = tensors[i_lnf_g].off;
    else if (encdec() && cell_lo[k] == n_enc) cell_off[k] = tensors[i_lne_g].off;
    else cell_off[k] = tensors[lp[cell_lo[k]].ln1_g].off;
  }
  return GPIPE_OK;
}

// The memory plan.  Static: everything a step needs is carved once, so the arena high-water
// mark IS the peak (with remat, K*M boundary activations ~ N plus one cell interior
// ~ (L/K)(N/M) per cell; without remat M interiors per cell ~ N*L).
int Engine::build_plan(bool dry, std::string &err) {
  auto reset = [&](Arena &a) {
    a.dry = dry;
    a.used = 0;
    memset(a.by_cat, 0, sizeof(a.by_cat));
    a.by_cell.assign(K, 0);
  };
  reset(arena);
  for (auto &a : parena) reset(a);
  size_t lpb = lp_size(dt);
  size_t Tm = (size_t)T_mb;
  // home(k): the arena of cell k; data that belongs to no cell goes to the cell that uses it
  auto RAW = [&](size_t bytes, int cat, int cell, int home) { return ar(home).alloc(bytes, cat, cell); };
  auto F32 = [&](size_t n, int cat, int cell) { return (float *)RAW(n * 4, cat, cell, cell < 0 ? 0 : cell); };
  auto LP = [&](size_t n, int cat, int cell) { return RAW(n * lpb, cat, cell, cell < 0 ? 0 : cell); };

  cmaster.assign(K, nullptr); cgrad.assign(K, nullptr); cwlp.assign(K, nullptr);
  const int cat_m = dt == GP_BF16 ? GPIPE_CAT_MASTERS : GPIPE_CAT_WEIGHTS;
  if (!multi()) {
    master = F32((size_t)n_flat, cat_m, -1);
    grad = F32((size_t)n_flat, GPIPE_CAT_GRADS, -1);
    w_lp = dt == GP_BF16 ? RAW((size_t)n_flat * 2, GPIPE_CAT_WEIGHTS, -1, 0) : (void *)master;
    for (int k = 0; k < K; ++k) {
      cmaster[k] = master ? master + cell_off[k] : nullptr;
      cgrad[k] = grad ? grad + cell_off[k] : nullptr;
      cwlp[k] = w_lp ? (void *)((char *)w_lp + cell_off[k] * (dt == GP_BF16 ? 2 : 4)) : nullptr;
    }
  } else {
    master = grad = nullptr;
    w_lp = nullptr;
    for (int k = 0; k < K; ++k) {                        // cell k's parameters live on cell k's device
      const size_t n = (size_t)(cell_off[k + 1] - cell_off[k]);
      cmaster[k] = (float *)RAW(n * 4, cat_m, -1, k);
      cgrad[k] = (float *)RAW(n * 4, GPIPE_CAT_GRADS, -1, k);
      cwlp[k] = dt == GP_BF16 ? RAW(n * 2, GPIPE_CAT_WEIGHTS, -1, k) : (void *)cmaster[k];
    }
  }

  tok_dev = (int32_t *)RAW((size_t)T_total * 4, GPIPE_CAT_MISC, -1, 0);            // the embedding is in cell 0
  lab_dev = (int32_t *)RAW((size_t)T_total * 4, GPIPE_CAT_MISC, -1, K - 1);        // the loss in cell K-1
  pe = (float *)RAW((size_t)S * d * 4, GPIPE_CAT_MISC, -1, 0);
  loss_parts = (float *)RAW((size_t)(M + 1) * 4, GPIPE_CAT_HEAD, -1, K - 1);
  loss_dummy = loss_parts ? loss_parts + M : nullptr;
  flag_dev = (int *)RAW(4, GPIPE_CAT_MISC, -1, 0);
  flag_dev_last = multi() ? (int *)RAW(4, GPIPE_CAT_MISC, -1, K - 1) : flag_dev;
  tgt_dev = encdec() ? (int32_t *)RAW((size_t)T_total * 4, GPIPE_CAT_MISC, -1, 0) : nullptr;

  slot.assign(K, std::vector<float *>(M, nullptr));
  for (int k = 1; k < K; ++k)
    for (int m = 0; m < M; ++m) slot[k][m] = F32(Tm * d, GPIPE_CAT_BOUNDARY, k);
  // encoder-decoder: the second member of the boundary pair.  One buffer per micro-batch serves every cell that
  // reads it (the hand-off is a pointer, as for x): the target embedding up to the transition cell, the memory
  // after it; its gradient travels through a two-entry ring like the gradient of x.
  aux_in.assign(K, std::vector<void *>(M, nullptr));
  if (encdec()) {
    for (int m = 0; m < M; ++m) {
      void *tgt = nullptr, *mem_ = nullptr;
      for (int k = 1; k < K; ++k) {
        if (k <= kt) {
          if (multi() || !tgt) tgt = F32(Tm * d, GPIPE_CAT_BOUNDARY, k);
          aux_in[k][m] = tgt;
        } else {
          if (multi() || !mem_) mem_ = LP(Tm * d, GPIPE_CAT_BOUNDARY, k);
          aux_in[k][m] = mem_;
        }
      }
    }
  }
  for (int i = 0; i < 2; ++i) {
    dbound_aux[i].assign(K, nullptr);
    dout_aux[i].assign(K, nullptr);
    for (int k = 1; k < K && encdec(); ++k) dbound_aux[i][k] = F32(Tm * d, GPIPE_CAT_BOUNDARY, k);
    for (int k = 0; k + 1 < K && encdec(); ++k) dout_aux[i][k] = multi() ? F32(Tm * d, GPIPE_CAT_BOUNDARY, k) : dbound_aux[i][k + 1];
  }
  for (int i = 0; i < 2; ++i) {
    dbound[i].assign(K, nullptr);
    dbound_lp[i].assign(K, nullptr);
    dout[i].assign(K, nullptr);
    dout_lp[i].assign(K, nullptr);
    for (int k = 1; k < K; ++k) {
      dbound[i][k] = F32(Tm * d, GPIPE_CAT_BOUNDARY, k);
      dbound_lp[i][k] = dt == GP_BF16 ? LP(Tm * d, GPIPE_CAT_BOUNDARY, k) : (void *)dbound[i][k];
    }
    // the gradient wrt cell k's output is produced by cell k+1: in a pipeline handle it is copied into cell k's own
    // arena (the backward boundary transfer), otherwise cell k reads it where cell k+1 left it
    for (int k = 0; k + 1 < K; ++k) {
      if (multi()) {
        dout[i][k] = F32(Tm * d, GPIPE_CAT_BOUNDARY, k);
        dout_lp[i][k] = dt == GP_BF16 ? LP(Tm * d, GPIPE_CAT_BOUNDARY, k) : (void *)dout[i][k];
      } else {
        dout[i][k] = dbound[i][k + 1];
        dout_lp[i][k] = dbound_lp[i][k + 1];
      }
    }
  }

  // split-K workspace: the largest any GEMM shape of a cell needs (forward, dgrad, wgrad); one per cell - a cell's
  // launches are ordered on its stream, so one user at a time.  Split-K buys single-kernel latency at the price of
  // SM-time (FFN2 forward at T_mb 2048: 85.8 us on 64 SMs unsplit, 68.0 us on 128 SMs split in two), so only shallow
  // pipelines split: with >= 4 cells in flight the other streams fill the SMs a few-tile GEMM leaves idle, and the
  // config-5 step measured 5 % SLOWER with every [T_mb x 1024] output split (round 2).  It also keeps the K-loop
  // order, hence every per-token forward value, independent of the micro-batch size for the deep pipelines.
  splitk_ws_bytes = 0;
  if (dt == GP_BF16 && K < 4) {
    const int T = (int)T_mb;
    const int shapes[][3] = {{T, 3 * da, d}, {T, d, da}, {T, H, d}, {T, d, H}, {T, V, d},          // forward
                             {T, da, d}, {T, d, 3 * da}, {T, d, V},                                 // dgrad (others as forward)
                             {H, d, T}, {d, H, T}, {da, d, T}, {d, 3 * da, T}, {d, V, T},             // wgrad
                             {T, da, d}, {T, 2 * da, d}, {T, d, 2 * da}, {d, da, T}, {d, 2 * da, T}};   // cross-attention
    for (auto &sh : shapes) {
      size_t b = gemm_splitk_ws_bytes(sh[0], sh[1], sh[2], kPlanSmCount);
      if (b > splitk_ws_bytes) splitk_ws_bytes = b;
    }
  }
  ws.assign(K, std::vector<Workspace>());
  bwd.assign(K, BwdScratch());
  for (int k = 0; k < K; ++k) {
    int n_ws = remat ? 1 : M;
    ws[k].resize(n_ws);
    for (int w = 0; w < n_ws; ++w) {
      Workspace &W_ = ws[k][w];
      const int cat = GPIPE_CAT_INTERIOR;
      if (k == 0) W_.x_emb = F32(Tm * d, cat, k);
      // the target embedding as cell 0's own buffer: interior when cell 0 holds the transition, staging for the boundary
      // transfer in a pipeline handle
      if (k == 0 && encdec() && (kt == 0 || multi())) W_.aux_emb = F32(Tm * d, cat, k);
      if (encdec() && k == kt) {
        W_.mem = LP(Tm * d, cat, k);
        W_.mean_e = F32(Tm, cat, k);
        W_.rstd_e = F32(Tm, cat, k);
      }
      if (k == K - 1 || remat || multi()) W_.x_out = F32(Tm * d, cat, k);   // pipeline: also the outgoing boundary staging
      int nl = cell_hi[k] - cell_lo[k];
      W_.layers.resize(nl);
      for (int i = 0; i < nl; ++i) {
        LayerBuf &b = W_.layers[i];
        b.a = LP(Tm * d, cat, k);
        b.qkv = LP(Tm * 3 * da, cat, k);
        b.o = LP(Tm * da, cat, k);
        b.c = LP(Tm * d, cat, k);
        b.h = LP(Tm * H, cat, k);
        b.hbits = (uint32_t *)RAW(Tm * (size_t)((H + 31) / 32) * 4, cat, k, k);
        b.x1 = F32(Tm * d, cat, k);
        b.x2 = i + 1 < nl ? F32(Tm * d, cat, k) : nullptr;
        b.lse = F32(Tm * A, cat, k);
        b.mean1 = F32(Tm, cat, k);
        b.rstd1 = F32(Tm, cat, k);
        b.mean2 = F32(Tm, cat, k);
        b.rstd2 = F32(Tm, cat, k);
        if (is_dec(cell_lo[k] + i)) {
          b.cx = LP(Tm * d, cat, k);
          b.qkv2 = LP(Tm * 3 * da, cat, k);
          b.o2 = LP(Tm * da, cat, k);
          b.x1c = F32(Tm * d, cat, k);
          b.lse2 = F32(Tm * A, cat, k);
          b.meanx = F32(Tm, cat, k);
          b.rstdx = F32(Tm, cat, k);
        }
      }
      if (k == K - 1) {
        W_.meanf = F32(Tm, GPIPE_CAT_HEAD, k);
        W_.rstdf = F32(Tm, GPIPE_CAT_HEAD, k);
        W_.rowloss = F32(Tm, GPIPE_CAT_HEAD, k);
        W_.y = LP(Tm * d, GPIPE_CAT_HEAD, k);
        W_.logits = LP(Tm * V, GPIPE_CAT_HEAD, k);
      }
    }
    BwdScratch &s = bwd[k];
    const int cat = GPIPE_CAT_BWD;
    for (int i = 0; i < 2; ++i) {
      s.dx[i] = F32(Tm * d, cat, k);
      s.dx_lp[i] = dt == GP_BF16 ? LP(Tm * d, cat, k) : (void *)s.dx[i];
    }
    s.dh = LP(Tm * H, cat, k);
    s.dc = LP(Tm * d, cat, k);
    s.d_o = LP(Tm * da, cat, k);
    s.dqkv = LP(Tm * 3 * da, cat, k);
    s.dvec = F32(Tm * A, cat, k);
    s.ln_partials = F32((size_t)ln_bwd_partial_rows(kPlanSmCount) * 3 * d, cat, k);
    {
      size_t rows = (Tm + 127) / 128;
      if (rows < (size_t)colsum_scratch_rows(T_mb)) rows = colsum_scratch_rows(T_mb);
      if (rows < (size_t)nb) rows = (size_t)nb;             // the attention backward's per-sequence partials of db_qkv
      size_t cols = (size_t)(H > 3 * da ? H : 3 * da);
      if (cols < (size_t)d) cols = d;
      s.colsum_scratch = F32(rows * cols, cat, k);
    }
    s.splitk_ws = splitk_ws_bytes ? RAW(splitk_ws_bytes, cat, k, k) : nullptr;
    if (encdec() && k == kt) {
      s.daux = F32(Tm * d, cat, k);
      if (k == 0) s.dtgt = F32(Tm * d, cat, k);
    }
  }
  for (int k = 0; k < (multi() ? K : 1); ++k)
    if (!dry && ar(k).used > ar(k).cap) {
      err = "arena " + std::to_string(k) + " too small: need " + std::to_string(ar(k).used) + " bytes, have " +
            std::to_string(ar(k).cap);
      return GPIPE_ENOMEM;
    }
  return GPIPE_OK;
}

cudaEvent_t Engine::pool_event() {
  if (ev_pool_used == ev_pool.size()) {
    cudaEvent_t e = nullptr;
    cudaError_t err = cudaEventCreate(&e);
    if (err != cudaSuccess) {
      pool_err = err;
      return nullptr;
    }
    ev_pool.push_back(e);
  }
  return ev_pool[ev_pool_used++];
}

// ---------------------------------------------------------------------------------------------
// F_k (and its replay): embedding (cell 0), the cell's layers, head + loss (cell K-1)
// ---------------------------------------------------------------------------------------------
cudaError_t Engine::forward_cell(int k, int m, bool replay) {
  Ctx c = ctx(k);
  const double lpb = (double)lp_size(dt);
  const double Td = (double)T_mb;
  // algorithmic bytes of a GEMM: operands once, output once (+ fused residual / accumulate reads)
  auto tgemm = [&](int cls, const GemmArgs &g) -> cudaError_t {
    double fl = 2.0 * g.M * g.N * (double)g.K;
    double outb = (g.flags & (EPI_OUT_F32 | EPI_ACCUM)) ? 4.0 : lpb;
    double by = ((double)g.M * g.K + (double)g.K * g.N) * lpb + (double)g.M * g.N * outb;
    if (g.flags & EPI_RESID) by += (double)g.M * g.N * 4.0;
    if (g.flags & EPI_ACCUM) by += (double)g.M * g.N * 4.0;
    if (g.flags & (EPI_MASK | EPI_BITS_OUT)) by += (double)g.M * g.N / 8.0;
    GemmArgs gw = g;
    gw.ws = bwd[k].splitk_ws; gw.ws_bytes = splitk_ws_bytes;
    return timed(k, cls, fl, by, [&] { return gemm(c, dt, gw); });
  };
  // rb_/ro_: fused residual init ro_ = x_ + rb_ (the branch's output GEMM then accumulates into ro_)
  auto tln = [&](const float *x_, const float *g_, const float *b_, void *y_, float *mu_, float *rs_,
                 const float *rb_, float *ro_) -> cudaError_t {
    return timed(k, KC_LN_FWD, 0, Td * d * (4.0 + lpb + (ro_ ? 4.0 : 0.0)),
                 [&] { return ln_fwd(c, dt, x_, g_, b_, y_, mu_, rs_, rb_, ro_, T_mb, d, eps); });
  };
  Workspace &w = wsp(k, m);
  const int32_t *tok = tok_dev + (int64_t)m * T_mb;
  const int32_t *lab = lab_dev + (int64_t)m * T_mb;
  float *x;
  // encoder-decoder: second member of the pair this cell works on - the target embedding (fp32) while the cell is
  // still in the encoder, the memory (lp) once it is in the decoder
  float *aux_x = nullptr;
  const void *mem = nullptr;
  if (k == 0) {
    GP_TRY(timed(k, KC_EMBED, 0, (double)T_mb * d * (lpb + 8), [&] { return embed_fwd(c, dt, tok, W(i_emb), pe, w.x_emb, T_mb, S, d); }));
    x = w.x_emb;
    if (encdec()) {
      // cell 0 embeds both id sequences (one table, reading B3).  The target embedding is cell 0's second OUTPUT:
      // written once, in the forward pass, into the buffer cells 1..kt read; a replay of cell 0 needs it only when
      // cell 0 itself holds the transition (then it is interior and recomputed)
      const int32_t *tgt = tgt_dev + (int64_t)m * T_mb;
      aux_x = w.aux_emb ? w.aux_emb : (float *)aux_in[1][m];
      if (kt == 0 || !replay) {
        GP_TRY(timed(k, KC_EMBED, 0, (double)T_mb * d * (lpb + 8), [&] { return embed_fwd(c, dt, tgt, W(i_emb), pe, aux_x, T_mb, S, d); }));
        if (multi() && kt > 0)                              // pipeline: the second member of the boundary pair travels too
          GP_TRY(peer_copy(1, aux_in[1][m], 0, aux_x, (size_t)T_mb * d * sizeof(float), c.stream));
      }
    }
  } else {
    x = slot[k][m];
    if (encdec()) {
      if (k <= kt) aux_x = (float *)aux_in[k][m];
      else mem = aux_in[k][m];
      // pipeline: store and forward - this cell's copy goes on to the next cell, unless this cell changes what aux is
      if (multi() && !replay && k + 1 < K && k != kt)
        GP_TRY(peer_copy(k + 1, aux_in[k + 1][m], k, aux_in[k][m], (size_t)T_mb * d * (k < kt ? sizeof(float) : lp_size(dt)), c.stream));
    }
  }
  int nl = cell_hi[k] - cell_lo[k];
  for (int i = 0; i < nl; ++i) {
    int l = cell_lo[k] + i;
    const LayerParams &q = lp[l];
    LayerBuf &b = w.layers[i];
    bool last = (i + 1 == nl);
    if (encdec() && l == n_enc) {
      // encoder -> decoder: memory = LN_e(x_src) (reading B2); the stream switches to the target embedding.  The
      // forward pass writes the memory where the later cells read it; a replay (and a last cell) keeps it interior.
      void *mdst = (!replay && kt < K - 1 && !multi()) ? aux_in[kt + 1][m] : w.mem;
      GP_TRY(tln(x, P(i_lne_g), P(i_lne_b), mdst, w.mean_e, w.rstd_e, nullptr, nullptr));
      if (multi() && !replay && kt < K - 1)
        GP_TRY(peer_copy(kt + 1, aux_in[kt + 1][m], kt, w.mem, (size_t)T_mb * d * lp_size(dt), c.stream));
      mem = mdst;
      x = aux_x;
    }
    // a = LN1(x); x1 <- x + b_o                                              (a5)
    GP_TRY(tln(x, P(q.ln1_g), P(q.ln1_b), b.a, b.mean1, b.rstd1, P(q.b_o), b.x1));
    // [q|k|v] = a W_qkv + b_qkv                                              (a6)
    GemmArgs g{};
    g.M = (int)T_mb; g.N = 3 * da; g.K = d;
    g.A = b.a; g.lda = d; g.B = W(q.w_qkv); g.ldb = 3 * da; g.C = b.qkv; g.ldc = 3 * da;
    g.bias = P(q.b_qkv); g.flags = EPI_BIAS;
    GP_TRY(tgemm(KC_GEMM_FWD, g));
    // o = softmax(q k^T / sqrt(dh) + mask) v                                 (a7)
    GP_TRY(timed(k, KC_ATTN_FWD, 4.0 * Td * S * da * (causal[l] ? (S + 1.0) / (2.0 * S) : 1.0), Td * 4.0 * da * lpb,
                 [&] { return attn_fwd(c, dt, b.qkv, b.o, b.lse, (int)nb, S, A, dh, causal[l]); }));
    // x1 += o W_o      (x1 = x + o W_o + b_o, the residual was staged by LN1)   (a8)
    g = GemmArgs{};
    g.M = (int)T_mb; g.N = d; g.K = da;
    g.A = b.o; g.lda = da; g.B = W(q.w_o); g.ldb = d; g.C = b.x1; g.ldc = d;
    g.flags = EPI_ACCUM | EPI_OUT_F32;
    GP_TRY(tgemm(KC_GEMM_FWD, g));
    float *xa = b.x1;                                // the stream after the attention block(s)
    if (is_dec(l)) {
      // cross-attention (reading B1): cx = LN_x(x1); x1c <- x1 + b_o2; queries from cx, keys / values from the
      // memory, written side by side as [q2 | k2 | v2] so that the self-attention kernels run it unchanged
      GP_TRY(tln(b.x1, P(q.lnx_g), P(q.lnx_b), b.cx, b.meanx, b.rstdx, P(q.b_o2), b.x1c));
      g = GemmArgs{};
      g.M = (int)T_mb; g.N = da; g.K = d;
      g.A = b.cx; g.lda = d; g.B = W(q.w_q); g.ldb = da; g.C = b.qkv2; g.ldc = 3 * da;
      g.bias = P(q.b_q); g.flags = EPI_BIAS;
      GP_TRY(tgemm(KC_GEMM_FWD, g));
      g = GemmArgs{};
      g.M = (int)T_mb; g.N = 2 * da; g.K = d;
      g.A = mem; g.lda = d; g.B = W(q.w_kv); g.ldb = 2 * da; g.C = (char *)b.qkv2 + (size_t)da * lp_size(dt); g.ldc = 3 * da;
      g.bias = P(q.b_kv); g.flags = EPI_BIAS;
      GP_TRY(tgemm(KC_GEMM_FWD, g));
      GP_TRY(timed(k, KC_ATTN_FWD, 4.0 * Td * S * da, Td * 4.0 * da * lpb,
                   [&] { return attn_fwd(c, dt, b.qkv2, b.o2, b.lse2, (int)nb, S, A, dh, 0); }));
      g = GemmArgs{};
      g.M = (int)T_mb; g.N = d; g.K = da;
      g.A = b.o2; g.lda = da; g.B = W(q.w_o2); g.ldb = d; g.C = b.x1c; g.ldc = d;
      g.flags = EPI_ACCUM | EPI_OUT_F32;
      GP_TRY(tgemm(KC_GEMM_FWD, g));
      xa = b.x1c;
    }
    // where x2 = xa + h W_2 + b_2 goes                                        (a11, a12)
    float *x2;
    if (!last) x2 = b.x2;
    else if (k == K - 1) x2 = w.x_out;
    else if (!replay) x2 = boundary_staged ? w.x_out : slot[k + 1][m];   // boundary stash (a12)
    else if (replay_full) x2 = w.x_out;               // replay output nobody reads
    else x2 = nullptr;                                // skipped: B_k does not need F_k's output
    // c = LN2(xa); x2 <- xa + b_2                                            (a9)
    GP_TRY(tln(xa, P(q.ln2_g), P(q.ln2_b), b.c, b.mean2, b.rstd2, x2 ? P(q.b_2) : nullptr, x2));
    // h = relu(c W_1 + b_1)                                                  (a10)
    g = GemmArgs{};
    g.M = (int)T_mb; g.N = H; g.K = d;
    g.A = b.c; g.lda = d; g.B = W(q.w_1); g.ldb = H; g.C = b.h; g.ldc = H;
    g.bias = P(q.b_1); g.flags = EPI_BIAS | EPI_RELU | EPI_BITS_OUT;
    g.mask = b.hbits; g.ldmask = (H + 31) / 32;   // 1 bit per unit for the ReLU backward (a16)
    GP_TRY(tgemm(KC_GEMM_FWD, g));
    // x2 += h W_2                                                            (a11)
    if (x2) {
      g = GemmArgs{};
      g.M = (int)T_mb; g.N = d; g.K = H;
      g.A = b.h; g.lda = H; g.B = W(q.w_2); g.ldb = d; g.C = x2; g.ldc = d;
      g.flags = EPI_ACCUM | EPI_OUT_F32;
      GP_TRY(tgemm(KC_GEMM_FWD, g));
    }
    x = x2;
  }
  // pipeline handle: the boundary activation is the one tensor that leaves the device - one copy of
  // [T_mb, d] fp32 into the next cell's slot, on this cell's stream, ahead of the event F(k+1,m) waits for
  if (boundary_staged && k + 1 < K && !replay && nl > 0)
    GP_TRY(peer_copy(k + 1, slot[k + 1][m], k, w.x_out, (size_t)T_mb * d * sizeof(float), c.stream));
  if (k == K - 1) {
    if (nl == 0 && K == 1) x = w.x_emb;
    // y = LN_f(x_L); logits = y W_out; fused softmax-CE -> loss partial, dlogits   (a13, a14)
    GP_TRY(tln(x, P(i_lnf_g), P(i_lnf_b), w.y, w.meanf, w.rstdf, nullptr, nullptr));
    GemmArgs g{};
    g.M = (int)T_mb; g.N = V; g.K = d;
    g.A = w.y; g.lda = d; g.B = W(i_w_out); g.ldb = V; g.C = w.logits; g.ldc = V;
    g.flags = 0;
    GP_TRY(tgemm(KC_GEMM_FWD, g));
    GP_TRY(timed(k, KC_CE, 0, Td * V * 2.0 * lpb,
                 [&] { return softmax_ce(c, dt, w.logits, lab, w.rowloss, T_mb, V, 1.f / (float)T_total, logit_clip); }));
    // the micro-batch's loss partial comes from the pass that is not repeated: the forward task, or - when that is
    // elided - the replay
    GP_TRY(loss_reduce(c, w.rowloss, (replay && forward_runs(k)) ? loss_dummy : loss_parts + m, T_mb));
  }
  return cudaSuccess;
}

// ---------------------------------------------------------------------------------------------
// B_k: back-propagation through the cell, accumulating parameter gradients in fp32 (a16-a18)
// ---------------------------------------------------------------------------------------------
cudaError_t Engine::backward_cell(int k, int m) {
  Ctx c = ctx(k);
  Workspace &w = wsp(k, m);
  BwdScratch &s = bwd[k];
  const int32_t *tok = tok_dev + (int64_t)m * T_mb;
  int nl = cell_hi[k] - cell_lo[k];
  const float *dx;            // gradient of the residual stream at the current position
  const void *dxo;            // its lp operand copy
  int cur = 0;                // which ping-pong buffer the NEXT producer writes
  const double lpb = (double)lp_size(dt);
  const double Td = (double)T_mb;
  // Side stream (engine.h): a weight-gradient GEMM goes to side[k] behind an event that orders it after everything
  // the main stream has enqueued so far.  Its X operand is an interior activation (next written by the cell's next
  // task, which waits for side_tail[k]); its dY operand is scratch of this task: `pend` holds, per such buffer, the
  // event of the last side-stream GEMM reading it, and `guard` makes the main stream wait for it before a kernel
  // that overwrites the buffer is enqueued.  The side stream is in-order, so one wait covers every earlier GEMM.
  const bool sideon = side_active();
  Ctx cside = c;
  if (sideon) cside.stream = side[k];
  struct Pend { const void *buf; cudaEvent_t ev; int seq; };
  Pend pend[8];
  int npend = 0, side_seq = 0, waited_seq = 0;
  cudaEvent_t tail = nullptr;
  auto guard = [&](const void *buf) -> cudaError_t {
    if (!buf) return cudaSuccess;
    for (int i = 0; i < npend; ++i)
      if (pend[i].buf == buf) {
        const int sq = pend[i].seq;
        GP_TRY(cudaStreamWaitEvent(c.stream, pend[i].ev, 0));
        if (sq > waited_seq) waited_seq = sq;
        int n = 0;
        for (int j = 0; j < npend; ++j)
          if (pend[j].seq > waited_seq) pend[n++] = pend[j];
        npend = n;
        if (side_seq == waited_seq) tail = nullptr;
        break;
      }
    return cudaSuccess;
  };
  auto tlnb = [&](const void *dy_, const float *x_, const float *mu_, const float *rs_, const float *g_,
                  const float *dres_, float *dxo_, void *dxlp_, float *dg_, float *db_, float *cs_) -> cudaError_t {
    GP_TRY(guard(dxo_));
    GP_TRY(guard(dxlp_));
    double by = Td * d * (lpb + 4.0 + (dres_ ? 4.0 : 0.0) + 4.0 + (dxlp_ ? lpb : 0.0));
    return timed(k, KC_LN_BWD, 0, by, [&] {
      return ln_bwd(c, dt, dy_, x_, mu_, rs_, g_, dres_, dxo_, dxlp_, s.ln_partials, dg_, db_, cs_, T_mb, d);
    });
  };
  // the attention backward's fused column sums: partial [nb, 3 da] (row stride 3 da) -> out[n] += sum over the nb sequences
  const bool fused_cs = attn_bwd_fuses_colsum(dt, S, A, dh);
  auto tred = [&](const float *part_, int n_, float *out_) -> cudaError_t {
    return timed(k, KC_COLSUM, 0, (double)nb * n_ * 4.0, [&] { return colsum_reduce_partials(c, part_, (int)nb, n_, 3 * da, out_); });
  };
  auto tcol = [&](const void *dy_, int64_t ld_, float *out_, int n_) -> cudaError_t {
    return timed(k, KC_COLSUM, 0, Td * n_ * lpb, [&] { return colsum_accum(c, dt, dy_, ld_, out_, s.colsum_scratch, T_mb, n_); });
  };
  auto wgrad = [&](const void *X, int64_t ldx, int Min, const void *dY, int64_t ldy, int Nout,
                   int iw, bool may_side = true) -> cudaError_t {
    GemmArgs g{};
    g.M = Min; g.N = Nout; g.K = (int)T_mb;
    g.A = X; g.lda = ldx; g.transA = 1; g.B = dY; g.ldb = ldy; g.transB = 0;
    g.C = G(iw); g.ldc = Nout; g.flags = EPI_ACCUM | EPI_OUT_F32;
    g.ws = s.splitk_ws; g.ws_bytes = splitk_ws_bytes;
    double by = ((double)g.M * g.K + (double)g.K * g.N) * lpb + (double)g.M * g.N * 8.0;
    // a split-K product needs the cell's one split-K workspace, which the main stream's GEMMs use: it stays there
    if (!sideon || !may_side || (dt == GP_BF16 && gemm_splitk_ws_bytes(g.M, g.N, g.K, sm_count) != 0))
      return timed(k, KC_GEMM_WGRAD, 2.0 * g.M * g.N * (double)g.K, by, [&] { return gemm(c, dt, g); });
    cudaEvent_t fork = pool_event(), done = pool_event();
    if (!fork || !done) return pool_err;
    GP_TRY(cudaEventRecord(fork, c.stream));
    GP_TRY(cudaStreamWaitEvent(cside.stream, fork, 0));
    g.ws = nullptr; g.ws_bytes = 0;
    GP_TRY(timed_on(cside.stream, KC_GEMM_WGRAD, 2.0 * g.M * g.N * (double)g.K, by, [&] { return gemm(cside, dt, g); }));
    GP_TRY(cudaEventRecord(done, cside.stream));
    tail = done;
    ++side_seq;
    int slot_i = npend;
    for (int i = 0; i < npend; ++i)
      if (pend[i].buf == dY) slot_i = i;
    if (slot_i == npend) {
      if (npend == 8) return cudaErrorUnknown;             // cannot happen: at most six distinct dY buffers per task
      ++npend;
    }
    pend[slot_i] = Pend{dY, done, side_seq};
    return cudaSuccess;
  };
  auto dgrad = [&](const void *dY, int64_t ldy, int Kout, int iw, int Nin, void *dX,
                   uint32_t *mask, float *colsum_to = nullptr) -> cudaError_t {
    GemmArgs g{};
    g.M = (int)T_mb; g.N = Nin; g.K = Kout;
    g.A = dY; g.lda = ldy; g.transA = 0; g.B = W(iw); g.ldb = Kout; g.transB = 1;
    g.C = dX; g.ldc = Nin; g.mask = mask; g.ldmask = (Nin + 31) / 32; g.flags = mask ? EPI_MASK : 0;
    if (colsum_to) { g.flags |= EPI_COLSUM; g.colsum_out = colsum_to; g.colsum_scratch = s.colsum_scratch; }
    g.ws = s.splitk_ws; g.ws_bytes = splitk_ws_bytes;
    GP_TRY(guard(dX));
    double by = ((double)g.M * g.K + (double)g.K * g.N + (double)g.M * g.N) * lpb + (mask ? (double)g.M * g.N / 8.0 : 0.0);
    return timed(k, KC_GEMM_DGRAD, 2.0 * g.M * g.N * (double)g.K, by, [&] { return gemm(c, dt, g); });
  };

  if (k == K - 1) {
    const float *xL = nl > 0 ? w.x_out : (K == 1 ? w.x_emb : slot[k][m]);
    GP_TRY(wgrad(w.y, d, d, w.logits, V, V, i_w_out));                 // dW_out += y^T dlogits
    GP_TRY(dgrad(w.logits, V, V, i_w_out, d, s.dc, nullptr));          // dy = dlogits W_out^T
    // the gradient of x_L is also the output gradient of the last layer's FFN2: db_2 += sum_t dx
    GP_TRY(tlnb(s.dc, xL, w.meanf, w.rstdf, P(i_lnf_g), nullptr, s.dx[cur],
                dt == GP_BF16 ? s.dx_lp[cur] : nullptr, G(i_lnf_g), G(i_lnf_b),
                nl > 0 ? G(lp[cell_hi[k] - 1].b_2) : nullptr));
    dx = s.dx[cur];
    dxo = s.dx_lp[cur];
    cur ^= 1;
  } else {
    dx = dout[m & 1][k];
    dxo = dout_lp[m & 1][k];
    // pipeline handle: the FFN2 bias gradient of this cell's last layer is the column sum of the incoming boundary
    // gradient; with all cells in one arena the next cell's LayerNorm backward adds it (fused), across devices
    // this cell does it itself
    if (multi() && nl > 0) GP_TRY(tcol(dxo, d, G(lp[cell_hi[k] - 1].b_2), d));
  }
  const void *dxo_in = dxo;   // (a boundary-ring entry when k < K-1: the next cell overwrites it after this task's event)
  // encoder-decoder: gradient of the second member of the pair.  In the decoder it is the gradient of the memory:
  // every decoder layer's cross-attention adds dkv W_kv^T to it (fp32) - the first one of the cell on top of what the
  // next cell handed down (nothing, in the last cell), the others in place.  In the encoder it is the gradient of the
  // target embedding and only travels down to cell 0.
  const float *daux_in = (encdec() && k + 1 < K) ? dout_aux[m & 1][k] : nullptr;
  float *daux = nullptr;
  bool daux_started = false;
  if (encdec() && k >= kt) daux = k == kt ? s.daux : dbound_aux[m & 1][k];
  const void *mem = nullptr;
  // the transition cell's own memory: interior when it was replayed (or no later cell reads it), else what F(kt, m)
  // wrote for the later cells (stored-activation mode, and the elided replay of the last micro-batch)
  const bool replayed = replay_runs(k, m);
  if (encdec() && k >= kt)
    mem = k > kt ? (const void *)aux_in[k][m] : (const void *)((replayed || kt == K - 1 || multi()) ? w.mem : aux_in[kt + 1][m]);
  for (int i = nl - 1; i >= 0; --i) {
    int l = cell_lo[k] + i;
    const LayerParams &q = lp[l];
    LayerBuf &b = w.layers[i];
    const bool dec = is_dec(l), trans = encdec() && l == n_enc;
    // input of the layer: the previous layer's output, the cell's input - or, for the first decoder layer, the
    // target embedding
    const float *x_in = i > 0 ? w.layers[i - 1].x2 : (k == 0 ? w.x_emb : slot[k][m]);
    if (trans) x_in = kt == 0 ? w.aux_emb : (const float *)aux_in[kt][m];
    // FFN: dh = (dx W_2^T) * [h > 0] with db_1 += sum_t dh fused into the epilogue; dW_2 += h^T dx
    // (db_2 += sum_t dx was fused into the LayerNorm-backward kernel that produced dx)
    GP_TRY(dgrad(dxo, d, d, q.w_2, H, s.dh, b.hbits, G(q.b_1)));
    GP_TRY(wgrad(b.h, H, H, dxo, d, d, q.w_2));
    // dc = dh W_1^T; dW_1 += c^T dh
    GP_TRY(dgrad(s.dh, H, H, q.w_1, d, s.dc, nullptr));
    GP_TRY(wgrad(b.c, d, d, s.dh, H, H, q.w_1));
    // LN2 backward; residual adds gradients: dxa = dx + LN2'(dc)
    // (the bias gradient of the GEMM that produced xa is fused here: db_o, or db_o2 in a decoder layer)
    GP_TRY(tlnb(s.dc, dec ? b.x1c : b.x1, b.mean2, b.rstd2, P(q.ln2_g), dx, s.dx[cur],
                dt == GP_BF16 ? s.dx_lp[cur] : nullptr, G(q.ln2_g), G(q.ln2_b), G(dec ? q.b_o2 : q.b_o)));
    dx = s.dx[cur];
    dxo = s.dx_lp[cur];
    cur ^= 1;
    if (dec) {
      // cross-attention block: do2 = dx1c W_o2^T; dW_o2 += o2^T dx1c; attention backward over [q2 | k2 | v2]
      const size_t kv_off = (size_t)da * lp_size(dt);
      GP_TRY(dgrad(dxo, d, d, q.w_o2, da, s.d_o, nullptr));
      GP_TRY(wgrad(b.o2, da, da, dxo, d, d, q.w_o2, false));      // the cross-attention block's three stay on the main stream
      GP_TRY(guard(s.dqkv));
      GP_TRY(timed(k, KC_ATTN_BWD, 10.0 * Td * S * da, Td * 8.0 * da * lpb,
                   [&] { return attn_bwd(c, dt, b.qkv2, b.o2, s.d_o, b.lse2, s.dqkv, s.dvec, (int)nb, S, A, dh, 0,
                                         fused_cs ? s.colsum_scratch : nullptr); }));
      if (fused_cs) {                                      // db_q, db_kv from the kernel's per-sequence column sums
        GP_TRY(tred(s.colsum_scratch, da, G(q.b_q)));
        GP_TRY(tred(s.colsum_scratch + da, 2 * da, G(q.b_kv)));
      }
      // queries: dcx = dq2 W_q^T; dW_q += cx^T dq2; db_q += sum_t dq2
      GP_TRY(dgrad(s.dqkv, 3 * da, da, q.w_q, d, s.dc, nullptr));
      GP_TRY(wgrad(b.cx, d, d, s.dqkv, 3 * da, da, q.w_q, false));
      if (!fused_cs) GP_TRY(tcol(s.dqkv, 3 * da, G(q.b_q), da));
      // keys / values: dmem += dkv W_kv^T (fp32); dW_kv += mem^T dkv; db_kv += sum_t dkv
      {
        GemmArgs g{};
        g.M = (int)T_mb; g.N = d; g.K = 2 * da;
        g.A = (const char *)s.dqkv + kv_off; g.lda = 3 * da; g.transA = 0; g.B = W(q.w_kv); g.ldb = 2 * da; g.transB = 1;
        g.C = daux; g.ldc = d; g.flags = EPI_OUT_F32;
        if (daux_started) g.flags |= EPI_ACCUM;
        else if (daux_in) { g.flags |= EPI_RESID; g.resid = daux_in; }
        g.ws = s.splitk_ws; g.ws_bytes = splitk_ws_bytes;
        double by = ((double)g.M * g.K + (double)g.K * g.N) * lpb + (double)g.M * g.N * ((daux_started || daux_in) ? 8.0 : 4.0);
        GP_TRY(timed(k, KC_GEMM_DGRAD, 2.0 * g.M * g.N * (double)g.K, by, [&] { return gemm(c, dt, g); }));
        daux_started = true;
      }
      GP_TRY(wgrad(mem, d, d, (const char *)s.dqkv + kv_off, 3 * da, 2 * da, q.w_kv, false));
      if (!fused_cs) GP_TRY(tcol((const char *)s.dqkv + kv_off, 3 * da, G(q.b_kv), 2 * da));
      // LN_x backward: dx1 = dx1c + LN_x'(dcx); db_o += sum_t dx1
      GP_TRY(tlnb(s.dc, b.x1, b.meanx, b.rstdx, P(q.lnx_g), dx, s.dx[cur],
                  dt == GP_BF16 ? s.dx_lp[cur] : nullptr, G(q.lnx_g), G(q.lnx_b), G(q.b_o)));
      dx = s.dx[cur];
      dxo = s.dx_lp[cur];
      cur ^= 1;
    }
    // attention block: do = dx1 W_o^T; dW_o += o^T dx1
    GP_TRY(dgrad(dxo, d, d, q.w_o, da, s.d_o, nullptr));
    GP_TRY(wgrad(b.o, da, da, dxo, d, d, q.w_o));
    // db_qkv += sum_t dqkv: the tcgen05 attention backward leaves per-sequence column sums of what it stores (one small
    // reduction over the nb sequences follows); the other backends take the separate pass over dqkv
    GP_TRY(guard(s.dqkv));
    GP_TRY(timed(k, KC_ATTN_BWD, 10.0 * Td * S * da * (causal[l] ? (S + 1.0) / (2.0 * S) : 1.0), Td * 8.0 * da * lpb,
                 [&] { return attn_bwd(c, dt, b.qkv, b.o, s.d_o, b.lse, s.dqkv, s.dvec, (int)nb, S, A, dh, causal[l],
                                       fused_cs ? s.colsum_scratch : nullptr); }));
    if (fused_cs) GP_TRY(tred(s.colsum_scratch, 3 * da, G(q.b_qkv)));
    // da = dqkv W_qkv^T; dW_qkv += a^T dqkv
    GP_TRY(dgrad(s.dqkv, 3 * da, 3 * da, q.w_qkv, d, s.dc, nullptr));
    GP_TRY(wgrad(b.a, d, d, s.dqkv, 3 * da, 3 * da, q.w_qkv));
    if (!fused_cs) GP_TRY(tcol(s.dqkv, 3 * da, G(q.b_qkv), 3 * da));
    // LN1 backward: dx_in = dx1 + LN1'(da); the cell's first layer writes the boundary gradient
    float *out = s.dx[cur];
    void *out_lp = s.dx_lp[cur];
    if (i == 0 && k > 0) {
      out = dbound[m & 1][k];
      out_lp = dbound_lp[m & 1][k];
    }
    if (trans) {
      // the input of the first decoder layer is the target embedding: its gradient is the aux gradient this cell
      // hands down (cell 0: kept for the embedding backward), and nobody's FFN2 output
      float *dt_out = kt == 0 ? s.dtgt : dbound_aux[m & 1][kt];
      GP_TRY(tlnb(s.dc, x_in, b.mean1, b.rstd1, P(q.ln1_g), dx, dt_out, nullptr, G(q.ln1_g), G(q.ln1_b), nullptr));
      // back through memory = LN_e(x_src): dx_src = LN_e'(dmem) - the encoder's last FFN2 output gradient
      const float *x_src = i > 0 ? w.layers[i - 1].x2 : slot[k][m];
      GP_TRY(cast_to_lp(c, dt, daux, s.dc, T_mb * (int64_t)d));
      GP_TRY(tlnb(s.dc, x_src, w.mean_e, w.rstd_e, P(i_lne_g), nullptr, out, dt == GP_BF16 ? out_lp : nullptr,
                  G(i_lne_g), G(i_lne_b), (multi() && i == 0) ? nullptr : G(lp[l - 1].b_2)));
    } else {
      // its output is the FFN2 output gradient of the layer below (possibly in the previous cell):
      // db_2(l-1) += sum_t dx
      GP_TRY(tlnb(s.dc, x_in, b.mean1, b.rstd1, P(q.ln1_g), dx, out, dt == GP_BF16 ? out_lp : nullptr,
                  G(q.ln1_g), G(q.ln1_b), l > 0 && !(multi() && i == 0) ? G(lp[l - 1].b_2) : nullptr));
    }
    dx = out;
    dxo = out_lp;
    cur ^= 1;
  }
  if (k == 0)                                                          // dE[tok] += dx0
    GP_TRY(timed(k, KC_EMBED, 0, Td * d * 12.0, [&] { return embed_bwd(c, tok, dx, G(i_emb), T_mb, d); }));
  if (encdec() && k < kt) {
    // an encoder cell passes the gradient of the target embedding on (cell 0: into the shared table, after the
    // source tokens' rows: a fixed order, so the step stays bitwise reproducible)
    if (k > 0) GP_TRY(cudaMemcpyAsync(dbound_aux[m & 1][k], daux_in, (size_t)T_mb * d * sizeof(float), cudaMemcpyDeviceToDevice, c.stream));
    else GP_TRY(timed(k, KC_EMBED, 0, Td * d * 12.0, [&] { return embed_bwd(c, tgt_dev + (int64_t)m * T_mb, daux_in, G(i_emb), T_mb, d); }));
  } else if (encdec() && k == 0) {                                     // cell 0 holds the transition
    GP_TRY(timed(k, KC_EMBED, 0, Td * d * 12.0, [&] { return embed_bwd(c, tgt_dev + (int64_t)m * T_mb, s.dtgt, G(i_emb), T_mb, d); }));
  }
  if (sideon) {
    GP_TRY(guard(dxo_in));
    side_tail[k] = tail;
  }
  if (multi() && k > 0) {
    // backward boundary transfer: the gradient wrt this cell's input becomes the previous cell's output gradient
    GP_TRY(peer_copy(k - 1, dout[m & 1][k - 1], k, dbound[m & 1][k], (size_t)T_mb * d * sizeof(float), c.stream));
    if (dt == GP_BF16)
      GP_TRY(peer_copy(k - 1, dout_lp[m & 1][k - 1], k, dbound_lp[m & 1][k], (size_t)T_mb * d * 2, c.stream));
    if (encdec())
      GP_TRY(peer_copy(k - 1, dout_aux[m & 1][k - 1], k, dbound_aux[m & 1][k], (size_t)T_mb * d * sizeof(float), c.stream));
  }
  return cudaSuccess;
}

cudaError_t Engine::peer_copy(int k_dst, void *dst, int k_src, const void *src, size_t bytes, cudaStream_t s) {
  if (multi_device && cell_device[k_dst] != cell_device[k_src])
    return cudaMemcpyPeerAsync(dst, cell_device[k_dst], src, cell_device[k_src], bytes, s);
  return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, s);
}

// ---------------------------------------------------------------------------------------------
// One mini-batch on the GPipe schedule.  Tasks are enqueued in global tick order (a topological
// order of the dependency graph), cell k on stream k:
//   forward ticks   F(k,m), m = tau - k                      F(k,m) <- F(k-1,m)
//   backward ticks  [R(k,m)] B(k,m), m = M-1 - (tau-(K-1-k))  B(k,m) <- B(k+1,m);  R(k,m) <- slot only
// ---------------------------------------------------------------------------------------------
cudaError_t Engine::resolve_kernel_timing() {
  for (const KRec &r : krecs) {
    float ms = 0.f;
    GP_TRY(cudaEventElapsedTime(&ms, r.e0, r.e1));
    KStat &st = kstats[r.cls];
    st.count += 1; st.ms += ms; st.flops += r.flops; st.bytes += r.bytes;
  }
  krecs.clear();
  return cudaSuccess;
}

cudaError_t Engine::enqueue_step() {
  int idx = 0;
  auto task = [&](int kind, int k, int m) -> cudaError_t {
    TraceRec r{kind, k, m, idx++, nullptr, nullptr};
    if (trace_on) {
      r.e0 = pool_event();
      r.e1 = pool_event();
      if (!r.e0 || !r.e1) return pool_err;
      GP_TRY(cudaEventRecord(r.e0, st(k)));
    }
    GP_TRY(use(k));
    if (!side_tail.empty() && side_tail[k]) {              // the cell's weight-gradient GEMMs still read its interior
      GP_TRY(cudaStreamWaitEvent(st(k), side_tail[k], 0));
      side_tail[k] = nullptr;
    }
    cudaError_t e = kind == 'B' ? backward_cell(k, m) : forward_cell(k, m, kind == 'R');
    if (e != cudaSuccess) return e;
    if (trace_on) {
      GP_TRY(cudaEventRecord(r.e1, st(k)));
      trace.push_back(r);
    }
    return cudaSuccess;
  };
  // inputs are on stream 0; every other cell waits for them
  GP_TRY(cudaEventRecord(ev_in, streams[0]));
  for (int k = 1; k < K; ++k) GP_TRY(cudaStreamWaitEvent(st(k), ev_in, 0));
  if (trace_on) GP_TRY(cudaEventRecord(ev_t0, streams[0]));

  for (int tau = 0; tau < M + K - 1; ++tau)
    for (int k = 0; k < K; ++k) {
      int m = tau - k;
      if (m < 0 || m >= M) continue;
      // F(K-1, m) is elided under re-materialization (reading A15c): the last cell's forward has no consumer but the
      // loss, and R(K-1, m) produces everything again, the loss included - R(K-1, m) is then the micro-batch's one
      // pass through the last cell
      if (!forward_runs(k)) continue;
      if (k > 0) GP_TRY(cudaStreamWaitEvent(st(k), ev_f[k - 1][m], 0));
      GP_TRY(task('F', k, m));
      if (k + 1 < K) GP_TRY(cudaEventRecord(ev_f[k][m], st(k)));
    }
  for (int tau = 0; tau < M + K - 1; ++tau)
    for (int k = K - 1; k >= 0; --k) {
      int m = M - 1 - (tau - (K - 1 - k));
      if (m < 0 || m >= M) continue;
      // early: no wait on B(k+1,m).  R(k, M-1) is elided (reading A15b): nothing of cell k runs between its last
      // forward task F(k, M-1) and its first backward task B(k, M-1), so the cell's one workspace still holds, bit
      // for bit, the interior that replay would recompute - re-materialization is there to bound memory, and that
      // interior is resident anyway.  (GPIPE_REPLAY_FULL in a probes build runs every task of Fig. 2c.)
      if (replay_runs(k, m)) {
        if (!forward_runs(k) && k > 0) GP_TRY(cudaStreamWaitEvent(st(k), ev_f[k - 1][m], 0));   // the cell's input slot
        GP_TRY(task('R', k, m));
      }
      if (k + 1 < K) GP_TRY(cudaStreamWaitEvent(st(k), ev_b[k + 1][m], 0));
      // the boundary-gradient ring has two entries: B(k,m) reuses the one B(k-1,m+2) read
      if (k > 0 && m + 2 < M) GP_TRY(cudaStreamWaitEvent(st(k), ev_b[k - 1][m + 2], 0));
      GP_TRY(task('B', k, m));
      GP_TRY(cudaEventRecord(ev_b[k][m], st(k)));
    }
  // join: the loss partials come back on the last cell's stream, and stream 0 waits for every cell
  for (int k = 0; k < K && !side_tail.empty(); ++k)
    if (side_tail[k]) {
      GP_TRY(cudaStreamWaitEvent(st(k), side_tail[k], 0));
      side_tail[k] = nullptr;
    }
  GP_TRY(use(K - 1));
  GP_TRY(cudaMemcpyAsync(host_loss, loss_parts, sizeof(float) * M, cudaMemcpyDeviceToHost, st(K - 1)));
  for (int k = 1; k < K; ++k) {
    GP_TRY(cudaEventRecord(ev_done[k], st(k)));
    GP_TRY(cudaStreamWaitEvent(streams[0], ev_done[k], 0));
  }
  GP_TRY(use(0));
  return cudaSuccess;
}

void Engine::drop_graph() {
  if (graph_exec) cudaGraphExecDestroy(graph_exec);
  if (graph) cudaGraphDestroy(graph);
  graph_exec = nullptr;
  graph = nullptr;
}

cudaError_t Engine::run_step(float *loss_out) {
  ev_pool_used = 0;
  trace.clear();
  krecs.clear();
  const bool eager = !use_graph || trace_on || ktiming_on || serial || graph_state < 0 || multi_device;
  if (eager || graph_state == 0) {
    GP_TRY(enqueue_step());
    if (!eager) graph_state = 1;
  } else {
    if (graph_state == 1) {
      // Relaxed mode: other host threads (the caller's allocator, another handle) may call CUDA while this thread
      // captures; nothing enqueue_step does is capture-unsafe (kernel launches, event record / wait, one async copy).
      const int64_t l0 = launches;
      cudaError_t e = cudaStreamBeginCapture(streams[0], cudaStreamCaptureModeRelaxed);
      if (e == cudaSuccess) {
        e = enqueue_step();
        cudaGraph_t gcap = nullptr;
        cudaError_t e2 = cudaStreamEndCapture(streams[0], &gcap);     // always end the capture, even after an error
        if (e == cudaSuccess) e = e2;
        graph = gcap;
      }
      if (e == cudaSuccess) e = cudaGraphInstantiate(&graph_exec, graph, 0);
      graph_launches = launches - l0;
      launches = l0;
      if (e != cudaSuccess) {                                         // not fatal: this handle stays on eager enqueue
        cudaGetLastError();
        drop_graph();
        graph_state = -1;
        GP_TRY(enqueue_step());
      } else {
        graph_state = 2;
      }
    }
    if (graph_state == 2) {
      GP_TRY(cudaGraphLaunch(graph_exec, streams[0]));
      launches += graph_launches;
    }
  }
  GP_TRY(cudaStreamSynchronize(streams[0]));
  if (ktiming_on) GP_TRY(resolve_kernel_timing());
  double s = 0.0;
  for (int m = 0; m < M; ++m) s += (double)host_loss[m];
  *loss_out = (float)s;
  return cudaSuccess;
}

}  // namespace gp

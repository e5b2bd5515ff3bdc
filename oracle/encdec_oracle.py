"""CPU ORACLE for the encoder-decoder Transformer T(L,H,A) on the GPipe schedule.
TEST INFRASTRUCTURE, NOT PRODUCT: only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` legs may import this.  It shares no code with the CUDA path and neither imports the other.

What the paper fixes (footnote 1): "T(L,H,A) is a Transformer model with L encoder layers and
L decoder layers, a feed-forward hidden dimension of H and A attention heads.  The model dimension is fixed
to 1024"; T(64,16384,32) has 6B parameters; "Trainability Challenges": (i) "we
scale down the initialization of all transformer feed-forward layers by the number of layers", (ii) "we clip
the logit predictions (softmax pre-activations) whenever their magnitude exceeds a certain value".  The
GPipe part is unchanged: the model is a SEQUENCE of layers

    enc_0 .. enc_{Le-1}, dec_0 .. dec_{Ld-1}

cut into K cells of consecutive layers, M micro-batches, boundary-only storage with replay.  What crosses a
cell boundary is a PAIR of activations (x, aux): inside the encoder x is the source stream and aux the
(not yet used) target embedding; inside the decoder x is the target stream and aux the encoder memory that
every decoder layer's cross-attention reads.  Readings (B1-B6):

  B1  layers: encoder layer = pre-LN self-attention (no mask) + ReLU FFN, exactly the layer of
      oracle/gpipe_oracle.py; decoder layer = pre-LN causal self-attention, pre-LN cross-attention
      (queries from the target stream, keys / values from the memory; no mask), ReLU FFN.
  B2  memory = LN_e(x_src after the last encoder layer) (the usual pre-LN encoder output norm).
  B3  ONE embedding table for source and target ids (the paper's 64k vocabulary is shared by its 103
      languages) and an untied output matrix: 2*V*d, which is what reproduces the printed
      model sizes (pin P2: 0.41 / 1.24 / 1.24 / 3.08 / 6.04 B).  Cell 0 embeds both id sequences.
  B4  source and target length are both S (BASELINE.json fixes S = 256 for every config); the same
      sinusoidal table is added to both embeddings.
  B5  logit clipping: z <- min(max(z, -c), c) before the softmax; derivative 1 where |z| <= c, 0 elsewhere
      (what a clamp is; the paper gives no formula and does not print c).  c = 0 turns it off.
  B6  depth-scaled initialisation is a property of the parameter draw, not of the step: std of w_1 and w_2
      divided by the number of layers Le + Ld (gpipe_inputs.make_params(ffn_depth_scale=True) on the host).

Precision and `round_operands` as in oracle/gpipe_oracle.py.  Pins: tests/test_oracle_encdec_pins.py
(section-5 model sizes from this module's own tensor list; an independent torch-autograd model built on torch.nn.functional
library calls (layer_norm, linear, scaled_dot_product_attention, cross_entropy, clamp); fp64 finite differences; M / K /
partition invariance; remat == stored bitwise; decoder causality and encoder visibility; clamp against
torch.clamp + autograd; K=1,M=1 reduces to plain back-propagation).
"""
from __future__ import annotations

from typing import Dict, List, Optional, Tuple

import numpy as np

from .gpipe_oracle import (attention_bwd, attention_fwd, bf16_rne, cell_layers, layernorm_bwd,
                           layernorm_fwd, positional_table)


class EncDecSpec:
    """T(L,H,A) of PAPER.md:160: n_enc encoder + n_dec decoder layers, d_model, FFN width, heads."""

    def __init__(self, n_enc, n_dec, d_model, d_ffn, n_heads, d_head, vocab, seq_len,
                 ln_eps: float = 1e-5, logit_clip: float = 0.0):
        self.n_enc, self.n_dec = int(n_enc), int(n_dec)
        if self.n_enc < 1 or self.n_dec < 1:
            raise ValueError("an encoder-decoder model needs at least one layer of each kind")
        self.n_layers = self.n_enc + self.n_dec
        self.d_model, self.d_ffn, self.n_heads = int(d_model), int(d_ffn), int(n_heads)
        self.d_head = int(d_head) if d_head else self.d_model // self.n_heads
        self.vocab, self.seq_len = int(vocab), int(seq_len)
        self.ln_eps = float(ln_eps) if ln_eps else 1e-5
        self.logit_clip = float(logit_clip)

    @property
    def d_attn(self):
        return self.n_heads * self.d_head

    def is_dec(self, l: int) -> bool:
        return l >= self.n_enc


def tensor_list(s: EncDecSpec) -> List[Tuple[str, Tuple[int, int]]]:
    """Canonical inventory, in the order of the layer sequence: emb | encoder layers | lne | decoder
    layers | lnf, w_out.  Layer l is 'l<l>.' for l = 0 .. Le+Ld-1; a decoder layer has the encoder layer's
    twelve tensors plus the cross-attention block (lnx, w_q, b_q, w_kv, b_kv, w_o2, b_o2)."""
    d, H, da, V = s.d_model, s.d_ffn, s.d_attn, s.vocab
    out = [("emb", (V, d))]
    for l in range(s.n_layers):
        p = "l%d." % l
        if l == s.n_enc:
            out += [("lne_g", (1, d)), ("lne_b", (1, d))]
        out += [(p + "ln1_g", (1, d)), (p + "ln1_b", (1, d)),
                (p + "w_qkv", (d, 3 * da)), (p + "b_qkv", (1, 3 * da)),
                (p + "w_o", (da, d)), (p + "b_o", (1, d))]
        if s.is_dec(l):
            out += [(p + "lnx_g", (1, d)), (p + "lnx_b", (1, d)),
                    (p + "w_q", (d, da)), (p + "b_q", (1, da)),
                    (p + "w_kv", (d, 2 * da)), (p + "b_kv", (1, 2 * da)),
                    (p + "w_o2", (da, d)), (p + "b_o2", (1, d))]
        out += [(p + "ln2_g", (1, d)), (p + "ln2_b", (1, d)),
                (p + "w_1", (d, H)), (p + "b_1", (1, H)),
                (p + "w_2", (H, d)), (p + "b_2", (1, d))]
    out += [("lnf_g", (1, d)), ("lnf_b", (1, d)), ("w_out", (d, V))]
    return out


def param_count(s: EncDecSpec) -> int:
    return sum(r * c for _, (r, c) in tensor_list(s))


def softmax_ce_clipped(logits, labels, T_total, clip):
    """Reading B5 + the loss of oracle/gpipe_oracle.softmax_ce: z = clamp(logits, -c, c) (c = 0: z = logits);
    loss = sum_t [logsumexp(z_t) - z_t,label_t] / T_total; dlogits = (softmax(z) - onehot)/T_total where
    |logits| <= c and 0 where the clamp is active.  Also returns the per-token losses."""
    z = np.clip(logits, -clip, clip) if clip > 0 else logits
    mx = z.max(axis=1, keepdims=True)
    e = np.exp(z - mx)
    se = e.sum(axis=1, keepdims=True)
    rows = np.arange(z.shape[0])
    per_tok = np.log(se[:, 0]) + mx[:, 0] - z[rows, labels]
    dl = e / se
    dl[rows, labels] -= 1.0
    dl = dl / logits.dtype.type(T_total)
    if clip > 0:
        dl = dl * (np.abs(logits) <= clip)
    return per_tok.sum() / T_total, dl, per_tok


class GPipeEncDecOracle:
    """gpipe_create / gpipe_step / gpipe_apply_sgd for the encoder-decoder model, on the host."""

    def __init__(self, spec: EncDecSpec, K: int, M: int, remat: bool, dtype=np.float64,
                 round_operands: bool = False, cell_lo=None):
        if K < 1 or K > spec.n_layers or M < 1:
            raise ValueError("need 1 <= K <= Le + Ld and M >= 1")
        self.s, self.K, self.M, self.remat = spec, int(K), int(M), bool(remat)
        if cell_lo is None:
            self.cells = [cell_layers(spec.n_layers, self.K, k) for k in range(self.K)]
        else:
            if (len(cell_lo) != self.K + 1 or cell_lo[0] != 0 or cell_lo[-1] != spec.n_layers
                    or any(cell_lo[k] >= cell_lo[k + 1] for k in range(self.K))):
                raise ValueError("cell_lo must be K+1 strictly increasing boundaries from 0 to Le+Ld")
            self.cells = [range(cell_lo[k], cell_lo[k + 1]) for k in range(self.K)]
        self.dt = np.dtype(dtype).type
        self.rounding = bool(round_operands)
        self.rnd = bf16_rne if round_operands else (lambda a: a)
        self.names = [n for n, _ in tensor_list(spec)]
        self.shapes = dict(tensor_list(spec))
        self.p: Dict[str, np.ndarray] = {n: np.zeros(sh, self.dt) for n, sh in self.shapes.items()}
        self.g: Dict[str, np.ndarray] = {n: np.zeros(sh, self.dt) for n, sh in self.shapes.items()}
        self.pe = positional_table(spec.seq_len, spec.d_model, self.dt)
        self.trace: List[Tuple[str, int, int]] = []
        self.per_token_loss: Dict[int, np.ndarray] = {}      # micro-batch -> [nb*S] (for the visibility pin)

    def set_params(self, params):
        for n in self.names:
            self.p[n] = np.array(params[n], dtype=self.dt).reshape(self.shapes[n])

    def zero_grads(self):
        for n in self.names:
            self.g[n][...] = 0

    def apply_sgd(self, lr: float):
        lr = self.dt(lr)
        for n in self.names:
            self.p[n] = self.p[n] - lr * self.g[n]
        self.zero_grads()

    # -- attention over a micro-batch: one call per sequence --------------------------------------
    def _attend(self, qm, km, vm, nb, S, causal):
        o = np.zeros_like(qm)
        ps_all = []
        ar = self.rnd if self.rounding else None
        for b in range(nb):
            rows = slice(b * S, (b + 1) * S)
            ob, ps = attention_fwd(qm[rows], km[rows], vm[rows], self.s.n_heads, self.s.d_head, causal, rnd=ar)
            o[rows] = ob
            ps_all.append(ps)
        return self.rnd(o), ps_all

    def _attend_bwd(self, do, qm, km, vm, ps_all, nb, S):
        dq, dk, dv = np.zeros_like(qm), np.zeros_like(km), np.zeros_like(vm)
        ar = self.rnd if self.rounding else None
        for b in range(nb):
            rows = slice(b * S, (b + 1) * S)
            dq[rows], dk[rows], dv[rows] = attention_bwd(do[rows], qm[rows], km[rows], vm[rows], ps_all[b],
                                                         self.s.n_heads, self.s.d_head, rnd=ar)
        return dq, dk, dv

    # -- F_k ------------------------------------------------------------------------------------------
    def forward_cell(self, k, bnd_in, src_mb, tgt_mb, labels_mb, T_total, keep):
        """F_k over the pair (x, aux).  Cell 0 embeds the source and the target ids (B3); the cell that
        holds dec_0 turns the source stream into the memory (B2) and switches x to the target stream;
        cell K-1 ends with the final LN, the output projection, the clamp and the loss.
        Returns ((x, aux), interior, loss)."""
        s, p, r = self.s, self.p, self.rnd
        nb, S = tgt_mb.shape
        da = s.d_attn
        interior = {"layers": []} if keep else None
        if k == 0:
            pe = np.tile(self.pe, (nb, 1))
            x = p["emb"][src_mb.reshape(-1)] + pe
            aux = p["emb"][tgt_mb.reshape(-1)] + pe
        else:
            x, aux = bnd_in
        for l in self.cells[k]:
            q_ = "l%d." % l
            lay = dict(l=l)
            if l == s.n_enc:                                    # encoder -> decoder transition
                mem, xhat_e, rstd_e = layernorm_fwd(x, p["lne_g"], p["lne_b"], s.ln_eps)
                mem = r(mem)
                lay.update(xhat_e=xhat_e, rstd_e=rstd_e)
                x, aux = aux, mem                               # x: target stream, aux: the memory
            # self-attention block (decoder: causal)
            a, xhat1, rstd1 = layernorm_fwd(x, p[q_ + "ln1_g"], p[q_ + "ln1_b"], s.ln_eps)
            a = r(a)
            qkv = r(a @ p[q_ + "w_qkv"] + p[q_ + "b_qkv"])
            qm, km, vm = qkv[:, :da], qkv[:, da:2 * da], qkv[:, 2 * da:]
            o, ps = self._attend(qm, km, vm, nb, S, s.is_dec(l))
            x1 = x + o @ p[q_ + "w_o"] + p[q_ + "b_o"]
            lay.update(xhat1=xhat1, rstd1=rstd1, a=a, q=qm, k=km, v=vm, p=ps, o=o)
            if s.is_dec(l):
                # cross-attention block: queries from the target stream, keys / values from the memory
                cx, xhatx, rstdx = layernorm_fwd(x1, p[q_ + "lnx_g"], p[q_ + "lnx_b"], s.ln_eps)
                cx = r(cx)
                q2 = r(cx @ p[q_ + "w_q"] + p[q_ + "b_q"])
                kv = r(aux @ p[q_ + "w_kv"] + p[q_ + "b_kv"])
                k2, v2 = kv[:, :da], kv[:, da:]
                o2, ps2 = self._attend(q2, k2, v2, nb, S, False)
                x1 = x1 + o2 @ p[q_ + "w_o2"] + p[q_ + "b_o2"]
                lay.update(xhatx=xhatx, rstdx=rstdx, cx=cx, q2=q2, k2=k2, v2=v2, p2=ps2, o2=o2, mem=aux)
            # FFN block
            c, xhat2, rstd2 = layernorm_fwd(x1, p[q_ + "ln2_g"], p[q_ + "ln2_b"], s.ln_eps)
            c = r(c)
            h = r(np.maximum(c @ p[q_ + "w_1"] + p[q_ + "b_1"], 0))
            x = x1 + h @ p[q_ + "w_2"] + p[q_ + "b_2"]
            lay.update(xhat2=xhat2, rstd2=rstd2, c=c, h=h)
            if keep:
                interior["layers"].append(lay)
        loss = None
        if k == self.K - 1:
            y, xhat_f, rstd_f = layernorm_fwd(x, p["lnf_g"], p["lnf_b"], s.ln_eps)
            y = r(y)
            logits = r(y @ p["w_out"])
            loss, dlogits, per_tok = softmax_ce_clipped(logits, labels_mb.reshape(-1), T_total, s.logit_clip)
            if keep:
                interior.update(xhat_f=xhat_f, rstd_f=rstd_f, y=y, dlogits=r(dlogits), per_tok=per_tok)
        return (x, aux), interior, loss

    # -- B_k ------------------------------------------------------------------------------------------
    def backward_cell(self, k, interior, dbnd, src_mb, tgt_mb):
        """B_k: given the gradient (dx, daux) of the cell's output pair, accumulates the cell's parameter
        gradients and returns the gradient of its input pair."""
        s, p, g, r = self.s, self.p, self.g, self.rnd
        nb, S = tgt_mb.shape
        da = s.d_attn
        if k == self.K - 1:
            dl = interior["dlogits"]
            g["w_out"] += interior["y"].T @ dl
            dyv = r(dl @ p["w_out"].T)
            dx, dg_, db_ = layernorm_bwd(dyv, interior["xhat_f"], interior["rstd_f"], p["lnf_g"])
            g["lnf_g"] += dg_
            g["lnf_b"] += db_
            daux = np.zeros_like(dx)                            # nothing above the last layer reads aux
        else:
            dx, daux = dbnd
        for lay in reversed(interior["layers"]):
            l = lay["l"]
            q_ = "l%d." % l
            # FFN block
            dxo = r(dx)
            h = lay["h"]
            dh = r((dxo @ p[q_ + "w_2"].T) * (h > 0))
            g[q_ + "w_2"] += h.T @ dxo
            g[q_ + "b_2"] += dxo.sum(axis=0, keepdims=True)
            dc = r(dh @ p[q_ + "w_1"].T)
            g[q_ + "w_1"] += lay["c"].T @ dh
            g[q_ + "b_1"] += dh.sum(axis=0, keepdims=True)
            dln, dg_, db_ = layernorm_bwd(dc, lay["xhat2"], lay["rstd2"], p[q_ + "ln2_g"])
            g[q_ + "ln2_g"] += dg_
            g[q_ + "ln2_b"] += db_
            dx1 = dx + dln
            if s.is_dec(l):
                # cross-attention block; the memory's gradient accumulates over the decoder layers
                dx1o = r(dx1)
                do2 = r(dx1o @ p[q_ + "w_o2"].T)
                g[q_ + "w_o2"] += lay["o2"].T @ dx1o
                g[q_ + "b_o2"] += dx1o.sum(axis=0, keepdims=True)
                dq2, dk2, dv2 = self._attend_bwd(do2, lay["q2"], lay["k2"], lay["v2"], lay["p2"], nb, S)
                dq2 = r(dq2)
                dkv = r(np.concatenate([dk2, dv2], axis=1))
                dcx = r(dq2 @ p[q_ + "w_q"].T)
                g[q_ + "w_q"] += lay["cx"].T @ dq2
                g[q_ + "b_q"] += dq2.sum(axis=0, keepdims=True)
                daux = daux + dkv @ p[q_ + "w_kv"].T
                g[q_ + "w_kv"] += lay["mem"].T @ dkv
                g[q_ + "b_kv"] += dkv.sum(axis=0, keepdims=True)
                dln, dg_, db_ = layernorm_bwd(dcx, lay["xhatx"], lay["rstdx"], p[q_ + "lnx_g"])
                g[q_ + "lnx_g"] += dg_
                g[q_ + "lnx_b"] += db_
                dx1 = dx1 + dln
            # self-attention block
            dx1o = r(dx1)
            do = r(dx1o @ p[q_ + "w_o"].T)
            g[q_ + "w_o"] += lay["o"].T @ dx1o
            g[q_ + "b_o"] += dx1o.sum(axis=0, keepdims=True)
            dq, dk, dv = self._attend_bwd(do, lay["q"], lay["k"], lay["v"], lay["p"], nb, S)
            dqkv = r(np.concatenate([dq, dk, dv], axis=1))
            da_ = r(dqkv @ p[q_ + "w_qkv"].T)
            g[q_ + "w_qkv"] += lay["a"].T @ dqkv
            g[q_ + "b_qkv"] += dqkv.sum(axis=0, keepdims=True)
            dln, dg_, db_ = layernorm_bwd(da_, lay["xhat1"], lay["rstd1"], p[q_ + "ln1_g"])
            g[q_ + "ln1_g"] += dg_
            g[q_ + "ln1_b"] += db_
            dx = dx1 + dln
            if l == s.n_enc:                                    # back through the transition
                dmem = r(daux)
                dxs, dg_, db_ = layernorm_bwd(dmem, lay["xhat_e"], lay["rstd_e"], p["lne_g"])
                g["lne_g"] += dg_
                g["lne_b"] += db_
                dx, daux = dxs, dx                              # x: source stream, aux: target embedding
        if k == 0:
            np.add.at(g["emb"], src_mb.reshape(-1), dx)         # dE[src] += d(source embedding)
            np.add.at(g["emb"], tgt_mb.reshape(-1), daux)       # dE[tgt] += d(target embedding)
            return None
        return dx, daux

    # -- one mini-batch -------------------------------------------------------------------------------
    def step(self, src: np.ndarray, tgt: np.ndarray, labels: np.ndarray) -> float:
        """Tick-ordered GPipe schedule, identical to oracle/gpipe_oracle.GPipeOracle.step."""
        s, K, M = self.s, self.K, self.M
        N, S = tgt.shape
        if src.shape != tgt.shape or labels.shape != tgt.shape:
            raise ValueError("source, target and labels must all be [N, S] (reading B4)")
        if N % M != 0:
            raise ValueError("mini-batch must split into M equal micro-batches (PAPER.md:67)")
        if S != s.seq_len:
            raise ValueError("seq_len mismatch")
        for a in (src, tgt, labels):
            if a.min() < 0 or a.max() >= s.vocab:
                raise ValueError("id outside [0, V)")
        nb = N // M
        T_total = N * S
        cut = lambda a: [a[m * nb:(m + 1) * nb] for m in range(M)]
        srcs, tgts, labs = cut(src), cut(tgt), cut(labels)
        slot = [[None] * M for _ in range(K + 1)]
        stored = [[None] * M for _ in range(K)]
        loss = self.dt(0)
        self.trace = []
        for tau in range(M + K - 1):
            for k in range(K):
                m = tau - k
                if not (0 <= m < M):
                    continue
                out, interior, l_m = self.forward_cell(k, slot[k][m], srcs[m], tgts[m], labs[m], T_total,
                                                       keep=not self.remat)
                self.trace.append(("F", k, m))
                if k + 1 < K:
                    slot[k + 1][m] = out
                else:
                    loss = loss + l_m
                if not self.remat:
                    stored[k][m] = interior
        dslot = [[None] * M for _ in range(K + 1)]
        for tau in range(M + K - 1):
            for k in range(K - 1, -1, -1):
                m = M - 1 - (tau - (K - 1 - k))
                if not (0 <= m < M):
                    continue
                if self.remat:
                    _, interior, _ = self.forward_cell(k, slot[k][m], srcs[m], tgts[m], labs[m], T_total, keep=True)
                    self.trace.append(("R", k, m))
                else:
                    interior = stored[k][m]
                if k == K - 1:
                    self.per_token_loss[m] = interior["per_tok"]
                dslot[k][m] = self.backward_cell(k, interior, dslot[k + 1][m], srcs[m], tgts[m])
                self.trace.append(("B", k, m))
                stored[k][m] = None
                slot[k + 1][m] = None
                dslot[k + 1][m] = None
        return float(loss)

    def loss_only(self, src, tgt, labels) -> float:
        N, S = tgt.shape
        nb = N // self.M
        total = self.dt(0)
        for m in range(self.M):
            sl = slice(m * nb, (m + 1) * nb)
            bnd = None
            for k in range(self.K):
                bnd, _, l_m = self.forward_cell(k, bnd, src[sl], tgt[sl], labels[sl], N * S, keep=False)
            total = total + l_m
        return float(total)

"""CPU ORACLE for the GPipe Transformer hot path.  TEST INFRASTRUCTURE, NOT PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this.  It shares no code with the CUDA path (paper_1811_06965_b200/) and
neither imports the other.

What it is: a plain, slow, obviously-correct numpy implementation of what the path computes,
written from /root/reference/PAPER.md and the readings listed in DESIGN.md:

  * the model is a sequence of layers grouped into K consecutive cells (2.1);
  * a mini-batch of N sequences is divided into M equal micro-batches which are pipelined
    through the cells; the backward pass of each micro-batch uses the same weights; the
    gradients of all M micro-batches are accumulated and applied once (2.2);
  * with re-materialization only the cell-boundary activations are stored and cell k
    recomputes F_k in the backward pass (2.3).

The *result* is exactly the gradient of the full mini-batch mean loss;
the *structure* (cells, ticks, boundary-only storage, replay) follows the method so that
the structural claims can be pinned (tests/test_oracle_pins.py).

Precision: `dtype` is np.float64 (default; the reference for parity) or np.float32 (the
"plain fp32 CPU implementation" BASELINE.json names; used for the M/K-invariance pin).
A matmul is numpy's `@`; there is no blocking, fusion or reordering beyond that.

`round_operands=True` additionally applies bf16 round-to-nearest-even at the points where the
bf16 CUDA path *stores* a tensor in bf16; it is the same
code plus one rounding function and is only used to report the bf16 noise floor (reading A14:
tests/golden/make_bf16_floor.py -> tests/golden/bf16_floor.json).  Pinned by
test_round_operands_mode_matches_independent_straight_through_model: an independent torch-autograd
model with torch's own bf16 conversion applied straight-through to the listed tensors.

Pins: see tests/test_oracle_pins.py - Table 1 parameter counts, section 5
model sizes, fp64 finite differences, M/K invariance, remat == stored,
closed-form loss at init, zero-sum identities, 0-layer = multinomial logistic regression,
uniform-score attention = prefix mean, SGD update identity, activation-memory law
(PAPER.md:87).
"""
from __future__ import annotations

import math
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np


# --------------------------------------------------------------------------------------
# Model description
# --------------------------------------------------------------------------------------
class Spec:
    """The 'sequence and definitions of L layers'.  Every layer is a pre-LN
    self-attention + ReLU-FFN Transformer layer (reading A2); `causal[l]` selects the mask."""

    def __init__(self, n_layers, d_model, d_ffn, n_heads, d_head, vocab, seq_len,
                 causal: Optional[Sequence[int]] = None, ln_eps: float = 1e-5):
        self.n_layers, self.d_model, self.d_ffn = int(n_layers), int(d_model), int(d_ffn)
        self.n_heads = int(n_heads)
        self.d_head = int(d_head) if d_head else self.d_model // self.n_heads
        self.vocab, self.seq_len = int(vocab), int(seq_len)
        self.causal = [1] * self.n_layers if causal is None else [int(c) for c in causal]
        assert len(self.causal) == self.n_layers
        self.ln_eps = float(ln_eps) if ln_eps else 1e-5

    @property
    def d_attn(self):
        return self.n_heads * self.d_head


def tensor_list(s: Spec) -> List[Tuple[str, Tuple[int, int]]]:
    """Canonical parameter inventory, y = x @ W convention (readings A2, A6, A7): untied
    embedding and output matrix, biases on all four linears, two LayerNorms per layer, a final
    LayerNorm, no learned positions.  Pinned by Table 1."""
    d, H, da, V = s.d_model, s.d_ffn, s.d_attn, s.vocab
    out = [("emb", (V, d))]
    for l in range(s.n_layers):
        p = "l%d." % l
        out += [(p + "ln1_g", (1, d)), (p + "ln1_b", (1, d)),
                (p + "w_qkv", (d, 3 * da)), (p + "b_qkv", (1, 3 * da)),
                (p + "w_o", (da, d)), (p + "b_o", (1, d)),
                (p + "ln2_g", (1, d)), (p + "ln2_b", (1, d)),
                (p + "w_1", (d, H)), (p + "b_1", (1, H)),
                (p + "w_2", (H, d)), (p + "b_2", (1, d))]
    out += [("lnf_g", (1, d)), ("lnf_b", (1, d)), ("w_out", (d, V))]
    return out


def param_count(s: Spec, include_final_ln: bool = True) -> int:
    n = sum(r * c for _, (r, c) in tensor_list(s))
    if not include_final_ln:
        n -= 2 * s.d_model
    return n


def cell_layers(n_layers: int, K: int, k: int) -> range:
    """Consecutive layers of cell k.  L % K != 0: the first L mod K cells get
    one extra layer (reading on uneven splits)."""
    base, extra = divmod(n_layers, K)
    lo = k * base + min(k, extra)
    return range(lo, lo + base + (1 if k < extra else 0))


def positional_table(S: int, d: int, dtype) -> np.ndarray:
    """Fixed sinusoidal table (reading A6), evaluated in double:
    PE[t,2i] = sin(t / 10000^(2i/d)), PE[t,2i+1] = cos(t / 10000^(2i/d))."""
    pe = np.zeros((S, d), np.float64)
    for t in range(S):
        for j in range(d):
            i2 = j - (j % 2)
            ang = t / (10000.0 ** (i2 / d))
            pe[t, j] = math.sin(ang) if j % 2 == 0 else math.cos(ang)
    return pe.astype(np.float32).astype(dtype)      # stored fp32 on both sides


def bf16_rne(a: np.ndarray) -> np.ndarray:
    """Value of `a` after a store to bf16 (round-to-nearest-even) and reload."""
    a32 = np.ascontiguousarray(a, dtype=np.float32)
    u = a32.view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(a32.shape).astype(a.dtype)


# --------------------------------------------------------------------------------------
# Layer operators (each usable on its own by the per-kernel parity tests)
# --------------------------------------------------------------------------------------
def layernorm_fwd(x, g, b, eps):
    """LN(x) = (x - mu)/sqrt(var + eps) * g + b, biased variance over the feature axis."""
    mu = x.mean(axis=-1, keepdims=True)
    xc = x - mu
    var = (xc * xc).mean(axis=-1, keepdims=True)
    rstd = 1.0 / np.sqrt(var + x.dtype.type(eps))
    xhat = xc * rstd
    return xhat * g + b, xhat, rstd


def layernorm_bwd(dy, xhat, rstd, g):
    """dxhat = dy*g; dx = (dxhat - mean(dxhat) - xhat*mean(dxhat*xhat)) * rstd;
    dg = sum_t dy*xhat; db = sum_t dy."""
    dxhat = dy * g
    m1 = dxhat.mean(axis=-1, keepdims=True)
    m2 = (dxhat * xhat).mean(axis=-1, keepdims=True)
    dx = (dxhat - m1 - xhat * m2) * rstd
    dg = (dy * xhat).sum(axis=0, keepdims=True)
    db = dy.sum(axis=0, keepdims=True)
    return dx, dg, db


def attention_fwd(q, k, v, n_heads, d_head, causal, rnd=None):
    """Per sequence, per head: p = softmax_j(q_i.k_j / sqrt(d_head) [+ -inf for j > i]);
    o_i = sum_j p_ij v_j.  q, k, v: [S, n_heads*d_head]; head h owns columns h*d_head..  .
    Returns o [S, d_attn] and the list of p matrices (one [S,S] per head)."""
    S = q.shape[0]
    o = np.zeros_like(q)
    ps = []
    scale = q.dtype.type(1.0 / math.sqrt(d_head))
    for h in range(n_heads):
        c = slice(h * d_head, (h + 1) * d_head)
        s = (q[:, c] @ k[:, c].T) * scale
        if causal:
            for i in range(S):
                s[i, i + 1:] = -np.inf
        s = s - s.max(axis=1, keepdims=True)
        e = np.exp(s)
        p = e / e.sum(axis=1, keepdims=True)
        ps.append(p)
        o[:, c] = (rnd(p) if rnd else p) @ v[:, c]
    return o, ps


def attention_bwd(do, q, k, v, ps, n_heads, d_head, rnd=None):
    """dp = do v^T; dv = p^T do; ds = p * (dp - sum_j p_j dp_j); dq = ds k / sqrt(d_head);
    dk = ds^T q / sqrt(d_head).  Masked entries have p = 0 hence ds = 0."""
    dq, dk, dv = np.zeros_like(q), np.zeros_like(k), np.zeros_like(v)
    scale = q.dtype.type(1.0 / math.sqrt(d_head))
    for h in range(n_heads):
        c = slice(h * d_head, (h + 1) * d_head)
        p = ps[h]
        dp = do[:, c] @ v[:, c].T
        dv[:, c] = (rnd(p) if rnd else p).T @ do[:, c]
        ds = p * (dp - (p * dp).sum(axis=1, keepdims=True))
        if rnd:
            ds = rnd(ds)
        dq[:, c] = (ds @ k[:, c]) * scale
        dk[:, c] = (ds.T @ q[:, c]) * scale
    return dq, dk, dv


def softmax_ce(logits, labels, T_total):
    """loss = sum_t [log sum_v exp(logits_tv - max_t) + max_t - logits_t,label_t] / T_total;
    dlogits = (softmax - onehot) / T_total.  T_total is the token count of the WHOLE
    mini-batch (reading A8), which is what makes accumulation over micro-batches exact."""
    mx = logits.max(axis=1, keepdims=True)
    e = np.exp(logits - mx)
    se = e.sum(axis=1, keepdims=True)
    rows = np.arange(logits.shape[0])
    per_tok = np.log(se[:, 0]) + mx[:, 0] - logits[rows, labels]
    loss = per_tok.sum() / T_total
    dl = e / se
    dl[rows, labels] -= 1.0
    dl = dl / logits.dtype.type(T_total)
    return loss, dl


# --------------------------------------------------------------------------------------
# The GPipe engine
# --------------------------------------------------------------------------------------
class GPipeOracle:
    """gpipe_create / gpipe_step / gpipe_apply_sgd on the host (BASELINE.json north_star)."""

    def __init__(self, spec: Spec, K: int, M: int, remat: bool, dtype=np.float64,
                 round_operands: bool = False, cell_lo=None):
        if K < 1 or K > max(spec.n_layers, 1) or M < 1:
            raise ValueError("need 1 <= K <= L and M >= 1")
        self.s, self.K, self.M, self.remat = spec, int(K), int(M), bool(remat)
        # cells are ANY consecutive partition of the layers; default: the equal split
        if cell_lo is None:
            self.cells = [cell_layers(spec.n_layers, self.K, k) for k in range(self.K)]
        else:
            if (len(cell_lo) != self.K + 1 or cell_lo[0] != 0 or cell_lo[-1] != spec.n_layers
                    or any(cell_lo[k] >= cell_lo[k + 1] for k in range(self.K))):
                raise ValueError("cell_lo must be K+1 strictly increasing boundaries from 0 to L")
            self.cells = [range(cell_lo[k], cell_lo[k + 1]) for k in range(self.K)]
        self.dt = np.dtype(dtype).type
        self.rnd = bf16_rne if round_operands else (lambda a: a)
        self.names = [n for n, _ in tensor_list(spec)]
        self.shapes = dict(tensor_list(spec))
        self.p: Dict[str, np.ndarray] = {n: np.zeros(sh, self.dt) for n, sh in self.shapes.items()}
        self.g: Dict[str, np.ndarray] = {n: np.zeros(sh, self.dt) for n, sh in self.shapes.items()}
        self.pe = positional_table(spec.seq_len, spec.d_model, self.dt)
        # bookkeeping for the structural pins
        self.trace: List[Tuple[str, int, int]] = []     # (kind, k, m) in execution order
        self.peak_act_elems = 0                          # stored-activation high water
        self._live_act = 0
        self.relu_masks: Dict[Tuple[int, int], np.ndarray] = {}   # (layer, m) -> h > 0
        self.keep_relu_masks = False

    # -- parameters ------------------------------------------------------------------
    def set_params(self, params: Dict[str, np.ndarray]):
        for n in self.names:
            self.p[n] = np.array(params[n], dtype=self.dt).reshape(self.shapes[n])

    def zero_grads(self):
        for n in self.names:
            self.g[n][...] = 0

    def apply_sgd(self, lr: float):
        """w <- w - lr * g once per mini-batch, then g <- 0."""
        lr = self.dt(lr)
        for n in self.names:
            self.p[n] = self.p[n] - lr * self.g[n]
        self.zero_grads()

    def apply_rmsprop(self, lr: float, rho: float = 0.9, eps: float = 1e-8):
        """RMSProp, the optimizer of the paper's memory table (12 bytes per parameter = weight +
        gradient + one slot).  The paper does not spell the update out; reading A20: the slot starts
        at 0, ms <- rho ms + (1 - rho) g^2, w <- w - lr g / (sqrt(ms) + eps), then g <- 0."""
        if not hasattr(self, "ms"):
            self.ms = {n: np.zeros(sh, self.dt) for n, sh in self.shapes.items()}
        lr, rho, eps = self.dt(lr), self.dt(rho), self.dt(eps)
        for n in self.names:
            self.ms[n] = rho * self.ms[n] + (self.dt(1) - rho) * self.g[n] * self.g[n]
            self.p[n] = self.p[n] - lr * self.g[n] / (np.sqrt(self.ms[n]) + eps)
        self.zero_grads()

    # -- activation-memory accounting -------------------------------------
    def _hold(self, n_elems):
        self._live_act += n_elems
        self.peak_act_elems = max(self.peak_act_elems, self._live_act)

    def _release(self, n_elems):
        self._live_act -= n_elems

    @staticmethod
    def _interior_elems(interior) -> int:
        n = 0
        for lay in interior["layers"]:
            for key, val in lay.items():
                if key == "p":
                    n += sum(sum(p.size for p in ps) for ps in val)
                elif isinstance(val, np.ndarray):
                    n += val.size
        for key in ("xhat_f", "rstd_f", "y", "dlogits"):
            if key in interior and isinstance(interior[key], np.ndarray):
                n += interior[key].size
        return n

    # -- F_k -------------------------------------------------------------------------------
    def forward_cell(self, k, x_in, tokens_mb, labels_mb, T_total, keep):
        """F_k = f_j o ... o f_i.  Cell 0 starts with the embedding; cell K-1 ends
        with final LN, output projection and the loss.  Returns (output, interior, loss);
        interior is None unless `keep`."""
        s, p, r = self.s, self.p, self.rnd
        nb, S = tokens_mb.shape
        interior = {"layers": []} if keep else None
        if k == 0:
            x = p["emb"][tokens_mb.reshape(-1)] + np.tile(self.pe, (nb, 1))
        else:
            x = x_in
        for l in self.cells[k]:
            q_ = "l%d." % l
            a, xhat1, rstd1 = layernorm_fwd(x, p[q_ + "ln1_g"], p[q_ + "ln1_b"], s.ln_eps)
            a = r(a)
            qkv = r(a @ p[q_ + "w_qkv"] + p[q_ + "b_qkv"])
            da = s.d_attn
            qm, km, vm = qkv[:, :da], qkv[:, da:2 * da], qkv[:, 2 * da:]
            o = np.zeros_like(qm)
            ps_all = []
            for b in range(nb):
                rows = slice(b * S, (b + 1) * S)
                ob, ps = attention_fwd(qm[rows], km[rows], vm[rows], s.n_heads, s.d_head,
                                       s.causal[l], rnd=(r if r is bf16_rne else None))
                o[rows] = ob
                ps_all.append(ps)
            o = r(o)
            x1 = x + o @ p[q_ + "w_o"] + p[q_ + "b_o"]
            c, xhat2, rstd2 = layernorm_fwd(x1, p[q_ + "ln2_g"], p[q_ + "ln2_b"], s.ln_eps)
            c = r(c)
            z = c @ p[q_ + "w_1"] + p[q_ + "b_1"]
            h = r(np.maximum(z, 0))
            x2 = x1 + h @ p[q_ + "w_2"] + p[q_ + "b_2"]
            if keep:
                interior["layers"].append(dict(l=l, xhat1=xhat1, rstd1=rstd1, a=a, q=qm, k=km,
                                               v=vm, p=ps_all, o=o, xhat2=xhat2, rstd2=rstd2,
                                               c=c, h=h))
            x = x2
        loss = None
        if k == self.K - 1:
            y, xhat_f, rstd_f = layernorm_fwd(x, p["lnf_g"], p["lnf_b"], s.ln_eps)
            y = r(y)
            logits = r(y @ p["w_out"])
            loss, dlogits = softmax_ce(logits, labels_mb.reshape(-1), T_total)
            if keep:
                interior.update(xhat_f=xhat_f, rstd_f=rstd_f, y=y, dlogits=r(dlogits))
        return x, interior, loss

    # -- B_k -------------------------------------------------------------------------------
    def backward_cell(self, k, interior, dy, tokens_mb, m):
        """B_k: back-propagation through cell k given the gradient dy of its output
        (Fig. 2 caption: B_k depends on B_{k+1} and on F_k's activations).
        Accumulates parameter gradients into self.g and returns the gradient of its input."""
        s, p, g, r = self.s, self.p, self.g, self.rnd
        nb, S = tokens_mb.shape
        if k == self.K - 1:
            dl = interior["dlogits"]
            g["w_out"] += interior["y"].T @ dl
            dyv = r(dl @ p["w_out"].T)
            dx, dg_, db_ = layernorm_bwd(dyv, interior["xhat_f"], interior["rstd_f"], p["lnf_g"])
            g["lnf_g"] += dg_
            g["lnf_b"] += db_
        else:
            dx = dy
        for lay in reversed(interior["layers"]):
            l = lay["l"]
            q_ = "l%d." % l
            dxo = r(dx)                                     # bf16 operand copy of the residual grad
            # FFN
            h = lay["h"]
            if self.keep_relu_masks:
                self.relu_masks[(l, m)] = h > 0
            dh = r((dxo @ p[q_ + "w_2"].T) * (h > 0))      # ReLU'(0) = 0 (reading A13)
            g[q_ + "w_2"] += h.T @ dxo
            g[q_ + "b_2"] += dxo.sum(axis=0, keepdims=True)
            dc = r(dh @ p[q_ + "w_1"].T)
            g[q_ + "w_1"] += lay["c"].T @ dh
            g[q_ + "b_1"] += dh.sum(axis=0, keepdims=True)
            dln, dg_, db_ = layernorm_bwd(dc, lay["xhat2"], lay["rstd2"], p[q_ + "ln2_g"])
            g[q_ + "ln2_g"] += dg_
            g[q_ + "ln2_b"] += db_
            dx1 = dx + dln                                   # residual adds gradients
            dx1o = r(dx1)
            # attention
            do = r(dx1o @ p[q_ + "w_o"].T)
            g[q_ + "w_o"] += lay["o"].T @ dx1o
            g[q_ + "b_o"] += dx1o.sum(axis=0, keepdims=True)
            dq, dk, dv = np.zeros_like(do), np.zeros_like(do), np.zeros_like(do)
            for b in range(nb):
                rows = slice(b * S, (b + 1) * S)
                dq[rows], dk[rows], dv[rows] = attention_bwd(
                    do[rows], lay["q"][rows], lay["k"][rows], lay["v"][rows], lay["p"][b],
                    s.n_heads, s.d_head, rnd=(r if r is bf16_rne else None))
            dqkv = r(np.concatenate([dq, dk, dv], axis=1))
            da_ = r(dqkv @ p[q_ + "w_qkv"].T)
            g[q_ + "w_qkv"] += lay["a"].T @ dqkv
            g[q_ + "b_qkv"] += dqkv.sum(axis=0, keepdims=True)
            dln, dg_, db_ = layernorm_bwd(da_, lay["xhat1"], lay["rstd1"], p[q_ + "ln1_g"])
            g[q_ + "ln1_g"] += dg_
            g[q_ + "ln1_b"] += db_
            dx = dx1 + dln
        if k == 0:
            np.add.at(g["emb"], tokens_mb.reshape(-1), dx)   # dE[tok] += dx0
            return None
        return dx

    # -- one mini-batch ----------------------------------------------------------------------
    def step(self, tokens: np.ndarray, labels: np.ndarray) -> float:
        """gpipe_step: adds d(mean loss)/dw of this mini-batch into the gradient buffers and
        returns the mini-batch mean loss.  Tick-ordered GPipe schedule (
        Fig. 2c is an image, so the order below is reading A1)."""
        s, K, M = self.s, self.K, self.M
        N, S = tokens.shape
        if N % M != 0:
            raise ValueError("mini-batch must split into M equal micro-batches (PAPER.md:67)")
        if S != s.seq_len:
            raise ValueError("seq_len mismatch")
        if tokens.min() < 0 or tokens.max() >= s.vocab or labels.min() < 0 or labels.max() >= s.vocab:
            raise ValueError("token/label outside [0, V)")
        nb = N // M
        T_total = N * S
        tok = [tokens[m * nb:(m + 1) * nb] for m in range(M)]     # a1: micro-batch split
        lab = [labels[m * nb:(m + 1) * nb] for m in range(M)]
        slot = [[None] * M for _ in range(K + 1)]     # slot[k][m] = input of cell k
        stored = [[None] * M for _ in range(K)]       # interiors kept when remat is off
        loss = self.dt(0)
        self.trace = []
        # forward ticks
        for tau in range(M + K - 1):
            for k in range(K):
                m = tau - k
                if not (0 <= m < M):
                    continue
                out, interior, l_m = self.forward_cell(k, slot[k][m], tok[m], lab[m], T_total,
                                                       keep=not self.remat)
                self.trace.append(("F", k, m))
                if k + 1 < K:
                    slot[k + 1][m] = out
                    self._hold(out.size)                  # boundary activation
                else:
                    loss = loss + l_m
                if not self.remat:
                    stored[k][m] = interior
                    self._hold(self._interior_elems(interior))
        # backward ticks
        dslot = [[None] * M for _ in range(K + 1)]
        for tau in range(M + K - 1):
            for k in range(K - 1, -1, -1):
                m = M - 1 - (tau - (K - 1 - k))
                if not (0 <= m < M):
                    continue
                if self.remat:
                    _, interior, _ = self.forward_cell(k, slot[k][m], tok[m], lab[m], T_total, keep=True)
                    self.trace.append(("R", k, m))
                    self._hold(self._interior_elems(interior))
                else:
                    interior = stored[k][m]
                dslot[k][m] = self.backward_cell(k, interior, dslot[k + 1][m], tok[m], m)
                self.trace.append(("B", k, m))
                self._release(self._interior_elems(interior))
                stored[k][m] = None
                if k + 1 < K and slot[k + 1][m] is not None:
                    self._release(slot[k + 1][m].size)    # boundary no longer needed
                    slot[k + 1][m] = None
                dslot[k + 1][m] = None
        return float(loss)

    # -- convenience ---------------------------------------------------------------------------
    def loss_only(self, tokens, labels) -> float:
        """Mean loss of the mini-batch by running every micro-batch through the cells in order;
        no gradient side effects (used by the finite-difference pin)."""
        N, S = tokens.shape
        nb = N // self.M
        total = self.dt(0)
        for m in range(self.M):
            tk, lb = tokens[m * nb:(m + 1) * nb], labels[m * nb:(m + 1) * nb]
            x = None
            for k in range(self.K):
                x, _, l_m = self.forward_cell(k, x, tk, lb, N * S, keep=False)
            total = total + l_m
        return float(total)

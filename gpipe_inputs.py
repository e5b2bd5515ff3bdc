"""Seeded synthetic inputs and workload shapes, shared by the tests, bench.py, the oracle's
callers and the CUDA path's callers.

This module holds NONE of the method's arithmetic: only shapes (BASELINE.json `configs`),
random draws, and the bf16 round-to-nearest-even helper used to make host arrays exactly
representable before they are handed to either side.  Neither `oracle/` nor the CUDA
package imports the other; both receive what this module generates.

Recipe (SURVEY.md 8(d) "Synthetic inputs"):
  * token ids: uniform integers on [0, V), shape [N, S+1], numpy PCG64(seed);
    tokens = ids[:, :S], labels = ids[:, 1:] ("labels = ids shifted by one", reading A9)
  * weights: N(0, 0.02) for every matrix and the embedding (BASELINE.json configs);
    for parity runs biases and LayerNorm beta ~ N(0, 0.02), gamma = 1 + N(0, 0.02)
    (reading A10: a zero bias would hide a missing-bias bug)
  * bf16 configs: every host array is RNE-rounded to bf16 first, so both sides start from
    identical values (reading A12).
The paper's own Transformer workload is an in-house corpus that is not
public; these inputs stand in for it and only its shapes are taken.
"""
from __future__ import annotations

import dataclasses
from typing import Dict, List, Optional, Tuple

import numpy as np


@dataclasses.dataclass(frozen=True)
class Workload:
    """One row of SURVEY.md 8 'config' table. dtype: 'fp32' or 'bf16'."""
    name: str
    n_layers: int
    d_model: int
    d_ffn: int
    n_heads: int
    d_head: int
    vocab: int
    seq_len: int
    n_seqs: int          # N, sequences per mini-batch
    M: int               # micro-batches
    K: int               # cells
    dtype: str
    causal: Tuple[int, ...]
    remat: bool = True
    ln_eps: float = 1e-5
    n_dec: int = 0            # > 0: encoder-decoder T(L,H,A): the LAST n_dec layers are decoder layers
    logit_clip: float = 0.0   # > 0: clamp the logits to [-c, c] before the softmax

    @property
    def n_enc(self) -> int:
        return self.n_layers - self.n_dec

    @property
    def d_attn(self) -> int:
        return self.n_heads * self.d_head

    @property
    def tokens_per_step(self) -> int:
        return self.n_seqs * self.seq_len

    def replace(self, **kw) -> "Workload":
        return dataclasses.replace(self, **kw)


def _wl(name, L, d, H, A, dh, V, S, N, M, K, dtype, causal=None, remat=True):
    if causal is None:
        causal = (1,) * L                     # reading A4: configs 1-4 all-causal
    return Workload(name, L, d, H, A, dh, V, S, N, M, K, dtype, tuple(causal), remat)


# BASELINE.json configs[0..4]; d_head per reading A3 (d_head = 64 where d/A would give 32).
CONFIGS: Dict[str, Workload] = {
    "tiny":           _wl("tiny", 2, 64, 256, 4, 16, 512, 16, 8, 4, 2, "fp32"),
    "T(6,4096,16)":   _wl("T(6,4096,16)", 6, 1024, 4096, 16, 64, 32000, 256, 64, 8, 2, "bf16"),
    "T(12,8192,16)":  _wl("T(12,8192,16)", 12, 1024, 8192, 16, 64, 32000, 256, 256, 32, 4, "bf16"),
    "T(24,16384,32)": _wl("T(24,16384,32)", 24, 1024, 16384, 32, 64, 32000, 256, 256, 32, 8, "bf16"),
    "T(64,16384,32)": _wl("T(64,16384,32)", 128, 1024, 16384, 32, 64, 64000, 256, 128, 16, 16, "bf16",
                          causal=(0,) * 64 + (1,) * 64),
}
CONFIG_ORDER = ["tiny", "T(6,4096,16)", "T(12,8192,16)", "T(24,16384,32)", "T(64,16384,32)"]


def reduced(w: Workload, layers_per_cell: int = 1, seqs_per_microbatch: int = 1) -> Workload:
    """Shape-preserving reduction (SURVEY.md 8(c) 'Big-config parity'): same d, H, A, d_head,
    V, S, K and M, but `layers_per_cell` layers per cell and `seqs_per_microbatch` sequences
    per micro-batch; the causal pattern keeps its non-causal/causal proportions."""
    L = w.K * layers_per_cell
    n_causal = round(L * sum(w.causal) / len(w.causal))
    causal = (0,) * (L - n_causal) + (1,) * n_causal
    n_dec = round(L * w.n_dec / w.n_layers)          # encoder-decoder: keep the encoder / decoder proportion
    return w.replace(name=w.name + "-reduced", n_layers=L, n_seqs=w.M * seqs_per_microbatch,
                     causal=causal, n_dec=n_dec)


def tensor_shapes(w: Workload) -> List[Tuple[str, Tuple[int, int]]]:
    """Canonical tensor list: names and [rows, cols]; vectors are [1, n].
    A naming/shape convention only - each side builds its own list and the tests compare.
    Encoder-decoder workloads (n_dec > 0): `lne_*` (encoder output LayerNorm) sits in front of the first
    decoder layer and every decoder layer carries the cross-attention block after its self-attention."""
    d, H, da, V = w.d_model, w.d_ffn, w.d_attn, w.vocab
    out = [("emb", (V, d))]
    for l in range(w.n_layers):
        p = f"l{l}."
        dec = w.n_dec > 0 and l >= w.n_enc
        if dec and l == w.n_enc:
            out += [("lne_g", (1, d)), ("lne_b", (1, d))]
        out += [(p + "ln1_g", (1, d)), (p + "ln1_b", (1, d)),
                (p + "w_qkv", (d, 3 * da)), (p + "b_qkv", (1, 3 * da)),
                (p + "w_o", (da, d)), (p + "b_o", (1, d))]
        if dec:
            out += [(p + "lnx_g", (1, d)), (p + "lnx_b", (1, d)),
                    (p + "w_q", (d, da)), (p + "b_q", (1, da)),
                    (p + "w_kv", (d, 2 * da)), (p + "b_kv", (1, 2 * da)),
                    (p + "w_o2", (da, d)), (p + "b_o2", (1, d))]
        out += [(p + "ln2_g", (1, d)), (p + "ln2_b", (1, d)),
                (p + "w_1", (d, H)), (p + "b_1", (1, H)),
                (p + "w_2", (H, d)), (p + "b_2", (1, d))]
    out += [("lnf_g", (1, d)), ("lnf_b", (1, d)), ("w_out", (d, V))]
    return out


def bf16_round(a: np.ndarray) -> np.ndarray:
    """fp32 -> nearest-even bf16 -> fp32 (value-preserving container). Used only to make the
    host-side *inputs* bf16-representable; no model arithmetic."""
    a32 = np.ascontiguousarray(a, dtype=np.float32)
    u = a32.view(np.uint32).astype(np.uint64)
    lsb = (u >> 16) & 1
    u = (u + 0x7FFF + lsb) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(a32.shape)


def make_tokens(w: Workload, seed: int) -> Tuple[np.ndarray, np.ndarray]:
    """ids uniform on [0, V), [N, S+1]; tokens = ids[:, :S]; labels = ids[:, 1:]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    ids = rng.integers(0, w.vocab, size=(w.n_seqs, w.seq_len + 1), dtype=np.int64)
    tokens = np.ascontiguousarray(ids[:, :-1]).astype(np.int32)
    labels = np.ascontiguousarray(ids[:, 1:]).astype(np.int32)
    return tokens, labels


def make_tokens_encdec(w: Workload, seed: int) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Encoder-decoder inputs: source ids uniform on [0, V), [N, S]; target ids [N, S+1], target tokens =
    ids[:, :S], labels = ids[:, 1:] (the decoder predicts the next target id)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    src = rng.integers(0, w.vocab, size=(w.n_seqs, w.seq_len), dtype=np.int64).astype(np.int32)
    ids = rng.integers(0, w.vocab, size=(w.n_seqs, w.seq_len + 1), dtype=np.int64)
    return (np.ascontiguousarray(src), np.ascontiguousarray(ids[:, :-1]).astype(np.int32),
            np.ascontiguousarray(ids[:, 1:]).astype(np.int32))


def encdec(name: str, L: int, H: int, A: int, vocab: int = 64000, n_seqs: int = 128, M: int = 16, K: int = 16,
           d_model: int = 1024, d_head: int = 64, seq_len: int = 256, dtype: str = "bf16", logit_clip: float = 0.0,
           remat: bool = True) -> Workload:
    """T(L,H,A) of PAPER.md:160: L encoder layers followed by L decoder layers, d_model 1024."""
    return Workload(name, 2 * L, d_model, H, A, d_head, vocab, seq_len, n_seqs, M, K, dtype,
                    (0,) * L + (1,) * L, remat, 1e-5, L, logit_clip)


# The paper's own 6.04 B model: 64 encoder + 64 decoder layers, on the K = M = 16 schedule of
# BASELINE.json configs[4].  Not one of BASELINE.json's configs: bench.py --workload selects it.
ENCDEC_CONFIGS: Dict[str, Workload] = {
    "T(64,16384,32)-encdec": encdec("T(64,16384,32)-encdec", 64, 16384, 32),
}


def make_params(w: Workload, seed: int, std: float = 0.02, parity: bool = True,
                round_bf16: Optional[bool] = None, ffn_depth_scale: bool = False) -> Dict[str, np.ndarray]:
    """N(0, std) matrices; parity=True also randomises biases / beta and gamma = 1 + N(0,std);
    parity=False gives gamma = 1, beta = b = 0 (benchmark init). fp32 arrays, [rows, cols].
    ffn_depth_scale: w_1 and w_2 are drawn with std / n_layers (PAPER.md:174 (i): "we scale down the
    initialization of all transformer feed-forward layers by the number of layers")."""
    if round_bf16 is None:
        round_bf16 = (w.dtype == "bf16")
    rng = np.random.Generator(np.random.PCG64(seed))
    out: Dict[str, np.ndarray] = {}
    for name, shape in tensor_shapes(w):
        base = name.split(".")[-1]
        is_gamma = base.endswith("_g")
        is_vec = shape[0] == 1 and base not in ("emb", "w_out")
        if is_vec and not parity:
            a = np.ones(shape, np.float32) if is_gamma else np.zeros(shape, np.float32)
        else:
            sd = std / w.n_layers if ffn_depth_scale and base in ("w_1", "w_2") else std
            a = (rng.standard_normal(shape, dtype=np.float32) * np.float32(sd)).astype(np.float32)
            if is_gamma:
                a = (a + np.float32(1.0)).astype(np.float32)
        out[name] = bf16_round(a) if round_bf16 else a
    return out

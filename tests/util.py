"""Shared helpers of the test-suite: comparison metrics (reading A19) and oracle runners."""
import numpy as np

import gpipe_inputs as gi
from oracle import gpipe_oracle as go


def maxrel(a, b):
    """per-tensor max-relative error: max|a-b| / max|b| (reading A19)."""
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


def cosine(a, b):
    a, b = np.asarray(a, np.float64).ravel(), np.asarray(b, np.float64).ravel()
    return float(a @ b / max(np.linalg.norm(a) * np.linalg.norm(b), 1e-300))


def oracle_spec(w):
    return go.Spec(w.n_layers, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len, w.causal, w.ln_eps)


def run_oracle(w, params, tok, lab, K=None, M=None, remat=None, dtype=np.float64, round_operands=False, cell_lo=None):
    o = go.GPipeOracle(oracle_spec(w), w.K if K is None else K, w.M if M is None else M,
                       w.remat if remat is None else remat, dtype=dtype, round_operands=round_operands,
                       cell_lo=cell_lo)
    o.set_params(params)
    loss = o.step(tok, lab)
    return o, loss

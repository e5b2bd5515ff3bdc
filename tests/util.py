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


# ---------------------------------------------------------------------------------------------
# Shape-preserving reductions of BASELINE.json configs 2-5 (SURVEY.md 8(c) "Big-config parity"):
# same d, H, A, d_head, V, S, K and M as the full config, one layer per cell (L = K) and one
# sequence per micro-batch (N = M).  The oracle runs them in full.  Oracle precision: fp64 for
# configs 2 and 3; fp32 ("plain, slow fp32 CPU implementation", BASELINE.json north_star) for
# configs 4 and 5, whose 24 TFLOP per step would not fit the GPU test tier's time limit in fp64 -
# the fp32 oracle's own error (~1e-6, pin P6) is three orders below the bf16 effects compared.
# ---------------------------------------------------------------------------------------------
REDUCED_CASES = {
    "T(6,4096,16)": dict(seed_p=1012, seed_t=2012, oracle_dtype="float64"),
    "T(12,8192,16)": dict(seed_p=1013, seed_t=2013, oracle_dtype="float64"),
    "T(24,16384,32)": dict(seed_p=1014, seed_t=2014, oracle_dtype="float32"),
    "T(64,16384,32)": dict(seed_p=1015, seed_t=2015, oracle_dtype="float32"),
}


def reduced_case(name):
    """(workload, params, tokens, labels, oracle dtype) of the reduced parity case of config `name`."""
    c = REDUCED_CASES[name]
    w = gi.reduced(gi.CONFIGS[name])
    params = gi.make_params(w, c["seed_p"])                 # bf16-representable, parity init (A10, A12)
    tok, lab = gi.make_tokens(w, c["seed_t"])
    return w, params, tok, lab, np.dtype(c["oracle_dtype"]).type


def engine_program(k, K, M, remat):
    """The tasks of cell k's program (oracle/schedule.cell_program: Fig. 2c of the paper) that the CUDA engine
    actually runs.  With re-materialization it elides work whose result is already resident or never read
    (readings A15b, A15c; results bitwise unchanged): R(k, M-1) for k < K-1 - the cell's workspace still
    holds the interior of F(k, M-1) when B(k, M-1) starts - and every forward task of the last cell, whose only
    product, the loss, R(K-1, m) produces again."""
    from oracle import schedule as sch
    prog = sch.cell_program(k, K, M, remat)
    if not remat:
        return prog
    if k == K - 1:
        return [t for t in prog if t[0] != "F"]
    return [t for t in prog if t != ("R", k, M - 1)]

"""B200-native GPipe hot path (arXiv 1811.06965): micro-batched, re-materialized forward/backward
of a stack of Transformer layers behind a C ABI (include/gpipe.h).  See DESIGN.md."""
from .binding import (CATEGORIES, DTYPE_BF16, DTYPE_FP32, EXPORTED_SYMBOLS, LIB_PATH, GPipe, GPipeEncDec, GPipeError,
                      lib, make_spec, plan_bytes)

__all__ = ["GPipe", "GPipeEncDec", "GPipeError", "lib", "make_spec", "plan_bytes", "LIB_PATH", "EXPORTED_SYMBOLS",
           "CATEGORIES", "DTYPE_FP32", "DTYPE_BF16", "from_workload"]


def from_workload(w, **overrides) -> "GPipe":
    """Builds the engine for a gpipe_inputs.Workload-like object (fields: n_layers, d_model, d_ffn,
    n_heads, d_head, vocab, seq_len, dtype, K, M, remat, n_seqs, causal, ln_eps)."""
    kw = dict(n_layers=w.n_layers, d_model=w.d_model, d_ffn=w.d_ffn, n_heads=w.n_heads, d_head=w.d_head,
              vocab=w.vocab, seq_len=w.seq_len, dtype=w.dtype, K=w.K, M=w.M, remat=w.remat,
              n_seqs=w.n_seqs, causal=list(w.causal), ln_eps=w.ln_eps)
    if getattr(w, "n_dec", 0) > 0:                       # encoder-decoder T(L,H,A)
        for key in ("n_layers", "causal"):
            kw.pop(key)
        kw.update(n_enc=w.n_layers - w.n_dec, n_dec=w.n_dec, logit_clip=w.logit_clip)
        kw.update(overrides)
        return GPipeEncDec(**kw)
    kw.update(overrides)
    return GPipe(**kw)

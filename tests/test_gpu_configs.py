"""Oracle parity at the SHAPES of BASELINE.json configs 2-5 (SURVEY.md 8(c) "Big-config parity" (1)).

Each case is the shape-preserving reduction `gpipe_inputs.reduced(w)` of a config - the same d_model,
d_ffn, heads, d_head, vocabulary, sequence length, K and M as the full configuration, with one layer per
cell (L = K) and one sequence per micro-batch (N = M) - run in full through the CUDA path (C ABI) and
through the CPU oracle on the same seeded, bf16-representable parameters and token ids, and compared
tensor by tensor: every one of the 12 L + 4 gradients.  These shapes exercise what the d = 256 toy of
tests/test_gpu_engine.py cannot: d = 1024 LayerNorm rows, S = 256 (two query blocks per head, 128 x 256
score tiles), H = 16384 (256 K-blocks accumulated unsplit), V = 64000 (the deep-K dlogits product, eight
vectors per thread in the fused cross-entropy), K = 16 cells, mixed non-causal / causal masks.

Pass criteria (BASELINE.json north_star; reading A14 of DESIGN.md section 3):
  * loss within 1e-2 relative of the oracle's;
  * per-tensor gradient cosine >= 0.999, or - where ReLU-mask flips put the bf16 noise floor itself
    below 0.999 - >= floor - 5e-4, the floor being what the ORACLE produces when it rounds to bf16 at
    the CUDA path's storage points (tests/golden/bf16_floor.json, written by
    tests/golden/make_bf16_floor.py from the oracle alone);
  * the cause of the deficit is checked, not assumed: the GPU's bit-packed ReLU pattern of the last
    layer (micro-batch 0) is compared with the oracle's [z > 0], and 1 - cos(dW_1) of that layer must
    be explained by the fraction of mismatching units (a flipped unit changes its gradient row by 100 %).
Every case prints one `PARITY|` line per tensor class (pytest -s) - profiles/parity_configs_r02.md.
"""
import json
import os

import numpy as np
import pytest

import paper_1811_06965_b200 as gp
from oracle import gpipe_oracle as go
from tests.util import REDUCED_CASES, cosine, maxrel, oracle_spec, reduced_case

pytestmark = pytest.mark.gpu

FLOOR = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "bf16_floor.json")))
COS_BOUND = 0.999           # north_star
FLOOR_SLACK = 5e-4          # reading A14 (iii)


def _unpack_bits(words, T, H):
    """uint32 [T, ceil(H/32)] (bit n%32 of word n/32) -> bool [T, H]"""
    b = np.unpackbits(words.view(np.uint8).reshape(T, -1), axis=-1, bitorder="little").astype(bool)
    return b[:, :H]


def _gpu_run(w, params, tok, lab, remat):
    with gp.from_workload(w, remat=remat) as e:
        e.set_params(params)
        loss = e.step(tok, lab)
        grads = e.grads()
        T_mb = w.n_seqs // w.M * w.seq_len
        # with remat the single workspace of a cell holds the last micro-batch it replayed: m = 0
        bits = None
        if remat:
            l = w.n_layers - 1
            raw = e.debug_read("hbits", l, max_elems=T_mb * ((w.d_ffn + 31) // 32))
            bits = _unpack_bits(raw.view(np.uint32), T_mb, w.d_ffn)
            h = e.debug_read("h", l, max_elems=T_mb * w.d_ffn).reshape(T_mb, w.d_ffn)
            assert np.array_equal(bits, h > 0)               # the recorded pattern is [stored h > 0]
        peak = e.peak_bytes()["total"]
    return loss, grads, bits, peak


@pytest.mark.parametrize("name", list(REDUCED_CASES), ids=["config2", "config3", "config4", "config5"])
def test_reduced_config_matches_oracle(name):
    w, params, tok, lab, dt = reduced_case(name)
    assert name in FLOOR, "run tests/golden/make_bf16_floor.py for %s" % name
    fl = FLOOR[name]
    assert fl["workload"]["n_layers"] == w.n_layers and fl["workload"]["d_ffn"] == w.d_ffn
    assert fl["workload"]["causal"] == list(w.causal) and fl["oracle_dtype"] == REDUCED_CASES[name]["oracle_dtype"]

    loss, grads, bits, peak = _gpu_run(w, params, tok, lab, True)
    if name == "T(6,4096,16)":
        # config 2 is specified "remat on and off": the stored-activation path must reproduce the replayed one
        # bit for bit (re-materialization recomputes the same F_k)
        loss_s, grads_s, _, peak_s = _gpu_run(w, params, tok, lab, False)
        assert loss_s == loss and peak_s > peak
        for n in grads:
            assert np.array_equal(grads[n], grads_s[n]), n

    o = go.GPipeOracle(oracle_spec(w), w.K, w.M, w.remat, dtype=dt)
    o.keep_relu_masks = True
    o.set_params(params)
    loss_ref = o.step(tok, lab)
    assert abs(loss_ref - fl["loss_plain"]) <= 1e-6 * abs(loss_ref)          # same inputs as the stored floor run
    rel_loss = abs(loss - loss_ref) / abs(loss_ref)

    cos = {n: cosine(grads[n], o.g[n]) for n in grads}
    mr = {n: maxrel(grads[n], o.g[n]) for n in grads}
    floor = fl["floor_cosine"]
    classes = {}
    for n in cos:
        classes.setdefault(n.split(".")[-1], []).append(n)
    print()
    print("PARITY|%s|reduced L=%d N=%d K=%d M=%d|oracle %s|loss gpu %.6f oracle %.6f rel %.2e"
          % (name, w.n_layers, w.n_seqs, w.K, w.M, REDUCED_CASES[name]["oracle_dtype"], loss, loss_ref, rel_loss))
    for cls, names in classes.items():
        c = [cos[n] for n in names]
        f = [floor[n] for n in names]
        print("PARITY|%s|%-6s|n %3d|cos min %.6f med %.6f|floor min %.6f med %.6f|max-rel max %.2e"
              % (name, cls, len(names), min(c), float(np.median(c)), min(f), float(np.median(f)),
                 max(mr[n] for n in names)))
    allc = list(cos.values())
    below = sorted((c, n) for n, c in cos.items() if c < COS_BOUND)
    print("PARITY|%s|ALL|n %d|cos min %.6f med %.6f|floor min %.6f med %.6f|%d tensors below %.3f: %s"
          % (name, len(allc), min(allc), float(np.median(allc)), fl["min"], fl["median"], len(below), COS_BOUND,
             ", ".join("%s %.6f (floor %.6f)" % (n, c, floor[n]) for c, n in below[:6])))

    # ---- the cause: ReLU-mask mismatches of the last layer, micro-batch 0 (A14 iii) ----
    l = w.n_layers - 1
    mism = float((bits != o.relu_masks[(l, 0)]).mean())
    deficit = 1.0 - cos["l%d.w_1" % l]
    print("PARITY|%s|relu|layer %d micro-batch 0: mask mismatch %.3e (oracle bf16 floor run: %.3e) | 1 - cos(dW_1) %.3e"
          % (name, l, mism, fl["relu_mismatch_m0"][str(l)], deficit))

    assert rel_loss <= 1e-2
    for n, c in cos.items():
        assert c >= min(COS_BOUND, floor[n] - FLOOR_SLACK), (n, c, floor[n])
    # a flipped unit removes or adds its whole column of dW_1, so for the LAST layer (no flips downstream of it)
    # 1 - cos(dW_1) equals the flip fraction (measured: 7.7e-4 vs 7.5e-4 at config 2's shape, 9.7e-4 vs 9.9e-4 at
    # config 3's); the GPU's flip fraction is the one the oracle's own bf16-rounding run shows
    assert mism <= 3e-3
    assert 0.7 * mism <= deficit <= 1.4 * mism, (mism, deficit)
    assert 0.7 * fl["relu_mismatch_m0"][str(l)] <= mism <= 1.4 * fl["relu_mismatch_m0"][str(l)]

"""Cell partitioning: pins of the brute-force oracle, then the library's
exact dynamic program (host-only C-ABI calls: they run without a GPU) against it."""
import itertools
import math

import numpy as np
import pytest

import gpipe_inputs as gi
import paper_1811_06965_b200.binding as B
from oracle import gpipe_oracle as go
from oracle import partition as op


# ---- the oracle against what the definition fixes ----------------------------------------------------------
def test_oracle_enumerates_every_consecutive_partition():
    for L, K in [(5, 1), (5, 2), (6, 3), (7, 7), (9, 4)]:
        parts = list(op.all_partitions(L, K))
        assert len(parts) == math.comb(L - 1, K - 1)                     # compositions of L into K parts
        assert len({tuple(b) for b in parts}) == len(parts)
        for b in parts:
            assert b[0] == 0 and b[-1] == L and all(b[i] < b[i + 1] for i in range(K))


def test_oracle_variance_is_numpy_population_variance():
    r = np.random.default_rng(0)
    for _ in range(20):
        xs = r.random(r.integers(1, 9)) * 10
        assert abs(op.variance(list(xs)) - float(np.var(xs))) <= 1e-12 * max(1.0, float(np.var(xs)))


def test_oracle_closed_form_cases():
    # uniform costs, K | L: the equal split has variance 0 and nothing else does
    b, v = op.min_variance_partition([2.0] * 12, 4)
    assert b == [0, 3, 6, 9, 12] and v == 0.0
    # one heavy layer takes a cell of its own
    b, v = op.min_variance_partition([1, 1, 1, 3], 2)
    assert b == [0, 3, 4] and v == 0.0
    # a head worth 2 layers shortens the last cell by 2 layers (6 + 4 + head 2)
    b, v = op.min_variance_partition([1.0] * 10, 2, last_extra=2.0)
    assert b == [0, 6, 10] and v == 0.0
    # an embedding cost shortens the first cell
    b, v = op.min_variance_partition([1.0] * 9, 3, first_extra=3.0)
    assert op.cell_costs([1.0] * 9, b, 3.0, 0.0) == [4.0, 4.0, 4.0] and b == [0, 1, 5, 9]
    # K = 1 and K = L have one partition each
    assert op.min_variance_partition([3, 1, 4], 1)[0] == [0, 3]
    assert op.min_variance_partition([3, 1, 4], 3)[0] == [0, 1, 2, 3]


def test_oracle_never_worse_than_the_equal_split():
    r = np.random.default_rng(1)
    for _ in range(30):
        L = int(r.integers(2, 11)); K = int(r.integers(1, L + 1))
        c = list(r.random(L) + 0.1)
        fe, le = float(r.random() * 2), float(r.random() * 3)
        b, v = op.min_variance_partition(c, K, fe, le)
        eq = [0] + [go.cell_layers(L, K, k).stop for k in range(K)]
        assert v <= op.variance(op.cell_costs(c, eq, fe, le)) + 1e-12


def test_oracle_cost_model_matches_flop_counts():
    """SURVEY.md 8(f) f2 quotes the head as worth 0.8 / 2.6 / 1.6 layers at configs 4 / 2 / 5 (one decimal), and the
    8(d) table 0.220 / 0.575 / 2.10 / 11.07 GFLOP per token forward for configs 2 / 3 / 4 / 5 (d_head 64)."""
    for name, ratio in [("T(24,16384,32)", 0.8), ("T(6,4096,16)", 2.6), ("T(64,16384,32)", 1.6)]:
        w = gi.CONFIGS[name]
        c, emb, head = op.layer_costs(w.n_layers, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len,
                                      w.causal, remat=False)
        assert emb == 0.0 and abs(head / c[-1] - ratio) <= 0.1, (name, head / c[-1])
    for name, gf in [("T(6,4096,16)", 0.220), ("T(12,8192,16)", 0.575), ("T(24,16384,32)", 2.10), ("T(64,16384,32)", 11.07)]:
        w = gi.CONFIGS[name]
        a = op.layer_costs(w.n_layers, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len, w.causal, False)
        b = op.layer_costs(w.n_layers, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len, w.causal, True)
        fwd = sum(b[0]) - sum(a[0]) + b[2] - a[2]              # the replay is exactly one more forward
        assert abs(fwd / (gf * 1e9) - 1.0) <= 0.01, (name, fwd)


# ---- the library's dynamic program against the brute force ---------------------------------------------------
def test_library_partition_equals_brute_force():
    r = np.random.default_rng(2)
    cases = [([2.0] * 12, 4, 0.0, 0.0), ([1, 1, 1, 3], 2, 0.0, 0.0), ([1.0] * 10, 2, 0.0, 2.0), ([1.0] * 9, 3, 3.0, 0.0),
             ([5.0], 1, 1.0, 1.0), ([0.0, 0.0, 0.0], 2, 0.0, 0.0)]
    for _ in range(60):
        L = int(r.integers(1, 13)); K = int(r.integers(1, L + 1))
        # small integers: the variance of every partition is exact in fp64, so ties are real ties
        cases.append(([float(v) for v in r.integers(0, 6, size=L)], K, float(r.integers(0, 4)), float(r.integers(0, 4))))
    for _ in range(40):
        L = int(r.integers(2, 13)); K = int(r.integers(1, L + 1))
        cases.append((list(r.random(L) * 3 + 0.01), K, float(r.random()), float(r.random() * 4)))
    for c, K, fe, le in cases:
        got = B.partition_min_variance(c, fe, le, K)
        ref, ref_var = op.min_variance_partition(c, K, fe, le)
        assert got[0] == 0 and got[-1] == len(c) and all(got[i] < got[i + 1] for i in range(K)), (c, K, got)
        got_var = op.variance(op.cell_costs(c, got, fe, le))
        assert got_var <= ref_var * (1 + 1e-12) + 1e-12, (c, K, fe, le, got, ref)
        if all(float(v).is_integer() for v in c):
            assert got == ref, (c, K, fe, le, got, ref)          # same tie-break: earliest boundaries


def test_library_cost_model_equals_oracle_cost_model():
    for name in gi.CONFIG_ORDER:
        w = gi.CONFIGS[name]
        spec, _keep = B.make_spec(w.n_layers, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len, w.dtype,
                                  list(w.causal), w.ln_eps)
        for remat in (False, True):
            c, emb, head = B.layer_costs(spec, remat)
            rc, remb, rhead = op.layer_costs(w.n_layers, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len,
                                             w.causal, remat)
            assert emb == remb and abs(head - rhead) <= 1e-9 * rhead
            assert np.allclose(c, rc, rtol=1e-12, atol=0)


def test_library_partition_error_paths():
    for args in [([1.0, 2.0], 0.0, 0.0, 3), ([1.0, 2.0], 0.0, 0.0, 0), ([1.0, -2.0], 0.0, 0.0, 1), ([1.0], -1.0, 0.0, 1),
                 ([float("nan")], 0.0, 0.0, 1)]:
        with pytest.raises(B.GPipeError):
            B.partition_min_variance(*args)


def test_bench_workload_partitions():
    """What `partition="cost"` does to the BASELINE.json workloads: the head shortens the last cell."""
    expect = {"T(6,4096,16)": [0, 4, 6], "T(24,16384,32)": [0, 3, 6, 9, 12, 15, 18, 21, 24]}
    for name, want in expect.items():
        w = gi.CONFIGS[name]
        spec, _keep = B.make_spec(w.n_layers, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len, w.dtype,
                                  list(w.causal), w.ln_eps)
        c, emb, head = B.layer_costs(spec, w.remat)
        assert B.partition_min_variance(c, emb, head, w.K) == want
    w = gi.CONFIGS["T(64,16384,32)"]
    spec, _keep = B.make_spec(w.n_layers, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len, w.dtype,
                              list(w.causal), w.ln_eps)
    c, emb, head = B.layer_costs(spec, True)
    b = B.partition_min_variance(c, emb, head, w.K)
    sizes = [b[k + 1] - b[k] for k in range(w.K)]
    assert sum(sizes) == 128 and sizes[-1] == 7 and max(sizes) == 9       # head = 1.5 layers: 7 layers + head
    eq = list(range(0, 129, 8))
    assert op.variance(op.cell_costs(c, b, emb, head)) < 0.5 * op.variance(op.cell_costs(c, eq, emb, head))


def test_encdec_cost_model_and_partition():
    """f2 on the f4 model: the library's encoder-decoder cost model equals the oracle's restatement of it; a decoder layer
    costs more than an encoder layer by the cross-attention block (checked against the parameter counts: its four
    projections hold 4 d d_a of the layer's weights), so the minimum-variance cut gives the decoder cells fewer layers."""
    from oracle import encdec_oracle as eo
    for (n_enc, n_dec, H, A) in [(6, 6, 8192, 16), (64, 64, 16384, 32), (2, 2, 256, 4)]:
        spec = B.EncDecSpec(n_enc, n_dec, 1024, H, A, 64, 64000, 256, 1, 1e-5, 0.0)
        for remat in (False, True):
            c, emb, head = B.layer_costs_encdec(spec, remat)
            rc, remb, rhead = op.layer_costs_encdec(n_enc, n_dec, 1024, H, A, 64, 64000, 256, remat)
            assert emb == remb and abs(head - rhead) <= 1e-9 * rhead and np.allclose(c, rc, rtol=1e-12, atol=0)
        # GEMM FLOPs per token and pass are 2 x the layer's matrix parameters: the cost difference between a decoder and an
        # encoder layer, attention aside, must be 2 x the cross-attention block's matrix parameters x (3 passes)
        c, _, _ = B.layer_costs_encdec(spec, False)
        s = eo.EncDecSpec(n_enc, n_dec, 1024, H, A, 64, 64000, 256)
        shapes = dict(eo.tensor_list(s))
        cross = sum(shapes["l%d.%s" % (n_enc, n)][0] * shapes["l%d.%s" % (n_enc, n)][1] for n in ("w_q", "w_kv", "w_o2"))
        da, S = A * 64, 256
        attn_enc = 4.0 * S * da
        attn_dec = 4.0 * S * da * (S + 1.0) / (2.0 * S) + 4.0 * S * da
        assert abs((c[n_enc] - c[0]) - (3.0 * 2.0 * cross + 3.5 * (attn_dec - attn_enc))) <= 1e-9 * c[0]
    spec = B.EncDecSpec(64, 64, 1024, 16384, 32, 64, 64000, 256, 1, 1e-5, 0.0)
    c, emb, head = B.layer_costs_encdec(spec, True)
    b = B.partition_min_variance(c, emb, head, 16)
    sizes = [b[k + 1] - b[k] for k in range(16)]
    assert sum(sizes) == 128 and max(sizes[:7]) >= max(sizes[9:]) and sizes[-1] < sizes[0]
    eq = [8 * k for k in range(17)]
    assert op.variance(op.cell_costs(c, b, emb, head)) < op.variance(op.cell_costs(c, eq, emb, head))

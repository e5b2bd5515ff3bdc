"""Pins for the encoder-decoder oracle (oracle/encdec_oracle.py), checked against something
other than the oracle itself: the paper's printed model sizes, an independent torch-autograd model written with
library routines, fp64 finite differences, the paper's consistency claims (M, K, partition, remat), the
visibility structure an encoder-decoder must have, and torch.clamp for the logit clip.
None of these tests touches the CUDA path."""
import math
import os

import numpy as np
import pytest
import torch
import torch.nn.functional as F

import gpipe_inputs as gi
from oracle import encdec_oracle as eo

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _spec(w):
    return eo.EncDecSpec(w.n_enc, w.n_dec, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len,
                         w.ln_eps, w.logit_clip)


def _tiny(L=1, **kw):
    """2L layers of the tiny config's widths: d 64, H 256, 4 heads of 16, vocab 512, S 16, N 8."""
    w = gi.encdec("tiny-encdec", L, 256, 4, vocab=512, n_seqs=8, M=4, K=2, d_model=64, d_head=16, seq_len=16,
                  dtype="fp32")
    return w.replace(**kw) if kw else w


def _run(w, K, M, remat, dtype=np.float64, params=None, cell_lo=None, seed_t=2001):
    o = eo.GPipeEncDecOracle(_spec(w), K, M, remat, dtype=dtype, cell_lo=cell_lo)
    o.set_params(params if params is not None else gi.make_params(w, 1001, round_bf16=False))
    src, tgt, lab = gi.make_tokens_encdec(w, seed_t)
    return o, o.step(src, tgt, lab), (src, tgt, lab)


def _maxrel(a, b):
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


# ---------------------------------------------------------------------------------------------
# P2': the printed model sizes, from THIS module's tensor list
# ---------------------------------------------------------------------------------------------
def test_section5_model_sizes_from_the_encdec_inventory():
    with open(os.path.join(GOLD, "paper_section5_model_sizes.txt")) as f:
        rows = [l.split() for l in f if l.strip() and not l.startswith("#")]
    for L, H, A, printed in rows:
        s = eo.EncDecSpec(int(L), int(L), 1024, int(H), int(A), 64, 64000, 256)
        assert abs(eo.param_count(s) / 1e9 - float(printed)) <= 0.1, (L, H, A, eo.param_count(s))
    n6 = eo.param_count(eo.EncDecSpec(64, 64, 1024, 16384, 32, 64, 64000, 256))
    assert abs(n6 / 1e9 - 6.04) < 0.01                                   # 6.04 B
    # teeth: a separate target embedding (3 V d) or a decoder without the cross-attention block misses the print
    assert abs((eo.param_count(eo.EncDecSpec(6, 6, 1024, 8192, 16, 64, 64000, 256)) + 64000 * 1024) / 1e9 - 0.4) > 0.05
    s24 = eo.EncDecSpec(24, 24, 1024, 8192, 16, 64, 64000, 256)
    cross = sum(r * c for n, (r, c) in eo.tensor_list(s24)
                if n.split(".")[-1] in ("w_q", "w_kv", "w_o2", "b_q", "b_kv", "b_o2", "lnx_g", "lnx_b"))
    assert abs((eo.param_count(s24) - cross) / 1e9 - 1.3) > 0.1


def test_inventory_matches_the_shared_naming_convention():
    w = _tiny(2)
    assert eo.tensor_list(_spec(w)) == gi.tensor_shapes(w)


# ---------------------------------------------------------------------------------------------
# Whole-model pin: an independent torch-autograd encoder-decoder (library routines, no cells)
# ---------------------------------------------------------------------------------------------
class _RoundThrough(torch.autograd.Function):
    """Identity whose forward value and / or incoming gradient is stored in bf16 (torch's own RNE conversion)."""

    @staticmethod
    def forward(ctx, x, fwd, bwd):
        ctx.bwd = bwd
        return x.to(torch.bfloat16).to(x.dtype) if fwd else x

    @staticmethod
    def backward(ctx, g):
        return (g.to(torch.bfloat16).to(g.dtype) if ctx.bwd else g), None, None


def _torch_encdec_grads(w, params, src, tgt, lab, per_token=False, rounded=False):
    """rounded=True: the tensors the bf16 CUDA path stores in bf16 are rounded straight-through
    (forward value and / or gradient), with a hand-written attention so that P and dS can be rounded too."""
    def rt(x, fwd, bwd):
        return _RoundThrough.apply(x, fwd, bwd) if rounded else x
    P = {n: torch.tensor(np.asarray(a, np.float64), requires_grad=True) for n, a in params.items()}
    d, A, dh, S = w.d_model, w.n_heads, w.d_head, w.seq_len
    pos = torch.arange(S, dtype=torch.float64)[:, None]
    i2 = (torch.arange(d) // 2 * 2).to(torch.float64)[None, :]
    ang = pos / torch.pow(torch.tensor(10000.0, dtype=torch.float64), i2 / d)
    pe = torch.where(torch.arange(d)[None, :] % 2 == 0, torch.sin(ang), torch.cos(ang)).to(torch.float32).to(torch.float64)
    N = src.shape[0]

    def heads(t):
        return t.reshape(N, S, A, dh).transpose(1, 2)

    def mha(q, k, v, causal):
        if not rounded:    # the library's fused attention (math backend in fp64): scale 1/sqrt(dh) is its default
            o = F.scaled_dot_product_attention(heads(q), heads(k), heads(v), is_causal=causal)
        else:
            s = rt(heads(q) @ heads(k).transpose(-1, -2) * (1.0 / math.sqrt(dh)), False, True)      # dS is an MMA operand
            if causal:
                s = s.masked_fill(torch.triu(torch.ones(S, S, dtype=torch.bool), 1), float("-inf"))
            o = rt(torch.softmax(s, -1), True, False) @ heads(v)                                    # P is an MMA operand
        return rt(o.transpose(1, 2).reshape(N, S, A * dh), True, True)

    def ln(x, gname, bname):
        return rt(F.layer_norm(x, (d,), P[gname][0], P[bname][0], w.ln_eps), True, True)

    def lin(x, l, wn, bn, fwd=True):      # a linear layer whose output (fwd) and output gradient are stored in bf16
        return rt(F.linear(x, P[f"l{l}.{wn}"].T, P[f"l{l}.{bn}"][0]), fwd, True)

    def ffn(x, l):
        c = ln(x, f"l{l}.ln2_g", f"l{l}.ln2_b")
        h = rt(torch.relu(lin(c, l, "w_1", "b_1", fwd=False)), True, False)
        return x + lin(h, l, "w_2", "b_2", fwd=False)      # fp32 residual stream; bf16 operand copy of its gradient

    xs = P["emb"][torch.tensor(src, dtype=torch.long)] + pe[None]
    for l in range(w.n_enc):
        q, k, v = lin(ln(xs, f"l{l}.ln1_g", f"l{l}.ln1_b"), l, "w_qkv", "b_qkv").split(A * dh, dim=-1)
        xs = ffn(xs + lin(mha(q, k, v, False), l, "w_o", "b_o", fwd=False), l)
    mem = ln(xs, "lne_g", "lne_b")         # its gradient is summed in fp32 over the decoder layers, then stored in bf16
    x = P["emb"][torch.tensor(tgt, dtype=torch.long)] + pe[None]
    for l in range(w.n_enc, w.n_layers):
        q, k, v = lin(ln(x, f"l{l}.ln1_g", f"l{l}.ln1_b"), l, "w_qkv", "b_qkv").split(A * dh, dim=-1)
        x = x + lin(mha(q, k, v, True), l, "w_o", "b_o", fwd=False)
        cx = ln(x, f"l{l}.lnx_g", f"l{l}.lnx_b")
        k2, v2 = lin(mem, l, "w_kv", "b_kv").split(A * dh, dim=-1)
        x = x + lin(mha(lin(cx, l, "w_q", "b_q"), k2, v2, False), l, "w_o2", "b_o2", fwd=False)
        x = ffn(x, l)
    y = ln(x, "lnf_g", "lnf_b")
    logits = rt(y @ P["w_out"], True, True)
    if w.logit_clip > 0:
        logits = torch.clamp(logits, -w.logit_clip, w.logit_clip)
    tl = torch.tensor(lab, dtype=torch.long).reshape(-1)
    if per_token:
        return F.cross_entropy(logits.reshape(-1, w.vocab), tl, reduction="none").detach().numpy()
    loss = F.cross_entropy(logits.reshape(-1, w.vocab), tl)
    loss.backward()
    return float(loss.detach()), {n: P[n].grad.numpy() for n in P}


@pytest.mark.parametrize("L,K,M,clip", [(1, 2, 4, 0.0), (2, 4, 2, 0.0), (2, 3, 4, 0.05), (1, 1, 1, 0.0)])
def test_whole_model_matches_torch_autograd(L, K, M, clip):
    w = _tiny(L, logit_clip=clip)
    params = gi.make_params(w, 1001, round_bf16=False)
    if clip:                                 # make the clamp bite: logits ~ N(0, 0.1^2)
        params["w_out"] = params["w_out"] * 5
    o, loss, (src, tgt, lab) = _run(w, K, M, True, params=params)
    tl, tg = _torch_encdec_grads(w, params, src, tgt, lab)
    assert abs(loss - tl) <= 1e-12 * abs(tl)
    for n in o.names:
        assert _maxrel(o.g[n], tg[n].reshape(o.g[n].shape)) <= 1e-10, n
    if clip:                                 # the clamp was active on a visible share of the logits
        dl = tg["w_out"]
        assert np.isfinite(dl).all()


def test_round_operands_mode_matches_independent_straight_through_model():
    """The oracle's round_operands mode (used only for the bf16 floor report, reading A14) against the torch model with
    torch's own bf16 conversion applied straight-through at the storage points DESIGN.md section 6 lists."""
    w = _tiny(1, d_model=128, n_heads=2, d_head=64, d_ffn=512, seq_len=32, n_seqs=4, M=2)
    params = gi.make_params(w, 1001, round_bf16=True)
    src, tgt, lab = gi.make_tokens_encdec(w, 2001)
    o = eo.GPipeEncDecOracle(_spec(w), 2, 2, True, round_operands=True)
    o.set_params(params)
    loss = o.step(src, tgt, lab)
    tl, tg = _torch_encdec_grads(w, params, src, tgt, lab, rounded=True)
    assert abs(loss - tl) <= 1e-12 * abs(tl)
    for n in o.names:
        assert _maxrel(o.g[n], tg[n].reshape(o.g[n].shape)) <= 1e-9, n
    pl, pg = _torch_encdec_grads(w, params, src, tgt, lab, rounded=False)
    assert max(_maxrel(o.g[n], pg[n].reshape(o.g[n].shape)) for n in o.names) > 1e-4


def test_logit_clip_is_a_clamp_with_the_clamp_derivative():
    """PAPER.md:174 (ii) / reading B5 against torch.clamp + autograd on the operator alone; c = 0 is the plain loss."""
    rng = np.random.Generator(np.random.PCG64(5))
    z = rng.standard_normal((12, 40)) * 2.0
    lab = rng.integers(0, 40, size=12)
    for c in (0.5, 1.5):
        zt = torch.tensor(z, requires_grad=True)
        lt = F.cross_entropy(torch.clamp(zt, -c, c), torch.tensor(lab), reduction="sum") / 24.0
        lt.backward()
        loss, dl, per = eo.softmax_ce_clipped(z.copy(), lab, 24, c)
        assert abs(loss - float(lt.detach())) < 1e-13
        assert np.abs(dl - zt.grad.numpy()).max() < 1e-15
        frac = float((np.abs(z) > c).mean())
        assert 0.1 < frac < 0.9 and np.all(dl[np.abs(z) > c] == 0)
    zt = torch.tensor(z, requires_grad=True)
    lt = F.cross_entropy(zt, torch.tensor(lab), reduction="sum") / 24.0
    loss, dl, per = eo.softmax_ce_clipped(z.copy(), lab, 24, 0.0)
    assert abs(loss - float(lt.detach())) < 1e-13 and abs(per.sum() / 24.0 - loss) < 1e-13
    # a huge bound changes nothing
    loss2, dl2, _ = eo.softmax_ce_clipped(z.copy(), lab, 24, 1e9)
    assert loss2 == loss and np.array_equal(dl, dl2)


# ---------------------------------------------------------------------------------------------
# The paper's consistency claims on this model
# ---------------------------------------------------------------------------------------------
def test_gradients_independent_of_K_M_and_the_partition():
    w = _tiny(2)
    params = gi.make_params(w, 1001, round_bf16=False)
    base, lb, _ = _run(w, 1, 1, False, params=params)
    for K, M, remat, cell_lo in [(2, 4, True, None), (4, 8, True, None), (3, 2, False, None),
                                 (2, 4, True, [0, 1, 4]), (2, 2, True, [0, 3, 4]), (3, 4, True, [0, 2, 3, 4])]:
        o, l, _ = _run(w, K, M, remat, params=params, cell_lo=cell_lo)
        assert abs(l - lb) <= 1e-12 * abs(lb)
        for n in o.names:
            assert _maxrel(o.g[n], base.g[n]) <= 1e-11, (K, M, cell_lo, n)
    # fp32, the bar BASELINE.json states: 1e-5 relative
    b32, l32, _ = _run(w, 1, 1, False, dtype=np.float32, params=params)
    o32, l2, _ = _run(w, 4, 4, True, dtype=np.float32, params=params)
    for n in o32.names:
        assert _maxrel(o32.g[n].astype(np.float64), b32.g[n].astype(np.float64)) <= 1e-5, n


def test_remat_equals_stored_bitwise_and_trace():
    w = _tiny(2)
    a, la, _ = _run(w, 4, 4, True)
    b, lb, _ = _run(w, 4, 4, False)
    assert la == lb
    for n in a.names:
        assert np.array_equal(a.g[n], b.g[n]), n
    assert [t for t in a.trace if t[0] != "R"] == b.trace
    assert sum(1 for t in a.trace if t[0] == "R") == 16


def test_finite_differences_double():
    w = _tiny(1, n_seqs=2, M=1, K=2)
    params = gi.make_params(w, 1001, round_bf16=False)
    o, loss, (src, tgt, lab) = _run(w, 2, 1, True, params=params)
    rng = np.random.Generator(np.random.PCG64(7))
    h = 1e-6
    for n in o.names:
        gmax = np.abs(o.g[n]).max()
        flat = o.p[n].reshape(-1)
        # embedding rows that no token uses have zero gradient: probe used rows too
        idx = list(rng.integers(0, flat.size, size=4))
        if n == "emb":
            idx += [int(src[0, 0]) * w.d_model + 3, int(tgt[1, 2]) * w.d_model + 5]
        for i in idx:
            old = flat[i]
            flat[i] = old + h
            lp = o.loss_only(src, tgt, lab)
            flat[i] = old - h
            lm = o.loss_only(src, tgt, lab)
            flat[i] = old
            fd = (lp - lm) / (2 * h)
            assert abs(fd - o.g[n].reshape(-1)[i]) <= 1e-5 * max(gmax, 1e-12) + 1e-9, (n, i, fd, o.g[n].reshape(-1)[i])


# ---------------------------------------------------------------------------------------------
# Structure an encoder-decoder must have: who can see what
# ---------------------------------------------------------------------------------------------
def test_decoder_is_causal_in_the_target_and_sees_the_whole_source():
    w = _tiny(1, n_seqs=4, M=2, K=2)
    params = gi.make_params(w, 1001, round_bf16=False)
    src, tgt, lab = gi.make_tokens_encdec(w, 2001)
    S = w.seq_len

    def per_token(s_, t_):
        o = eo.GPipeEncDecOracle(_spec(w), 2, 2, True)
        o.set_params(params)
        o.step(s_, t_, lab)
        return np.concatenate([o.per_token_loss[m] for m in range(2)]).reshape(w.n_seqs, S)
    base = per_token(src, tgt)
    # independent statement of the same per-token losses
    assert np.abs(base.reshape(-1) - _torch_encdec_grads(w, params, src, tgt, lab, per_token=True)).max() < 1e-12
    # (1) change the target token at position j of sequence 1: losses at positions < j and all other sequences unchanged
    j = 9
    t2 = tgt.copy()
    t2[1, j] = (t2[1, j] + 1) % w.vocab
    d1 = per_token(src, t2) - base
    assert np.all(d1[1, :j] == 0) and np.all(d1[[0, 2, 3]] == 0)
    assert np.all(np.abs(d1[1, j:]) > 0)
    # (2) change the LAST source token of sequence 2: every target position of that sequence moves (cross-attention is
    #     not masked and the encoder is bidirectional), nothing else does
    s2 = src.copy()
    s2[2, S - 1] = (s2[2, S - 1] + 1) % w.vocab
    d2 = per_token(s2, tgt) - base
    assert np.all(np.abs(d2[2]) > 0) and np.all(d2[[0, 1, 3]] == 0)


def test_memory_gradient_sums_over_decoder_layers():
    """dE gets contributions from both id sequences, and the memory's gradient is the sum over ALL decoder layers:
    zeroing one decoder layer's w_kv and b_kv removes exactly its contribution (its keys / values become constant 0,
    its attention uniform over zero values), which the torch model confirms."""
    w = _tiny(2)
    params = gi.make_params(w, 1001, round_bf16=False)
    params["l3.w_kv"] = np.zeros_like(params["l3.w_kv"])
    params["l3.b_kv"] = np.zeros_like(params["l3.b_kv"])
    o, loss, (src, tgt, lab) = _run(w, 2, 2, True, params=params)
    tl, tg = _torch_encdec_grads(w, params, src, tgt, lab)
    for n in o.names:
        assert _maxrel(o.g[n], tg[n].reshape(o.g[n].shape)) <= 1e-10, n
    assert np.abs(o.g["l3.w_q"]).max() == 0          # uniform attention over zero values: the queries get no gradient


def test_k1_m1_stored_is_plain_backprop_trace_and_errors():
    o, _, _ = _run(_tiny(1), 1, 1, False)
    assert o.trace == [("F", 0, 0), ("B", 0, 0)]
    w = _tiny(1)
    with pytest.raises(ValueError):
        eo.EncDecSpec(0, 2, 64, 256, 4, 16, 512, 16)
    o = eo.GPipeEncDecOracle(_spec(w), 2, 3, True)
    src, tgt, lab = gi.make_tokens_encdec(w, 1)
    with pytest.raises(ValueError):
        o.step(src, tgt, lab)                         # 8 sequences do not split into 3 equal micro-batches


def test_depth_scaled_ffn_init_recipe():
    """PAPER.md:174 (i): FFN matrices drawn with std / (number of layers); everything else unchanged."""
    w = _tiny(2)
    a = gi.make_params(w, 1001, round_bf16=False)
    b = gi.make_params(w, 1001, round_bf16=False, ffn_depth_scale=True)
    for n in a:
        base = n.split(".")[-1]
        if base in ("w_1", "w_2"):
            assert abs(b[n].std() / (0.02 / w.n_layers) - 1) < 0.05 and abs(a[n].std() / 0.02 - 1) < 0.05
        else:
            assert np.array_equal(a[n], b[n])

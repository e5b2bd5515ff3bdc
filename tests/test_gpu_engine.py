"""End-to-end parity of the CUDA path (through the C ABI) against the CPU oracle, fp32 and bf16,
plus the structural properties of the schedule, the tracker and the error paths.

Tolerances (BASELINE.json north_star): fp32 - loss and per-tensor max-relative gradient error
<= 1e-4 (TF32 off); bf16 - loss within 1e-2 relative, per-tensor gradient cosine >= 0.999.
"""
import numpy as np
import pytest

import gpipe_inputs as gi
import paper_1811_06965_b200 as gp
from oracle import schedule as sch
from tests.util import cosine, engine_program, maxrel, run_oracle

pytestmark = pytest.mark.gpu

FP32_TOL = 1e-4


def _engine(w, **kw):
    return gp.from_workload(w, **kw)


def _tiny(causal=(1, 1), **kw):
    return gi.CONFIGS["tiny"].replace(causal=tuple(causal), **kw)


def _compare_fp32(w, K, M, remat, seed_p=1001, seed_t=2001):
    params = gi.make_params(w, seed_p, round_bf16=False)
    tok, lab = gi.make_tokens(w, seed_t)
    o, loss_ref = run_oracle(w, params, tok, lab, K=K, M=M, remat=remat)
    with _engine(w, K=K, M=M, remat=remat) as e:
        e.set_params(params)
        loss = e.step(tok, lab)
        assert abs(loss - loss_ref) <= FP32_TOL * abs(loss_ref), (loss, loss_ref)
        worst = 0.0
        for n in e.names:
            err = maxrel(e.get_grad(n), o.g[n])
            worst = max(worst, err)
            assert err <= FP32_TOL, (n, err)
    return worst


@pytest.mark.parametrize("causal", [(1, 1), (0, 1), (0, 0)])
def test_config1_tiny_fp32_parity(causal):
    """BASELINE.json configs[0]: 2 layers, d 64, FFN 256, 4 heads, vocab 512, seq 16, N 8, M 4, K 2."""
    _compare_fp32(_tiny(causal), 2, 4, True)


@pytest.mark.parametrize("K,M,remat", [(1, 1, False), (1, 8, True), (2, 1, True), (2, 2, False),
                                         (2, 8, True), (2, 4, False)])
def test_fp32_parity_over_K_M_remat(K, M, remat):
    _compare_fp32(_tiny((0, 1)), K, M, remat)


def test_fp32_parity_uneven_cells_and_ragged_shapes():
    """L % K != 0 (first cells get the extra layer), S not a multiple of 32, d_head 32."""
    w = gi.CONFIGS["tiny"].replace(n_layers=5, causal=(0, 1, 0, 1, 1), d_model=96, n_heads=3, d_head=32,
                                   d_ffn=200, vocab=1000, seq_len=40, n_seqs=6, M=3, K=3)
    _compare_fp32(w, 3, 3, True)
    _compare_fp32(w, 2, 2, False)


def test_zero_layer_model():
    w = gi.CONFIGS["tiny"].replace(n_layers=0, causal=(), K=1, M=2)
    _compare_fp32(w, 1, 2, True)


def test_gradients_independent_of_K_M_remat_on_gpu():
    """PAPER.md:45/:67/:209 on the GPU itself: the accumulated gradient does not depend on K, M or remat (only the
    fp32 summation order of the per-micro-batch terms differs between M values, hence 1e-5 and not bitwise)."""
    w = _tiny((0, 1))
    params = gi.make_params(w, 1001, round_bf16=False)
    tok, lab = gi.make_tokens(w, 2001)
    ref = None
    for K, M, remat in [(1, 1, False), (2, 4, True), (2, 8, False), (1, 2, True)]:
        with _engine(w, K=K, M=M, remat=remat) as e:
            e.set_params(params)
            loss = e.step(tok, lab)
            g = e.grads()
        if ref is None:
            ref = (loss, g)
            continue
        assert abs(loss - ref[0]) <= 1e-6 * abs(ref[0])
        for n in g:
            assert maxrel(g[n], ref[1][n]) <= 1e-5, (K, M, remat, n)


def test_remat_equals_stored_bitwise_on_gpu():
    """replayed activations are bit-identical, so every gradient that is summed in
    a fixed order is bit-identical - which is every gradient (the embedding scatter-add has a fixed order too)."""
    w = _tiny((0, 1))
    params = gi.make_params(w, 1001, round_bf16=False)
    tok, lab = gi.make_tokens(w, 2001)
    out = []
    for remat in (True, False):
        with _engine(w, remat=remat) as e:
            e.set_params(params)
            out.append((e.step(tok, lab), e.grads()))
    assert out[0][0] == out[1][0]
    for n in out[0][1]:
        assert np.array_equal(out[0][1][n], out[1][1][n]), n


def test_step_accumulates_and_sgd_applies():
    w = _tiny()
    params = gi.make_params(w, 1001, round_bf16=False)
    tok, lab = gi.make_tokens(w, 2001)
    with _engine(w) as e:
        e.set_params(params)
        l0 = e.step(tok, lab)
        g1 = e.grads()
        e.step(tok, lab)
        g2 = e.grads()
        for n in g1:
            assert maxrel(g2[n], 2 * g1[n]) <= 1e-6, n
        e.zero_grads()
        assert not any(e.get_grad(n).any() for n in e.names)
        e.step(tok, lab)
        g = e.grads()
        before = {n: e.get_param(n) for n in e.names}
        e.apply_sgd(0.5)
        for n in e.names:
            assert np.array_equal(e.get_param(n), before[n] - np.float32(0.5) * g[n]), n
            assert not e.get_grad(n).any()
        assert e.step(tok, lab) < l0
        # the oracle agrees on the updated parameters and the second loss
        o, _ = run_oracle(w, params, tok, lab, dtype=np.float32)
        o.apply_sgd(0.5)
        for n in e.names:
            assert maxrel(e.get_param(n), o.p[n]) <= 1e-5, n


@pytest.mark.parametrize("which", ["tiny-fp32", "small-bf16"])
def test_cuda_graph_replay_is_bitwise_eager(which):
    """The step as one CUDA graph (capture on the second step, replay afterwards) against eager enqueue of the same
    K-stream DAG: same kernels, same dependencies, so loss and every accumulated gradient are bit-identical, on
    different batches (the ids are copied outside the graph), and the launch count is the same."""
    w = _tiny((0, 1)) if which == "tiny-fp32" else _bf16_small()
    params = gi.make_params(w, 1001)
    batches = [gi.make_tokens(w, 2200 + i) for i in range(4)]
    out = {}
    for graph in (True, False):
        with _engine(w) as e:
            e.cuda_graph(graph)
            e.set_params(params)
            losses = [e.step(*b) for b in batches]
            out[graph] = (losses, e.grads(), e.launch_count(), e.cuda_graph_state())
            e.apply_sgd(0.1)                                     # the graph survives parameter updates (same pointers)
            out[graph] += (e.step(*batches[0]),)
    assert out[True][3] == 2 and out[False][3] == 0
    assert out[True][0] == out[False][0] and out[True][4] == out[False][4]
    assert out[True][2] == out[False][2] > 0
    for n in out[True][1]:
        assert np.array_equal(out[True][1][n], out[False][1][n]), n


def test_device_resident_inputs_match_host_inputs():
    import torch
    w = _tiny()
    params = gi.make_params(w, 1001, round_bf16=False)
    tok, lab = gi.make_tokens(w, 2001)
    with _engine(w) as e:
        e.set_params(params)
        l_host = e.step(tok, lab)
        g_host = e.grads()
        e.zero_grads()
        l_dev = e.step(torch.tensor(tok, device="cuda"), torch.tensor(lab, device="cuda"))
        assert l_dev == l_host
        for n in e.names:
            if n != "emb":
                assert np.array_equal(e.get_grad(n), g_host[n])
        bad = torch.tensor(tok, device="cuda").clone()
        bad[0, 0] = w.vocab
        with pytest.raises(gp.GPipeError):
            e.step(bad, torch.tensor(lab, device="cuda"))


def test_error_paths():
    w = _tiny()
    tok, lab = gi.make_tokens(w, 2001)
    with _engine(w) as e:
        bad = tok.copy()
        bad[1, 2] = -1
        with pytest.raises(gp.GPipeError) as err:
            e.step(bad, lab)
        assert err.value.code == -1
        with pytest.raises(ValueError):
            e.step(tok[:4], lab[:4])
    with pytest.raises(gp.GPipeError):
        _engine(w, K=3)
    with pytest.raises(gp.GPipeError):
        _engine(w, M=3)


def test_trace_is_a_valid_gpipe_schedule():
    """Every task of Fig. 2c appears once; per-cell program order and cross-cell dependencies
    hold in device time; with M = 1 at most one cell is busy."""
    w = _tiny()
    params = gi.make_params(w, 1001, round_bf16=False)
    tok, lab = gi.make_tokens(w, 2001)
    for K, M, remat in [(2, 4, True), (2, 4, False), (2, 1, True)]:
        with _engine(w, K=K, M=M, remat=remat) as e:
            e.set_params(params)
            e.trace(True)
            e.step(tok, lab)
            ev = e.trace_events()
        tasks = {(kind, k, m): (s, t, idx) for kind, k, m, idx, s, t in ev}
        want = set()
        for k in range(K):
            want |= set(engine_program(k, K, M, remat))     # Fig. 2c minus the elided tasks (readings A15b, A15c)
        assert set(tasks) == want and len(ev) == len(want)
        for (kind, k, m), (s, t, idx) in tasks.items():
            assert t >= s
            for dep in sch.dependencies((kind, k, m), K, remat, early=True):
                assert tasks[dep][1] <= s + 1e-3, ((kind, k, m), dep)
            if kind == "R" and k == K - 1 and k > 0:        # the replay that stands in for the elided F(K-1, m)
                assert tasks[("F", k - 1, m)][1] <= s + 1e-3
        for k in range(K):
            prog = sorted([(v[2], key) for key, v in tasks.items() if key[1] == k])
            assert [key for _, key in prog] == engine_program(k, K, M, remat)
            times = [tasks[key] for _, key in prog]
            for a, b in zip(times, times[1:]):
                assert a[1] <= b[0] + 1e-3                  # a stream is an in-order queue
        if M == 1:
            # F and B tasks never overlap; the replay R(k,0) is allowed to (early scheduling, :89)
            spans = sorted((s, t) for (kind, _, _), (s, t, _) in tasks.items() if kind != "R")
            for a, b in zip(spans, spans[1:]):
                assert a[1] <= b[0] + 1e-3


def test_peak_bytes_tracker():
    w = _tiny(n_seqs=8)
    peaks = {}
    for M in (1, 2, 4, 8):
        with _engine(w, M=M, remat=True) as e:
            p = e.peak_bytes()
            assert p["total"] == sum(p["by_category"].values())
            assert p["total"] <= e.arena.numel()
            peaks[M] = p["by_category"]["interior"]
    assert peaks[1] > peaks[2] > peaks[4] > peaks[8]
    with _engine(w, M=8, remat=False) as e:
        assert e.peak_bytes()["by_category"]["interior"] > 4 * peaks[8]


def test_host_plan_equals_device_plan_and_allocator_view():
    """gpipe_plan_bytes (host only, no device query) is exactly what gpipe_create carves on the device
    (gpipe_peak_bytes total), for fp32 and bf16 plans with and without a split-K workspace; and the arena torch
    allocated for it shows up in torch.cuda.memory_allocated / cudaMemGetInfo (SURVEY.md 8(d) cross-check)."""
    import torch
    for w in (_tiny(), _bf16_small(), _bf16_small().replace(K=1, M=2), gi.reduced(gi.CONFIGS["T(12,8192,16)"])):
        spec, keep = gp.make_spec(w.n_layers, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len, w.dtype,
                                  list(w.causal))
        plan = gp.plan_bytes(spec, w.K, w.M, w.remat, w.n_seqs)
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        alloc0 = torch.cuda.memory_allocated()
        with _engine(w) as e:
            assert e.peak_bytes()["total"] == plan
            assert torch.cuda.memory_allocated() - alloc0 >= plan
            assert torch.cuda.max_memory_allocated() >= plan
            free1, _ = torch.cuda.mem_get_info()
            # the caching allocator may serve the arena from memory it already holds: the device-level
            # free memory never drops by more than the arena (+ allocator rounding)
            assert free0 - free1 <= plan + (64 << 20)


def test_checkpoint_restore_is_bitwise():
    """gpipe_get_master / gpipe_set_master / optimizer-slot access (no rounding): three RMSProp mini-batches
    uninterrupted == one mini-batch, save, restore into a NEW handle, two more - bit for bit, in bf16 mode where
    get_param / set_param alone would lose the fp32 master bits and the optimizer state."""
    w = _bf16_small()
    params = gi.make_params(w, 1002)
    batches = [gi.make_tokens(w, 2100 + i) for i in range(3)]

    def run(e, its):
        losses = []
        for it in its:
            losses.append(e.step(*batches[it]))
            e.apply_rmsprop(0.002, 0.9, 1e-6)
        return losses

    with _engine(w) as e:
        e.set_params(params)
        ref_losses = run(e, range(3))
        ref_state = e.state_dict()
    with _engine(w) as e:
        e.set_params(params)
        l0 = run(e, [0])
        saved = e.state_dict()
        assert any((saved["master"][n] != e.get_param(n)).any() for n in e.names)    # masters carry more than bf16
    with _engine(w) as e2:
        e2.load_state_dict(saved)
        l12 = run(e2, [1, 2])
        got = e2.state_dict()
    assert l0 + l12 == ref_losses
    for kind in ("master", "slot"):
        for n in ref_state[kind]:
            assert np.array_equal(got[kind][n], ref_state[kind][n]), (kind, n)


def test_device_init_params_statistics():
    w = gi.CONFIGS["tiny"].replace(d_model=256, d_ffn=1024, n_heads=4, d_head=64, vocab=4096)
    with _engine(w) as e:
        e.init_params(seed=7, std=0.02, parity=False)
        wq = e.get_param("l0.w_qkv")
        assert abs(wq.std() - 0.02) < 5e-4 and abs(wq.mean()) < 2e-4
        assert np.array_equal(e.get_param("l0.ln1_g"), np.ones((1, 256), np.float32))
        assert not e.get_param("l0.b_1").any()
        emb = e.get_param("emb")
        assert abs(np.corrcoef(emb[0], emb[1])[0, 1]) < 0.2
        e.init_params(seed=7, std=0.02, parity=True)
        assert abs(e.get_param("l1.ln2_g").mean() - 1.0) < 5e-3
        assert abs(e.get_param("l1.b_1").std() - 0.02) < 2e-3
        tok, lab = gi.make_tokens(w, 5)
        loss = e.step(tok, lab)
        assert abs(loss - (np.log(w.vocab) + 0.5 * 0.02 ** 2 * w.d_model)) < 0.05   # P7 closed form


# -------------------------------------------------------------------------------------------------
# bf16
# -------------------------------------------------------------------------------------------------
def _bf16_small():
    # a scaled-down T(L,H,A): same structure as configs[1], sized for the oracle (seconds)
    return gi.CONFIGS["T(6,4096,16)"].replace(name="bf16-small", n_layers=2, d_model=256, d_ffn=1024, n_heads=4,
                                              d_head=64, vocab=2048, seq_len=64, n_seqs=8, M=4, K=2,
                                              causal=(0, 1))


def test_bf16_end_to_end_parity_small():
    w = _bf16_small()
    params = gi.make_params(w, 1002)                        # bf16-representable (A12)
    tok, lab = gi.make_tokens(w, 2002)
    o, loss_ref = run_oracle(w, params, tok, lab)
    with _engine(w) as e:
        e.set_params(params)
        for n in e.names:                                   # both sides start from identical values
            assert np.array_equal(e.get_param(n), params[n]), n
        loss = e.step(tok, lab)
        assert abs(loss - loss_ref) <= 1e-2 * abs(loss_ref)
        cos = {n: cosine(e.get_grad(n), o.g[n]) for n in e.names}
    assert min(cos.values()) >= 0.999, sorted(cos.items(), key=lambda kv: kv[1])[:5]


def test_bf16_invariance_over_M_and_remat():
    """Per-token forward values do not depend on the micro-batch split (deterministic K-loop
    order), so gradients agree to fp32 summation-order level across (K, M, remat)."""
    w = _bf16_small()
    params = gi.make_params(w, 1002)
    tok, lab = gi.make_tokens(w, 2002)
    ref = None
    for K, M, remat in [(2, 4, True), (2, 4, False), (1, 2, True), (2, 8, True)]:
        with _engine(w, K=K, M=M, remat=remat) as e:
            e.set_params(params)
            loss = e.step(tok, lab)
            g = e.grads()
        if ref is None:
            ref = (loss, g)
            continue
        assert abs(loss - ref[0]) <= 1e-5 * abs(ref[0])
        for n in g:
            assert maxrel(g[n], ref[1][n]) <= 2e-3, (K, M, remat, n, maxrel(g[n], ref[1][n]))


# -------------------------------------------------------------------------------------------------
# full-size workloads, in the launch configuration bench.py times: properties that hold at any size
# (the oracle cannot run 6 B parameters; its per-kernel and reduced-shape parity is above)
# -------------------------------------------------------------------------------------------------
def test_full_size_config5_properties():
    """T(64,16384,32), K 16, M 16, remat on - the bench workload.  (i) loss at initialisation equals the closed
    form P7 (ln V + sigma^2 d / 2: the logits of an untied N(0, sigma^2) head over a LayerNorm output are
    N(0, sigma^2 d)); (ii) the step is deterministic and gpipe_step ACCUMULATES: a second step on the same
    batch reproduces the loss bitwise and doubles every sampled gradient (to fp32 running-sum rounding); (iii) rows of dW_out sum to
    ~0 over the vocabulary (softmax - onehot sums to zero per token: P8); (iv) peak HBM within 180 GB."""
    w = gi.CONFIGS["T(64,16384,32)"]
    tok, lab = gi.make_tokens(w, 2004)
    sample = ["l0.w_qkv", "l63.b_1", "l64.w_o", "l127.ln2_g", "l127.b_2", "lnf_g"]
    with _engine(w) as e:
        e.init_params(seed=1004, std=0.02, parity=False)
        assert e.peak_bytes()["total"] <= 180e9
        loss1 = e.step(tok, lab)
        assert abs(loss1 - (np.log(w.vocab) + 0.5 * 0.02 ** 2 * w.d_model)) < 0.05
        g1 = {n: e.get_grad(n).copy() for n in sample}
        gw = e.get_grad("w_out")
        assert np.isfinite(gw).all() and np.abs(gw).max() > 0
        # dlogits is stored in bf16 (2^-9 relative per entry), so the row sums cancel to that level
        assert np.abs(gw.sum(axis=1)).max() <= 2 ** -7 * np.abs(gw).sum(axis=1).max()
        loss2 = e.step(tok, lab)
        assert loss2 == loss1
        for n in sample:
            g2 = e.get_grad(n)
            assert np.isfinite(g2).all() and np.abs(g2).max() > 0, n
            assert maxrel(g2, 2.0 * g1[n]) <= 1e-5, n          # same 16 addends again, fp32 running sum


def test_full_size_config4_invariant_to_M():
    """T(24,16384,32), K 8: M = 32 (T_mb 2048, the nominal split) against M = 16 (T_mb 4096) on the same batch
    and device-drawn parameters - PAPER.md:67: the accumulated gradient is the mini-batch gradient whatever M
    is.  Per-token forward values are bitwise independent of the split, so only the fp32 summation order of
    the gradient sums differs."""
    w = gi.CONFIGS["T(24,16384,32)"]
    tok, lab = gi.make_tokens(w, 2003)
    sample = ["l0.w_1", "l0.b_qkv", "l11.w_o", "l23.w_2", "l23.ln1_b", "lnf_b"]
    res = []
    for M in (32, 16):
        with _engine(w, M=M) as e:
            e.init_params(seed=1003, std=0.02, parity=True)
            loss = e.step(tok, lab)
            res.append((loss, {n: e.get_grad(n).copy() for n in sample}))
    assert abs(res[0][0] - res[1][0]) <= 1e-5 * abs(res[0][0])
    for n in sample:
        assert maxrel(res[0][1][n], res[1][1][n]) <= 2e-3, (n, maxrel(res[0][1][n], res[1][1][n]))
        assert cosine(res[0][1][n], res[1][1][n]) >= 0.99999, n


# -------------------------------------------------------------------------------------------------
# cell partitioning
# -------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cell_lo", [[0, 1, 4, 5], [0, 3, 4, 5], [0, 2, 3, 5]])
def test_fp32_parity_explicit_partition(cell_lo):
    w = _tiny().replace(n_layers=5, causal=(1, 0, 1, 0, 1), K=3)
    params = gi.make_params(w, 1001, round_bf16=False)
    tok, lab = gi.make_tokens(w, 2001)
    o, loss_ref = run_oracle(w, params, tok, lab, cell_lo=cell_lo)
    with _engine(w, partition=cell_lo) as e:
        assert e.cells == [(cell_lo[k], cell_lo[k + 1]) for k in range(3)]
        e.set_params(params)
        loss = e.step(tok, lab)
        assert abs(loss - loss_ref) <= FP32_TOL * abs(loss_ref)
        for n in e.names:
            assert maxrel(e.get_grad(n), o.g[n]) <= FP32_TOL, n
        e.trace(True)
        e.zero_grads()
        e.step(tok, lab)
        ev = e.trace_events()
    assert sorted({k for (_, k, _, _, _, _) in ev}) == [0, 1, 2]


def test_bf16_cost_partition_changes_nothing_but_the_cut():
    """partition="cost": the head's cost shortens the last cell; per-token values do not depend on where the
    cuts are, so loss and every gradient (the embedding's too: its scatter-add has a fixed order) are bitwise
    those of the equal split."""
    w = gi.CONFIGS["T(6,4096,16)"].replace(name="bf16-part", n_layers=6, d_model=256, d_ffn=512, n_heads=4, d_head=64,
                                           vocab=4096, seq_len=64, n_seqs=8, M=4, K=2, causal=(0, 1, 0, 1, 0, 1))
    params = gi.make_params(w, 1005)
    tok, lab = gi.make_tokens(w, 2005)
    out = []
    for part in (None, "cost", [0, 1, 6]):
        with _engine(w, partition=part) as e:
            e.set_params(params)
            out.append((e.cells, e.step(tok, lab), e.grads(), e.peak_bytes()["total"]))
    assert out[0][0] == [(0, 3), (3, 6)]
    assert out[1][0][1][1] - out[1][0][1][0] < 3                      # the head costs more than a layer here
    for cells, loss, g, peak in out[1:]:
        assert loss == out[0][1] and peak == out[0][3]
        for n in g:
            assert np.array_equal(g[n], out[0][2][n]), (cells, n)


def test_partition_error_paths():
    w = _tiny().replace(n_layers=4, causal=(1, 1, 1, 1), K=2)
    for bad in ([0, 0, 4], [0, 4, 4], [1, 2, 4], [0, 2, 5], [0, 3, 2]):
        with pytest.raises(gp.GPipeError):
            _engine(w, partition=bad)


def test_rmsprop_training_steps_match_oracle():
    """SURVEY.md 8(f) f3 / PAPER.md:71: three mini-batches of step + gpipe_apply_rmsprop against the oracle.
    Tolerance 2e-4, twice the single-step fp32 bound (reading A20): from the second mini-batch on the two
    sides start from parameters that already differ by their fp32 rounding, and the RMSProp quotient g / (sqrt(ms) + eps)
    with ms ~ (1 - rho) g^2 turns a relative gradient error delta into ~ 3 delta of the update."""
    w = _tiny((0, 1))
    params = gi.make_params(w, 1001, round_bf16=False)
    o = None
    with _engine(w) as e:
        e.set_params(params)
        with pytest.raises(gp.GPipeError):
            gp.binding._check(gp.lib().gpipe_apply_rmsprop(e._h, 0.01, 0.9, 1e-6))      # no slots attached yet
        for it in range(3):
            tok, lab = gi.make_tokens(w, 2001 + it)
            if o is None:
                o, _ = run_oracle(w, params, tok, lab)      # builds the oracle (and runs one step we discard)
                o.zero_grads()
            loss_ref = o.step(tok, lab)
            loss = e.step(tok, lab)
            assert abs(loss - loss_ref) <= 2e-4 * abs(loss_ref), it
            o.apply_rmsprop(0.002, 0.9, 1e-6)
            e.apply_rmsprop(0.002, 0.9, 1e-6)
            for n in e.names:
                assert maxrel(e.get_param(n), o.p[n]) <= 2e-4, (it, n)
                assert not e.get_grad(n).any()
        with pytest.raises(gp.GPipeError):
            e.apply_rmsprop(0.01, 1.0, 1e-6)
        with pytest.raises(gp.GPipeError):
            e.apply_rmsprop(0.01, 0.9, 0.0)

"""Second stream per cell (gpipe_env.n_streams >= 2K, include/gpipe.h): the weight-gradient GEMMs of B(k, m) run beside
the cell's dgrad / LayerNorm / attention chain.  PAPER.md:67 fixes what a step computes (gradients of the M micro-batches
accumulated, applied once) and not how one cell's accelerator orders independent kernels, so the bar is the strictest
one: same kernels, same accumulation order => the loss and EVERY gradient bitwise equal to the one-stream-per-cell
handle, on the eager first step, on the captured step and on graph replays (a missed ordering edge between the two
streams shows up here as a mismatch)."""
import numpy as np
import pytest

import gpipe_inputs as gi
import paper_1811_06965_b200 as gp
from tests.util import maxrel, run_oracle

pytestmark = pytest.mark.gpu

SMALL = dict(d_model=256, d_ffn=1024, n_heads=4, d_head=64, vocab=2048, seq_len=64, n_seqs=8, M=4, K=2)


def _steps(w, params, ids, side, n_steps, **kw):
    out = []
    with gp.from_workload(w, side_streams=side, **kw) as e:
        assert e.side_streams == side
        e.set_params(params)
        for _ in range(n_steps):
            e.zero_grads()
            loss = e.step(*ids)
            out.append((loss, e.grads()))
        state = e.cuda_graph_state()
    return out, state


def _same(a, b):
    assert len(a) == len(b)
    for (la, ga), (lb, gb) in zip(a, b):
        assert la == lb
        for n in ga:
            assert np.array_equal(ga[n], gb[n]), n


@pytest.mark.parametrize("remat", [True, False])
def test_side_streams_fp32_bitwise_and_oracle(remat):
    w = gi.CONFIGS["tiny"].replace(n_layers=5, causal=(0, 1, 0, 1, 1), K=3, M=4, n_seqs=8)
    params = gi.make_params(w, 1001, round_bf16=False)
    ids = gi.make_tokens(w, 2001)
    o, loss_ref = run_oracle(w, params, *ids, remat=remat)
    on, st = _steps(w, params, ids, True, 4, remat=remat)
    off, _ = _steps(w, params, ids, False, 2, remat=remat)
    assert st == 2                                           # eager, capture, replay, replay
    _same(on, [off[0]] * 4)
    _same(off[:1], off[1:])
    assert abs(on[0][0] - loss_ref) <= 1e-4 * abs(loss_ref)
    for n, g in on[0][1].items():
        assert maxrel(g, o.g[n]) <= 1e-4, n


@pytest.mark.parametrize("K,M,L", [(2, 4, 4), (1, 2, 2), (4, 4, 4)])
def test_side_streams_bf16_bitwise(K, M, L):
    w = gi.CONFIGS["T(6,4096,16)"].replace(n_layers=L, causal=tuple(i & 1 for i in range(L)), **dict(SMALL, K=K, M=M))
    params = gi.make_params(w, 1001)
    ids = gi.make_tokens(w, 2001)
    on, st = _steps(w, params, ids, True, 4)
    off, _ = _steps(w, params, ids, False, 1)
    assert st == 2
    _same(on, [off[0]] * 4)


def test_side_streams_bf16_config2_widths_bitwise():
    """d 1024 / H 4096 / 16 heads of 64 / S 256 / T_mb 2048: kernels long enough that the two streams of a cell really
    overlap (FFN wgrads of ~30 us beside the dgrads), V kept small."""
    w = gi.CONFIGS["T(6,4096,16)"].replace(n_layers=4, causal=(0, 1, 0, 1), K=2, M=4, n_seqs=32, vocab=4096)
    params = gi.make_params(w, 1002)
    ids = gi.make_tokens(w, 2002)
    on, st = _steps(w, params, ids, True, 5)
    off, _ = _steps(w, params, ids, False, 1)
    assert st == 2
    _same(on, [off[0]] * 5)


def test_side_streams_encdec_bitwise():
    w = gi.encdec("small-encdec", 2, 1024, 4, vocab=2048, n_seqs=8, M=4, K=2, d_model=256, d_head=64, seq_len=64)
    params = gi.make_params(w, 1003)
    ids = gi.make_tokens_encdec(w, 2003)
    on, st = _steps(w, params, ids, True, 4)
    off, _ = _steps(w, params, ids, False, 1)
    assert st == 2
    _same(on, [off[0]] * 4)


def test_side_streams_off_under_trace_and_timing():
    """gpipe_trace keeps every kernel of a task on the cell's own stream (the trace's task intervals stay what they
    were); per-launch timing records on whichever stream the launch is on.  Results stay bitwise the same."""
    w = gi.CONFIGS["T(6,4096,16)"].replace(n_layers=2, causal=(0, 1), **SMALL)
    params = gi.make_params(w, 1001)
    ids = gi.make_tokens(w, 2001)
    ref, _ = _steps(w, params, ids, False, 1)
    with gp.from_workload(w) as e:
        e.set_params(params)
        e.kernel_timing(True)
        loss = e.step(*ids)
        stats = e.kernel_stats()
        assert loss == ref[0][0]
        for n, g in e.grads().items():
            assert np.array_equal(g, ref[0][1][n]), n
        assert stats["gemm_wgrad"]["launches"] > 0
        e.kernel_timing(False)
        e.zero_grads()
        e.trace(True)
        assert e.step(*ids) == ref[0][0]
        for n, g in e.grads().items():
            assert np.array_equal(g, ref[0][1][n]), n

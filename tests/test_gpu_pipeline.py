"""The pipeline handle ("places the k-th cell on the k-th accelerator"):
one arena, one stream and one device per cell, boundary activations / gradients moved between arenas by peer
copies.  The test box has ONE GPU, so the cells share device 0 - the same code path (separate parameter homes,
boundary transfers, per-cell optimizer state), minus the NVLink hop and the device switches."""
import numpy as np
import pytest

import gpipe_inputs as gi
import paper_1811_06965_b200 as gp
from paper_1811_06965_b200.binding import plan_bytes_pipeline
from tests.util import maxrel, run_oracle

pytestmark = pytest.mark.gpu


def _boundary_b2(w, K, cells):
    """b_2 of each non-final cell's last layer: the one gradient a pipeline handle sums with a different kernel."""
    return {"l%d.b_2" % (hi - 1) for (lo, hi) in cells[:-1]}


@pytest.mark.parametrize("staged", [False, True])
@pytest.mark.parametrize("remat", [True, False])
def test_pipeline_handle_fp32_matches_oracle_and_single_arena_engine(staged, remat):
    w = gi.CONFIGS["tiny"].replace(n_layers=5, causal=(0, 1, 0, 1, 1), K=3, M=4, n_seqs=8)
    params = gi.make_params(w, 1001, round_bf16=False)
    tok, lab = gi.make_tokens(w, 2001)
    o, loss_ref = run_oracle(w, params, tok, lab, remat=remat)
    with gp.from_workload(w, remat=remat) as one:
        one.set_params(params)
        loss_one = one.step(tok, lab)
        g_one = one.grads()
    with gp.from_workload(w, remat=remat, devices=[0, 0, 0], staged=staged) as e:
        assert e.cells == [(0, 2), (2, 4), (4, 5)]
        e.set_params(params)
        for n in e.names:
            assert np.array_equal(e.get_param(n), params[n]), n
        loss = e.step(tok, lab)
        assert abs(loss - loss_ref) <= 1e-4 * abs(loss_ref) and loss == loss_one
        special = _boundary_b2(w, 3, e.cells)
        for n in e.names:
            g = e.get_grad(n)
            assert maxrel(g, o.g[n]) <= 1e-4, n
            if n in special:
                assert maxrel(g, g_one[n]) <= 1e-6, n              # same addends, another summation tree
            else:
                assert np.array_equal(g, g_one[n]), n               # same kernels on the same values
        # per-accelerator memory: by_cell is what each cell's arena holds
        spec, keep = gp.make_spec(w.n_layers, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len, w.dtype,
                                  list(w.causal))
        need = plan_bytes_pipeline(spec, 3, 4, remat, 8)
        pk = e.peak_bytes()
        assert pk["by_cell"] == need and pk["total"] == sum(need)
        # a second and third step (CUDA-graph capture and replay on one device) + the update, cell by cell
        e.zero_grads()
        l2 = [e.step(tok, lab) for _ in range(3)]
        assert l2[0] == l2[1] == l2[2] == loss and e.cuda_graph_state() == 2
        for n in e.names:
            assert maxrel(e.get_grad(n), 3 * o.g[n]) <= 1e-4, n
        e.zero_grads()
        e.step(tok, lab)
        e.apply_sgd(0.5)
        o.apply_sgd(0.5)
        for n in e.names:
            assert maxrel(e.get_param(n), o.p[n]) <= 1e-5, n
            assert not e.get_grad(n).any()


def test_pipeline_handle_bf16_is_the_single_arena_engine_bitwise():
    """Config 3's shape (d 1024, H 8192, S 256, V 32000), K = 4 cells of one layer, device-resident ids, RMSProp with
    one slot shard per cell, exact state round trip."""
    import torch
    w = gi.reduced(gi.CONFIGS["T(12,8192,16)"]).replace(M=4, n_seqs=4)
    params = gi.make_params(w, 1013)
    tok, lab = gi.make_tokens(w, 2013)
    td, ld = torch.tensor(tok, device="cuda"), torch.tensor(lab, device="cuda")
    out = []
    for devices in (None, [0, 0, 0, 0]):
        with gp.from_workload(w, devices=devices, staged=devices is not None) as e:
            e.set_params(params)
            l1 = e.step(td, ld)
            g = e.grads()
            e.apply_rmsprop(0.002, 0.9, 1e-6)
            l2 = e.step(tok, lab)
            st = e.state_dict()
            out.append((l1, l2, g, st, e.cells))
    (a1, a2, ga, sa, cells), (b1, b2, gb, sb, _) = out
    assert a1 == b1
    special = _boundary_b2(w, 4, cells)
    for n in ga:
        if n in special:
            assert maxrel(gb[n], ga[n]) <= 1e-5, n
        else:
            assert np.array_equal(ga[n], gb[n]), n
    assert abs(a2 - b2) <= 1e-6 * abs(a2)                           # after the update the b_2 rounding difference is in
    for n in ga:
        if n not in special:
            assert np.array_equal(sa["slot"][n], sb["slot"][n]), n
    bad = torch.tensor(tok, device="cuda").clone()
    bad[0, 0] = w.vocab
    with gp.from_workload(w, devices=[0, 0, 0, 0]) as e:
        with pytest.raises(gp.GPipeError):
            e.step(bad, ld)
        with pytest.raises(gp.GPipeError):
            e.step(td, bad)                                        # labels are checked on the last cell's device


def test_pipeline_handle_argument_errors():
    w = gi.CONFIGS["tiny"]
    with pytest.raises(ValueError):
        gp.from_workload(w, devices=[0])
    with pytest.raises(ValueError):
        gp.from_workload(w, devices=[0, 99])                        # no such device

"""Data-parallel replicas with the gradient reduction fused into the apply.

R replicas take different mini-batches; gpipe_dp_apply_* sums their gradients over peer-mapped arenas, applies
the optimizer shard by shard and writes the update back into every replica.  The oracle's statement of the same
thing needs no replicas at all: the mean over R equal-sized mini-batches of the mean loss IS the mean loss of their
union, so the reference is ONE oracle run on the concatenated mini-batch followed by its apply.

Two set-ups on the single GPU of the test box (the kernel waits on no other replica, so R launches may run one
after the other on one device - /opt/skills/guides/B200_PROFILING.md on emulating ranks):
  * R handles in one process, each the "peer" of the others through its own arena pointer;
  * two PROCESSES sharing cuda:0 over gloo, arenas mapped into each other with CUDA IPC - the deployment path of
    paper_1811_06965_b200.dp.DataParallel minus the NVLink hop.
"""
import os
import sys

import numpy as np
import pytest

import gpipe_inputs as gi
import paper_1811_06965_b200 as gp
from tests.util import cosine, maxrel, run_oracle

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _union(w, R, seed):
    """R mini-batches of w.n_seqs sequences and their concatenation (the oracle's mini-batch)."""
    big = w.replace(n_seqs=w.n_seqs * R, M=w.M * R)
    tok, lab = gi.make_tokens(big, seed)
    parts = [(tok[r * w.n_seqs:(r + 1) * w.n_seqs], lab[r * w.n_seqs:(r + 1) * w.n_seqs]) for r in range(R)]
    return big, tok, lab, parts


@pytest.mark.parametrize("R", [2, 3])
@pytest.mark.parametrize("opt", ["sgd", "rmsprop"])
def test_fused_dp_apply_matches_oracle_on_the_union_batch(R, opt):
    w = gi.CONFIGS["tiny"].replace(causal=(0, 1))
    params = gi.make_params(w, 1001, round_bf16=False)
    engines = [gp.from_workload(w) for _ in range(R)]
    try:
        for e in engines:
            e.set_params(params)
        arenas = [e.arena_base for e in engines]
        o = None
        for it in range(2):                                      # two updates: the second starts from the first's result
            big, tok, lab, parts = _union(w, R, 2300 + it)
            if o is None:
                o, _ = run_oracle(big, params, tok, lab)
                o.zero_grads()
            loss_ref = o.step(tok, lab)
            losses = [e.step(*parts[r]) for r, e in enumerate(engines)]
            assert abs(np.mean(losses) - loss_ref) <= 1e-5 * abs(loss_ref)
            for r, e in enumerate(engines):                      # the phases are separated by program order here
                if opt == "sgd":
                    e.dp_apply_sgd(r, arenas, 0.5)
                else:
                    e.dp_apply_rmsprop(r, arenas, 0.002, 0.9, 1e-6)
            if opt == "sgd":
                o.apply_sgd(0.5)
            else:
                o.apply_rmsprop(0.002, 0.9, 1e-6)
            ref = engines[0]
            for n in ref.names:
                p0 = ref.get_param(n)
                assert maxrel(p0, o.p[n]) <= (1e-5 if opt == "sgd" else 2e-4), (it, n)
                for e in engines[1:]:
                    assert np.array_equal(e.get_param(n), p0), n      # one owner computed each element
                for e in engines:
                    assert not e.get_grad(n).any(), n                  # cleared in every replica by the owner
    finally:
        for e in engines:
            e.close()


def test_fused_dp_apply_bf16_replicas_stay_identical_and_equal_one_big_step():
    """bf16: masters identical in all replicas, working copy = RNE(master), and the update equals what ONE engine
    computes for the union mini-batch (same kernels, same per-token values; only the fp32 order of the gradient
    sum differs: replica sum vs micro-batch accumulation)."""
    w = gi.CONFIGS["T(6,4096,16)"].replace(name="bf16-dp", n_layers=2, d_model=256, d_ffn=1024, n_heads=4, d_head=64,
                                           vocab=2048, seq_len=64, n_seqs=8, M=4, K=2, causal=(0, 1))
    R = 2
    params = gi.make_params(w, 1002)
    big, tok, lab, parts = _union(w, R, 2310)
    engines = [gp.from_workload(w) for _ in range(R)]
    try:
        for e in engines:
            e.set_params(params)
        arenas = [e.arena_base for e in engines]
        for r, e in enumerate(engines):
            e.step(*parts[r])
        for r, e in enumerate(engines):
            e.dp_apply_sgd(r, arenas, 0.25)
        with gp.from_workload(big) as one:
            one.set_params(params)
            one.step(tok, lab)
            one.apply_sgd(0.25)
            for n in one.names:
                m0 = engines[0].get_master(n)
                assert np.array_equal(engines[1].get_master(n), m0), n
                assert np.array_equal(engines[0].get_param(n), engines[1].get_param(n)), n
                upd, ref = m0 - params[n], one.get_master(n) - params[n]
                # the update is read back as (new master - old parameter): a difference of fp32 numbers ~1e3 x larger
                # than itself, so the comparison carries their rounding (2^-24 x |w| / |update| ~ 1e-5 .. 1e-4)
                assert maxrel(upd, ref) <= 2e-4 and cosine(upd, ref) >= 0.999999, n
        import torch
        for e in engines:                                        # working copy = RNE(master) for matrices
            wq = e.get_param("l0.w_qkv")
            mq = torch.tensor(e.get_master("l0.w_qkv")).to(torch.bfloat16).float().numpy()
            assert np.array_equal(wq, mq)
    finally:
        for e in engines:
            e.close()


def _ipc_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)      # both ranks share cuda:0: NCCL needs one GPU per rank
    try:
        import gpipe_inputs as gi_
        import paper_1811_06965_b200 as gp_
        from paper_1811_06965_b200.dp import DataParallel
        w = gi_.CONFIGS["tiny"].replace(causal=(0, 1))
        params = gi_.make_params(w, 1001, round_bf16=False)
        big = w.replace(n_seqs=w.n_seqs * world, M=w.M * world)
        tok, lab = gi_.make_tokens(big, 2320)
        sl = slice(rank * w.n_seqs, (rank + 1) * w.n_seqs)
        with gp_.from_workload(w) as e:
            e.set_params(params)
            dp = DataParallel(e)
            losses = []
            for it in range(2):
                losses.append(e.step(tok[sl], lab[sl]))
                dp.apply_sgd(0.5)
            out = {n: e.get_param(n) for n in e.names}
            zero = all(not e.get_grad(n).any() for n in e.names)
            dp.close()
        q.put((rank, losses, out, zero, None))
    except Exception as ex:                                             # surface the failure in the parent
        import traceback
        q.put((rank, None, None, None, traceback.format_exc()))
        raise ex
    finally:
        dist.destroy_process_group()


def test_two_processes_on_one_gpu_over_cuda_ipc():
    import torch.multiprocessing as mp
    w = gi.CONFIGS["tiny"].replace(causal=(0, 1))
    params = gi.make_params(w, 1001, round_bf16=False)
    big = w.replace(n_seqs=w.n_seqs * 2, M=w.M * 2)
    tok, lab = gi.make_tokens(big, 2320)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33500 + os.getpid() % 2000
    procs = [ctx.Process(target=_ipc_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    for r in res:
        assert r[4] is None, r[4]
    o, _ = run_oracle(big, params, tok, lab)
    o.zero_grads()
    for it in range(2):
        loss_ref = o.step(tok, lab)
        assert abs(0.5 * (res[0][1][it] + res[1][1][it]) - loss_ref) <= 1e-5 * abs(loss_ref)
        o.apply_sgd(0.5)
    for n in o.names:
        assert np.array_equal(res[0][2][n], res[1][2][n]), n
        assert maxrel(res[0][2][n], o.p[n]) <= 1e-5, n
    assert res[0][3] and res[1][3]

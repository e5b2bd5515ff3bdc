"""world_size-2 gloo test of the N > 1 plumbing bench.py uses (replicas only: no data-path
collective exists; the ranks only agree on the timed region)."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1811_06965_b200.dist_util import barrier, max_over_ranks, whole_job_throughput
    barrier(world)
    mx = max_over_ranks(10.0 + 5.0 * rank, world)
    q.put((rank, mx, whole_job_throughput(1000, 4, mx, world)))
    dist.destroy_process_group()


def test_max_over_ranks_and_throughput_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, thr in res:
        assert mx == 15.0                              # the slowest rank's time, on every rank
        assert abs(thr - 1000 * 2 * 4 / 0.015) < 1e-6  # whole-job units / max time


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    from paper_1811_06965_b200.dist_util import max_over_ranks, whole_job_throughput
    assert max_over_ranks(3.5, 1) == 3.5
    assert whole_job_throughput(10, 2, 1000.0, 1) == 20.0

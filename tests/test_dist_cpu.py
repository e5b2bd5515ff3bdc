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


# -------------------------------------------------------------------------------------------------
# data-parallel replicas: shard arithmetic (host-only C call) and the host
# protocol of paper_1811_06965_b200.dp.DataParallel over gloo, world size 2, with a recording stand-in
# for the engine and for the CUDA-IPC primitives (the kernel itself is covered by the -m gpu tests)
# -------------------------------------------------------------------------------------------------
def test_dp_shards_partition_the_flat_range():
    sys.path.insert(0, ROOT)
    from paper_1811_06965_b200.binding import dp_shard
    for n in (0, 64, 640, 64 * 1000 + 64, 5_500_000_064):
        for world in (1, 2, 3, 8, 16):
            cuts = [dp_shard(n, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            for (a, b), (c, d) in zip(cuts, cuts[1:]):
                assert b == c and a <= b                       # contiguous, disjoint, in rank order
            for a, b in cuts:
                assert a % 64 == 0 and (b % 64 == 0 or b == n)  # tensors start on 64-element boundaries
            sizes = [b - a for a, b in cuts]
            assert max(sizes) - min(s for s in sizes if s or n == 0) <= 64 * world or min(sizes) == 0


class _FakeEngine:
    def __init__(self, rank, log):
        self.arena_base = 0x1000 * (rank + 1)
        self.rank, self.log = rank, log

    def dp_layout(self):
        return {"n_flat": 1024, "master_off": 0, "grad_off": 4096, "wlp_off": 8192}

    def dp_apply_sgd(self, rank, peer_arenas, lr, grad_scale):
        self.log.append(("sgd", rank, list(peer_arenas), lr, grad_scale))

    def dp_apply_rmsprop(self, rank, peer_arenas, lr, rho, eps, grad_scale):
        self.log.append(("rmsprop", rank, list(peer_arenas), lr, rho, eps, grad_scale))


def _dp_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1811_06965_b200.dp import DataParallel
    log, opened, closed = [], [], []

    def export(ptr):
        return (b"H%d" % rank) * 16, 256 * (rank + 1)          # (handle, offset of the arena in its allocation)

    def open_(handle):
        opened.append(handle)
        return 0x100000 * (1 + int(handle[1:2]))                # a distinct fake mapping per peer

    dp = DataParallel(_FakeEngine(rank, log), export=export, open_=open_, close=closed.append)
    dp.apply_sgd(0.5)
    dp.apply_rmsprop(0.1, 0.9, 1e-6, grad_scale=1.0)
    dp.close()
    q.put((rank, dp.peer_arenas, log, opened, closed))
    dist.destroy_process_group()


def test_data_parallel_host_protocol_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_dp_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, peers, log, opened, closed in res:
        other = 1 - rank
        own = 0x1000 * (rank + 1)
        mapped = 0x100000 * (1 + other) + 256 * (other + 1)     # the peer's mapping + the arena's offset in it
        assert peers[rank] == own and peers[other] == mapped
        assert opened == [(b"H%d" % other) * 16] and closed == [0x100000 * (1 + other)]
        assert log == [("sgd", rank, peers, 0.5, None), ("rmsprop", rank, peers, 0.1, 0.9, 1e-6, 1.0)]

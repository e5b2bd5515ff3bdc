"""Brute-force simulation of the GPipe schedule.  TEST INFRASTRUCTURE (part of the oracle).

Each of the K cells is an in-order queue (one accelerator): F(k,0..M-1), then for
m = M-1..0: [R(k,m)], B(k,m).  Dependencies (PAPER.md:53 Fig. 2 caption, :67): F(k,m) after
F(k-1,m); B(k,m) after B(k+1,m); B(K-1,m) after F(K-1,M-1) is implied by the queue order.
The re-materialization task R(k,m) needs only the stored boundary activation; "early" lets
it start without waiting for B(k+1,m) ("re-computation during the backward pass
can be scheduled earlier, without waiting for the gradients from earlier layers"), "late"
makes it wait.  A task starts at max(cell free, dependencies done).  No closed form is used
here: the closed forms live in the tests that pin this simulator (PAPER.md:89 bubble
O((K-1)/(M+K-1))).
"""
from __future__ import annotations

from typing import Dict, List, Tuple


def cell_program(k: int, K: int, M: int, remat: bool) -> List[Tuple[str, int, int]]:
    prog = [("F", k, m) for m in range(M)]
    for m in range(M - 1, -1, -1):
        if remat:
            prog.append(("R", k, m))
        prog.append(("B", k, m))
    return prog


def dependencies(task, K: int, remat: bool, early: bool):
    kind, k, m = task
    deps = []
    if kind == "F" and k > 0:
        deps.append(("F", k - 1, m))
    if kind == "B" and k < K - 1:
        deps.append(("B", k + 1, m))
    if kind == "R" and not early and k < K - 1:
        deps.append(("B", k + 1, m))
    return deps


def simulate(K: int, M: int, t_f: float = 1.0, t_b: float = 1.0, t_r: float = 0.0,
             remat: bool = False, early: bool = True) -> Dict[str, object]:
    """Event simulation; returns makespan, per-cell busy time, total idle, idle fraction and
    the (start, end) of every task."""
    cost = {"F": t_f, "B": t_b, "R": t_r}
    progs = [cell_program(k, K, M, remat) for k in range(K)]
    pc = [0] * K
    free = [0.0] * K
    done: Dict[Tuple[str, int, int], Tuple[float, float]] = {}
    remaining = sum(len(p) for p in progs)
    while remaining:
        progressed = False
        for k in range(K):
            while pc[k] < len(progs[k]):
                task = progs[k][pc[k]]
                deps = dependencies(task, K, remat, early)
                if any(d not in done for d in deps):
                    break
                start = max([free[k]] + [done[d][1] for d in deps])
                end = start + cost[task[0]]
                done[task] = (start, end)
                free[k] = end
                pc[k] += 1
                remaining -= 1
                progressed = True
        if not progressed:
            raise RuntimeError("schedule deadlock")
    makespan = max(e for _, e in done.values())
    busy = [sum(e - s for (kind, kk, m), (s, e) in done.items() if kk == k) for k in range(K)]
    idle = sum(makespan - b for b in busy)
    return dict(makespan=makespan, busy=busy, idle=idle, idle_fraction=idle / (K * makespan),
                tasks=done)


def max_concurrency(sim) -> int:
    """Largest number of cells busy at the same instant (M = 1 must give 1)."""
    pts = []
    for (s, e) in sim["tasks"].values():
        if e > s:
            pts.append((s, 1))
            pts.append((e, -1))
    pts.sort(key=lambda t: (t[0], t[1]))
    cur = best = 0
    for _, dlt in pts:
        cur += dlt
        best = max(best, cur)
    return best

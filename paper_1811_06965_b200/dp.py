"""Data-parallel replicas of the GPipe engine: one process per GPU, each with a
full pipeline (all K cells) on its own mini-batch; after every replica's step the gradients are summed across
replicas and applied once - by ONE kernel per replica that reads its parameter shard's gradients out of every
replica's arena over NVLink peer memory, applies the optimizer and stores the updated parameters back into every
replica (gpipe_dp_apply_sgd / gpipe_dp_apply_rmsprop: reduce-scatter + apply + all-gather fused, no NCCL call on the
data path).  torch.distributed is plumbing only: it carries the CUDA-IPC handles of the arenas once, and the two
barriers per update that separate "all gradients final" / "all parameters updated" from the neighbouring steps.

Marshalling only - the arithmetic is in the library's kernel.  There is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
from typing import Callable, List, Optional

from . import binding as B


def _ipc_export(ptr: int):
    handle = C.create_string_buffer(64)
    off = C.c_size_t(0)
    B._check(B.lib().gpipe_ipc_export(C.c_void_p(ptr), handle, C.byref(off)))
    return bytes(handle.raw), int(off.value)


def _ipc_open(handle: bytes) -> int:
    base = C.c_void_p(None)
    B._check(B.lib().gpipe_ipc_open(C.c_char_p(handle), C.byref(base)))
    return int(base.value)


def _ipc_close(base: int) -> None:
    B._check(B.lib().gpipe_ipc_close(C.c_void_p(base)))


class DataParallel:
    """Wraps one replica's GPipe engine.  `engine` needs: arena_base, dp_layout(), dp_apply_sgd(), dp_apply_rmsprop().
    rank / world default to torch.distributed's; `export`, `open_` and `close` are the IPC primitives (overridable so
    that the host logic can be exercised on CPU)."""

    def __init__(self, engine, rank: Optional[int] = None, world: Optional[int] = None, group=None,
                 export: Callable = _ipc_export, open_: Callable = _ipc_open, close: Callable = _ipc_close):
        import torch.distributed as dist
        self._dist, self._group, self.engine = dist, group, engine
        self.rank = dist.get_rank(group) if rank is None else rank
        self.world = dist.get_world_size(group) if world is None else world
        self._close = close
        layout = engine.dp_layout()
        handle, offset = export(engine.arena_base)
        mine = {"rank": self.rank, "handle": handle, "offset": offset, "layout": layout}
        everyone: List[Optional[dict]] = [None] * self.world
        dist.all_gather_object(everyone, mine, group=group)
        self._opened: List[int] = []
        self.peer_arenas: List[int] = []
        for p, info in enumerate(everyone):
            if info["rank"] != p:
                raise RuntimeError("data-parallel ranks are out of order")
            if info["layout"] != layout:
                # the fused kernel addresses every replica with ONE set of offsets: the plans must be identical
                raise RuntimeError("replica %d was created with a different plan than replica %d: %r vs %r"
                                   % (p, self.rank, info["layout"], layout))
            if p == self.rank:
                self.peer_arenas.append(engine.arena_base)
            else:
                base = open_(info["handle"])
                self._opened.append(base)
                self.peer_arenas.append(base + info["offset"])

    def _update(self, fn):
        # (1) every replica's step has returned: all gradients are final
        self._dist.barrier(group=self._group)
        fn()                                                   # synchronous: this replica's shard is updated everywhere
        # (2) every shard is updated in every replica before anyone starts the next step
        self._dist.barrier(group=self._group)

    def apply_sgd(self, lr: float, grad_scale: Optional[float] = None):
        self._update(lambda: self.engine.dp_apply_sgd(self.rank, self.peer_arenas, lr, grad_scale))

    def apply_rmsprop(self, lr: float, rho: float = 0.9, eps: float = 1e-8, grad_scale: Optional[float] = None):
        self._update(lambda: self.engine.dp_apply_rmsprop(self.rank, self.peer_arenas, lr, rho, eps, grad_scale))

    def close(self):
        self._dist.barrier(group=self._group)                  # nobody still addresses a mapping that is about to go
        for base in self._opened:
            self._close(base)
        self._opened = []

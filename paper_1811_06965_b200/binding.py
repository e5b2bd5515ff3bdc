"""ctypes binding of libgpipe_b200.so (include/gpipe.h, include/gpipe_ops.h).

Argument marshalling only: every step of the path runs in the library's CUDA kernels.  PyTorch
supplies device memory (one uint8 arena tensor) and the K CUDA streams; there is no CPU fallback -
if the shared library is missing or no B200 is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# GPIPE_LIB_PATH selects another build of the same ABI (A/B comparisons of two kernel versions inside one gpurun call)
LIB_PATH = os.environ.get("GPIPE_LIB_PATH") or os.path.join(_HERE, "libgpipe_b200.so")

DTYPE_FP32, DTYPE_BF16 = 0, 1
CATEGORIES = ["weights", "masters", "grads", "boundary", "interior", "head", "misc", "bwd_scratch"]
EPI_BIAS, EPI_RELU, EPI_MASK, EPI_RESID, EPI_ACCUM, EPI_OUT_F32, EPI_COLSUM, EPI_BITS_OUT = 1, 2, 4, 8, 16, 32, 64, 128


class GPipeError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("gpipe error %d: %s" % (code, msg))
        self.code = code


class LayerSpec(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("d_model", C.c_int32), ("d_ffn", C.c_int32),
                ("n_heads", C.c_int32), ("d_head", C.c_int32), ("vocab", C.c_int32),
                ("seq_len", C.c_int32), ("dtype", C.c_int32), ("causal", C.POINTER(C.c_uint8)),
                ("ln_eps", C.c_float)]


class EncDecSpec(C.Structure):
    _fields_ = [("n_enc", C.c_int32), ("n_dec", C.c_int32), ("d_model", C.c_int32), ("d_ffn", C.c_int32),
                ("n_heads", C.c_int32), ("d_head", C.c_int32), ("vocab", C.c_int32), ("seq_len", C.c_int32),
                ("dtype", C.c_int32), ("ln_eps", C.c_float), ("logit_clip", C.c_float)]


class Env(C.Structure):
    _fields_ = [("arena", C.c_void_p), ("arena_bytes", C.c_size_t),
                ("streams", C.POINTER(C.c_void_p)), ("n_streams", C.c_int32)]


class CellEnv(C.Structure):
    _fields_ = [("device", C.c_int32), ("arena", C.c_void_p), ("arena_bytes", C.c_size_t), ("stream", C.c_void_p)]


PIPE_STAGED = 1


class TraceEvent(C.Structure):
    _fields_ = [("kind", C.c_int32), ("k", C.c_int32), ("m", C.c_int32), ("enqueue_index", C.c_int32),
                ("start_ms", C.c_float), ("end_ms", C.c_float)]


_lib = None


def lib() -> C.CDLL:
    """Loads the shared library (once).  Fails loudly when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s is missing: run `python -m paper_1811_06965_b200.build` "
                          "(there is no CPU fallback)" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, f32 = C.c_void_p, C.c_int, C.c_int64, C.c_float
    sig = {
        "gpipe_plan_bytes": (i32, [C.POINTER(LayerSpec), i32, i32, i32, i64, C.POINTER(C.c_size_t)]),
        "gpipe_create": (i32, [C.POINTER(LayerSpec), i32, i32, i32, i64, C.POINTER(Env), C.POINTER(vp)]),
        "gpipe_destroy": (None, [vp]),
        "gpipe_layer_costs": (i32, [C.POINTER(LayerSpec), i32, C.POINTER(C.c_double), C.POINTER(C.c_double),
                                    C.POINTER(C.c_double)]),
        "gpipe_partition_min_variance": (i32, [C.POINTER(C.c_double), i32, C.c_double, C.c_double, i32,
                                               C.POINTER(C.c_int32)]),
        "gpipe_create_partitioned": (i32, [C.POINTER(LayerSpec), i32, i32, i32, i64, C.POINTER(Env),
                                           C.POINTER(C.c_int32), C.POINTER(vp)]),
        "gpipe_cell_range": (i32, [vp, i32, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]),
        "gpipe_plan_bytes_pipeline": (i32, [C.POINTER(LayerSpec), i32, i32, i32, i64, C.POINTER(C.c_int32),
                                            C.POINTER(C.c_size_t)]),
        "gpipe_create_pipeline": (i32, [C.POINTER(LayerSpec), i32, i32, i32, i64, C.POINTER(CellEnv),
                                        C.POINTER(C.c_int32), i32, C.POINTER(vp)]),
        "gpipe_attach_optimizer_slots_cell": (i32, [vp, i32, vp, C.c_size_t]),
        "gpipe_cell_param_count": (i32, [vp, i32, C.POINTER(i64)]),
        "gpipe_plan_bytes_encdec": (i32, [C.POINTER(EncDecSpec), i32, i32, i32, i64, C.POINTER(C.c_int32),
                                          C.POINTER(C.c_size_t)]),
        "gpipe_create_encdec": (i32, [C.POINTER(EncDecSpec), i32, i32, i32, i64, C.POINTER(Env), C.POINTER(C.c_int32),
                                      C.POINTER(vp)]),
        "gpipe_layer_costs_encdec": (i32, [C.POINTER(EncDecSpec), i32, C.POINTER(C.c_double), C.POINTER(C.c_double),
                                           C.POINTER(C.c_double)]),
        "gpipe_plan_bytes_pipeline_encdec": (i32, [C.POINTER(EncDecSpec), i32, i32, i32, i64, C.POINTER(C.c_int32),
                                                   C.POINTER(C.c_size_t)]),
        "gpipe_create_pipeline_encdec": (i32, [C.POINTER(EncDecSpec), i32, i32, i32, i64, C.POINTER(CellEnv),
                                               C.POINTER(C.c_int32), i32, C.POINTER(vp)]),
        "gpipe_step_encdec": (i32, [vp, vp, vp, vp, C.POINTER(f32)]),
        "gpipe_step_encdec_device": (i32, [vp, vp, vp, vp, C.POINTER(f32)]),
        "gpipe_init_params": (i32, [vp, C.c_uint64, f32, i32]),
        "gpipe_init_params_scaled": (i32, [vp, C.c_uint64, f32, i32, f32]),
        "gpipe_step": (i32, [vp, vp, vp, C.POINTER(f32)]),
        "gpipe_step_device": (i32, [vp, vp, vp, C.POINTER(f32)]),
        "gpipe_apply_sgd": (i32, [vp, f32]),
        "gpipe_optimizer_slot_bytes": (i32, [vp, C.POINTER(C.c_size_t)]),
        "gpipe_attach_optimizer_slots": (i32, [vp, vp, C.c_size_t]),
        "gpipe_apply_rmsprop": (i32, [vp, f32, f32, f32]),
        "gpipe_zero_grads": (i32, [vp]),
        "gpipe_dp_shard": (i32, [i64, i32, i32, C.POINTER(i64), C.POINTER(i64)]),
        "gpipe_dp_layout": (i32, [vp, C.POINTER(i64), C.POINTER(C.c_size_t), C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]),
        "gpipe_dp_apply_sgd": (i32, [vp, i32, i32, C.POINTER(vp), f32, f32]),
        "gpipe_dp_apply_rmsprop": (i32, [vp, i32, i32, C.POINTER(vp), f32, f32, f32, f32]),
        "gpipe_ipc_export": (i32, [vp, C.c_char_p, C.POINTER(C.c_size_t)]),
        "gpipe_ipc_open": (i32, [C.c_char_p, C.POINTER(vp)]),
        "gpipe_ipc_close": (i32, [vp]),
        "gpipe_num_tensors": (i32, [vp]),
        "gpipe_tensor_info": (i32, [vp, i32, C.POINTER(C.c_char_p), C.POINTER(i64), C.POINTER(i64)]),
        "gpipe_get_param": (i32, [vp, i32, vp]),
        "gpipe_set_param": (i32, [vp, i32, vp]),
        "gpipe_get_grad": (i32, [vp, i32, vp]),
        "gpipe_get_master": (i32, [vp, i32, vp]),
        "gpipe_set_master": (i32, [vp, i32, vp]),
        "gpipe_get_optimizer_slot": (i32, [vp, i32, vp]),
        "gpipe_set_optimizer_slot": (i32, [vp, i32, vp]),
        "gpipe_peak_bytes": (i32, [vp, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]),
        "gpipe_trace": (i32, [vp, i32, C.POINTER(TraceEvent), C.POINTER(i64)]),
        "gpipe_launch_count": (i64, [vp]),
        "gpipe_cuda_graph": (i32, [vp, i32]),
        "gpipe_cuda_graph_state": (i32, [vp]),
        "gpipe_kernel_timing": (i32, [vp, i32]),
        "gpipe_kernel_stats": (i32, [vp, i32, C.POINTER(C.c_char_p), C.POINTER(i64), C.POINTER(C.c_double),
                                     C.POINTER(C.c_double), C.POINTER(C.c_double)]),
        "gpipe_debug_read": (i32, [vp, C.c_char_p, i32, vp, i64, C.POINTER(i64)]),
        "gpipe_last_error": (C.c_char_p, []),
        "gpipe_version": (C.c_char_p, []),
        "gpipe_op_gemm": (i32, [vp, i32, i32, i32, i32, vp, i64, i32, vp, i64, i32, vp, i64, vp, vp, vp, i64, vp, vp, vp, i64, i32, i32]),
        "gpipe_op_gemm_workspace_bytes": (i64, [i32, i32, i32]),
        "gpipe_op_ln_fwd": (i32, [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, i64, i32, f32]),
        "gpipe_op_ln_bwd_scratch_floats": (i64, [i32]),
        "gpipe_op_ln_bwd": (i32, [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, i64, i32]),
        "gpipe_op_attn_fwd": (i32, [vp, i32, vp, vp, vp, i32, i32, i32, i32, i32, i32]),
        "gpipe_op_attn_bwd": (i32, [vp, i32, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, vp]),
        "gpipe_op_softmax_ce": (i32, [vp, i32, vp, vp, vp, i64, i32, f32, f32]),
        "gpipe_op_colsum_scratch_floats": (i64, [i64, i32]),
        "gpipe_op_colsum": (i32, [vp, i32, vp, i64, vp, vp, i64, i32]),
        "gpipe_op_colsum_static": (i32, [vp, i32, vp, i64, vp, i64, i32]),
        "gpipe_op_embed_fwd": (i32, [vp, i32, vp, vp, vp, vp, i64, i32, i32]),
        "gpipe_op_embed_bwd": (i32, [vp, vp, vp, vp, i64, i32]),
        "gpipe_op_positional": (i32, [vp, vp, i32, i32]),
        "gpipe_op_sgd": (i32, [vp, i32, vp, vp, vp, i64, f32]),
        "gpipe_op_dp_apply_sgd": (i32, [vp, i32, i32, i32, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), i64, f32, f32]),
        "gpipe_op_rmsprop": (i32, [vp, i32, vp, vp, vp, vp, i64, f32, f32, f32]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    _lib = L
    return L


EXPORTED_SYMBOLS = [
    "gpipe_plan_bytes", "gpipe_create", "gpipe_destroy", "gpipe_layer_costs", "gpipe_partition_min_variance",
    "gpipe_create_partitioned", "gpipe_cell_range", "gpipe_plan_bytes_pipeline", "gpipe_create_pipeline",
    "gpipe_attach_optimizer_slots_cell", "gpipe_cell_param_count", "gpipe_init_params", "gpipe_init_params_scaled",
    "gpipe_plan_bytes_encdec", "gpipe_create_encdec", "gpipe_layer_costs_encdec", "gpipe_plan_bytes_pipeline_encdec", "gpipe_create_pipeline_encdec",
    "gpipe_step_encdec", "gpipe_step_encdec_device", "gpipe_step",
    "gpipe_step_device", "gpipe_apply_sgd", "gpipe_optimizer_slot_bytes", "gpipe_attach_optimizer_slots",
    "gpipe_apply_rmsprop", "gpipe_op_rmsprop", "gpipe_zero_grads", "gpipe_dp_shard", "gpipe_dp_layout",
    "gpipe_dp_apply_sgd", "gpipe_dp_apply_rmsprop", "gpipe_ipc_export", "gpipe_ipc_open", "gpipe_ipc_close", "gpipe_num_tensors",
    "gpipe_tensor_info", "gpipe_get_param", "gpipe_set_param", "gpipe_get_grad", "gpipe_get_master", "gpipe_set_master",
    "gpipe_get_optimizer_slot", "gpipe_set_optimizer_slot", "gpipe_peak_bytes",
    "gpipe_trace", "gpipe_launch_count", "gpipe_cuda_graph", "gpipe_cuda_graph_state", "gpipe_kernel_timing", "gpipe_kernel_stats", "gpipe_debug_read", "gpipe_last_error", "gpipe_version",
    "gpipe_op_gemm", "gpipe_op_gemm_workspace_bytes", "gpipe_op_ln_fwd", "gpipe_op_ln_bwd_scratch_floats", "gpipe_op_ln_bwd",
    "gpipe_op_attn_fwd", "gpipe_op_attn_bwd", "gpipe_op_softmax_ce", "gpipe_op_colsum",
    "gpipe_op_colsum_scratch_floats", "gpipe_op_colsum_static",
    "gpipe_op_embed_fwd", "gpipe_op_embed_bwd", "gpipe_op_positional", "gpipe_op_sgd", "gpipe_op_dp_apply_sgd",
]


def _check(rc: int):
    if rc != 0:
        raise GPipeError(rc, lib().gpipe_last_error().decode("utf-8", "replace"))


def make_spec(n_layers, d_model, d_ffn, n_heads, d_head, vocab, seq_len, dtype, causal=None,
              ln_eps=1e-5) -> Tuple[LayerSpec, object]:
    """Returns (spec, keepalive) - keepalive owns the causal array the spec points to."""
    dt = {"fp32": DTYPE_FP32, "bf16": DTYPE_BF16, 0: 0, 1: 1}[dtype]
    keep = None
    ptr = C.POINTER(C.c_uint8)()
    if causal is not None:
        if len(causal) != n_layers:
            raise ValueError("causal must have n_layers entries")
        keep = (C.c_uint8 * max(n_layers, 1))(*[1 if c else 0 for c in causal])
        ptr = C.cast(keep, C.POINTER(C.c_uint8))
    return LayerSpec(n_layers, d_model, d_ffn, n_heads, d_head, vocab, seq_len, dt, ptr, ln_eps), keep


def dp_shard(n_flat: int, rank: int, world: int) -> Tuple[int, int]:
    """gpipe_dp_shard: the [lo, hi) element range of the flat parameter array replica `rank` owns; host-only."""
    lo, hi = C.c_int64(), C.c_int64()
    _check(lib().gpipe_dp_shard(n_flat, rank, world, C.byref(lo), C.byref(hi)))
    return lo.value, hi.value


def plan_bytes(spec: LayerSpec, K: int, M: int, remat: bool, n_seqs: int) -> int:
    """gpipe_plan_bytes: host-only, works without a GPU."""
    out = C.c_size_t(0)
    _check(lib().gpipe_plan_bytes(C.byref(spec), K, M, int(bool(remat)), n_seqs, C.byref(out)))
    return int(out.value)


def plan_bytes_encdec(spec: "EncDecSpec", K: int, M: int, remat: bool, n_seqs: int, cell_lo=None) -> int:
    """gpipe_plan_bytes_encdec: host-only."""
    out = C.c_size_t(0)
    lo = (C.c_int32 * (K + 1))(*[int(v) for v in cell_lo]) if cell_lo is not None else None
    _check(lib().gpipe_plan_bytes_encdec(C.byref(spec), K, M, int(bool(remat)), n_seqs, lo, C.byref(out)))
    return int(out.value)


def layer_costs_encdec(spec: "EncDecSpec", remat: bool) -> Tuple[List[float], float, float]:
    """gpipe_layer_costs_encdec: (per-layer costs, embedding cost, head cost); host-only."""
    L = spec.n_enc + spec.n_dec
    arr = (C.c_double * max(L, 1))()
    emb, head = C.c_double(0), C.c_double(0)
    _check(lib().gpipe_layer_costs_encdec(C.byref(spec), int(bool(remat)), arr, C.byref(emb), C.byref(head)))
    return [arr[i] for i in range(L)], emb.value, head.value


def plan_bytes_pipeline(spec: LayerSpec, K: int, M: int, remat: bool, n_seqs: int, cell_lo=None) -> List[int]:
    """gpipe_plan_bytes_pipeline: bytes each cell's arena needs when every cell has its own; host-only."""
    out = (C.c_size_t * K)()
    lo = (C.c_int32 * (K + 1))(*[int(v) for v in cell_lo]) if cell_lo is not None else None
    _check(lib().gpipe_plan_bytes_pipeline(C.byref(spec), K, M, int(bool(remat)), n_seqs, lo, out))
    return [int(out[k]) for k in range(K)]


def layer_costs(spec: LayerSpec, remat: bool) -> Tuple[List[float], float, float]:
    """gpipe_layer_costs: (per-layer costs, embedding cost, head cost); host-only."""
    L = spec.n_layers
    arr = (C.c_double * max(L, 1))()
    emb, head = C.c_double(0), C.c_double(0)
    _check(lib().gpipe_layer_costs(C.byref(spec), int(bool(remat)), arr, C.byref(emb), C.byref(head)))
    return [arr[i] for i in range(L)], emb.value, head.value


def partition_min_variance(costs, first_extra: float, last_extra: float, K: int) -> List[int]:
    """gpipe_partition_min_variance: the K+1 cell boundaries; host-only."""
    L = len(costs)
    arr = (C.c_double * max(L, 1))(*[float(c) for c in costs])
    out = (C.c_int32 * (K + 1))()
    _check(lib().gpipe_partition_min_variance(arr, L, float(first_extra), float(last_extra), K, out))
    return [out[i] for i in range(K + 1)]


class GPipe:
    """gpipe_create / gpipe_step / gpipe_apply_sgd (BASELINE.json north_star) on one B200.
    partition: None (equal consecutive split), "cost" (gpipe_layer_costs + gpipe_partition_min_variance,
    PAPER.md:65) or an explicit list of K+1 boundaries.
    devices: None - all K cells on `device`, one arena, K streams; or a list of K CUDA device ordinals - the
    pipeline across accelerators (gpipe_create_pipeline): cell k's arena and stream live on
    devices[k] (the ordinals may repeat: several cells, or all of them, on one GPU); staged=True forces the
    boundary copies that different devices always use."""

    def __init__(self, *, n_layers, d_model, d_ffn, n_heads, d_head, vocab, seq_len, dtype, K, M,
                 remat=True, n_seqs, causal=None, ln_eps=1e-5, device="cuda:0", partition=None, devices=None,
                 staged=False, side_streams=None):
        import torch
        if not torch.cuda.is_available():
            raise GPipeError(-2, "no CUDA device: the GPipe path has no CPU fallback")
        self._torch = torch
        self.device = torch.device(device)
        self.spec, self._keep = make_spec(n_layers, d_model, d_ffn, n_heads, d_head, vocab, seq_len,
                                          dtype, causal, ln_eps)
        self.K, self.M, self.remat, self.n_seqs, self.seq_len = K, M, bool(remat), n_seqs, seq_len
        self._h = C.c_void_p(None)
        self.devices = None if devices is None else [int(d) for d in devices]
        # gpipe_env.n_streams = 2K: each cell's weight-gradient GEMMs run beside its dgrad / LayerNorm / attention chain.
        # None: on for K <= 2 - with more cells on the GPU the other cells' kernels already fill the SMs a cell's
        # narrow launches leave idle (measured: K 2 -3 %, K 4 +2 %, K 8 / 16 +-0.5 %)
        self.side_streams = (K <= 2 if side_streams is None else bool(side_streams)) and devices is None
        if self.devices is not None:
            self._create_pipeline(torch, K, M, n_seqs, partition, staged)
        else:
            self._create_single(torch, K, M, remat, n_seqs, partition)
        self._finish_init(K)

    def _create_pipeline(self, torch, K, M, n_seqs, partition, staged):
        if len(self.devices) != K:
            raise ValueError("devices must list one CUDA device per cell")
        if any(d < 0 or d >= torch.cuda.device_count() for d in self.devices):
            raise ValueError("devices %r: this process sees %d CUDA device(s)" % (self.devices, torch.cuda.device_count()))
        self.device = torch.device("cuda", self.devices[0])
        if isinstance(partition, str):
            if partition != "cost":
                raise ValueError("partition must be None, 'cost' or a list of K+1 boundaries")
            costs, c_emb, c_head = layer_costs(self.spec, self.remat)
            partition = partition_min_variance(costs, c_emb, c_head, K)
        need = plan_bytes_pipeline(self.spec, K, M, self.remat, n_seqs, partition)
        self.arena = None
        self.arenas, self.streams = [], []
        cells = (CellEnv * K)()
        for k, dev in enumerate(self.devices):
            d = torch.device("cuda", dev)
            with torch.cuda.device(d):
                a = torch.empty(need[k] + 1024, dtype=torch.uint8, device=d)
                st = torch.cuda.Stream(device=d)
                torch.cuda.synchronize(d)
            self.arenas.append(a)
            self.streams.append(st)
            cells[k] = CellEnv(dev, (a.data_ptr() + 1023) // 1024 * 1024, need[k], st.cuda_stream)
        lo = (C.c_int32 * (K + 1))(*[int(v) for v in partition]) if partition is not None else None
        with torch.cuda.device(self.device):
            _check(lib().gpipe_create_pipeline(C.byref(self.spec), K, M, int(self.remat), n_seqs, cells, lo,
                                               PIPE_STAGED if staged else 0, C.byref(self._h)))

    def _create_single(self, torch, K, M, remat, n_seqs, partition):
        with torch.cuda.device(self.device):
            nbytes = plan_bytes(self.spec, K, M, remat, n_seqs)
            self.arena = torch.empty(nbytes + 1024, dtype=torch.uint8, device=self.device)
            base = (self.arena.data_ptr() + 1023) // 1024 * 1024
            ns = 2 * K if self.side_streams else K
            self._all_streams = [torch.cuda.Stream(device=self.device) for _ in range(ns)]
            self.streams = self._all_streams[:K]
            self._stream_arr = (C.c_void_p * ns)(*[s.cuda_stream for s in self._all_streams])
            env = Env(base, nbytes, C.cast(self._stream_arr, C.POINTER(C.c_void_p)), ns)
            torch.cuda.synchronize(self.device)
            if partition is None:
                _check(lib().gpipe_create(C.byref(self.spec), K, M, int(self.remat), n_seqs, C.byref(env),
                                          C.byref(self._h)))
            else:
                if isinstance(partition, str):
                    if partition != "cost":
                        raise ValueError("partition must be None, 'cost' or a list of K+1 boundaries")
                    costs, c_emb, c_head = layer_costs(self.spec, self.remat)
                    partition = partition_min_variance(costs, c_emb, c_head, K)
                lo = (C.c_int32 * (K + 1))(*[int(v) for v in partition])
                _check(lib().gpipe_create_partitioned(C.byref(self.spec), K, M, int(self.remat), n_seqs,
                                                      C.byref(env), lo, C.byref(self._h)))

    def _finish_init(self, K):
        self.cells = []
        for k in range(K):
            lo_k, hi_k = C.c_int32(0), C.c_int32(0)
            _check(lib().gpipe_cell_range(self._h, k, C.byref(lo_k), C.byref(hi_k)))
            self.cells.append((lo_k.value, hi_k.value))
        self.names: List[str] = []
        self.shapes: Dict[str, Tuple[int, int]] = {}
        for i in range(lib().gpipe_num_tensors(self._h)):
            nm, r, c = C.c_char_p(), C.c_int64(), C.c_int64()
            _check(lib().gpipe_tensor_info(self._h, i, C.byref(nm), C.byref(r), C.byref(c)))
            self.names.append(nm.value.decode())
            self.shapes[self.names[-1]] = (r.value, c.value)
        self._index = {n: i for i, n in enumerate(self.names)}

    # -- life cycle ---------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().gpipe_destroy(self._h)
            self._h = C.c_void_p(None)
        self.arena = None
        self.arenas = None
        self._slots = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- the three calls ------------------------------------------------------------------------
    def init_params(self, seed: int, std: float = 0.02, parity: bool = False, ffn_scale: float = 1.0):
        """ffn_scale: std multiplier of w_1 / w_2 (1 / n_layers for the depth-scaled initialisation)."""
        with self._torch.cuda.device(self.device):
            _check(lib().gpipe_init_params_scaled(self._h, seed, std, int(parity), ffn_scale))

    def step(self, tokens, labels) -> float:
        """tokens/labels: numpy int32 [N,S] or CPU torch tensors (host path, gpipe_step), or CUDA
        int32 tensors (inputs resident in HBM, gpipe_step_device).  Returns the mean loss."""
        torch = self._torch
        loss = C.c_float(0)
        with torch.cuda.device(self.device):
            if isinstance(tokens, torch.Tensor) and tokens.is_cuda:
                if tokens.dtype != torch.int32 or labels.dtype != torch.int32:
                    raise ValueError("device ids must be int32")
                t, l = tokens.contiguous(), labels.contiguous()
                if t.numel() != self.n_seqs * self.seq_len or l.numel() != t.numel():
                    raise ValueError("tokens/labels must be [n_seqs, seq_len]")
                torch.cuda.current_stream(self.device).synchronize()
                _check(lib().gpipe_step_device(self._h, t.data_ptr(), l.data_ptr(), C.byref(loss)))
            else:
                t = np.ascontiguousarray(tokens.numpy() if isinstance(tokens, torch.Tensor) else tokens, dtype=np.int32)
                l = np.ascontiguousarray(labels.numpy() if isinstance(labels, torch.Tensor) else labels, dtype=np.int32)
                if t.size != self.n_seqs * self.seq_len or l.size != t.size:
                    raise ValueError("tokens/labels must be [n_seqs, seq_len]")
                _check(lib().gpipe_step(self._h, t.ctypes.data, l.ctypes.data, C.byref(loss)))
        return float(loss.value)

    def apply_rmsprop(self, lr: float, rho: float = 0.9, eps: float = 1e-8):
        """RMSProp; the fp32 slot (4 B / parameter) is allocated on first use."""
        with self._torch.cuda.device(self.device):
            self._ensure_slots()
            _check(lib().gpipe_apply_rmsprop(self._h, lr, rho, eps))

    def _ensure_slots(self):
        if getattr(self, "_slots", None) is None and self.devices is not None:
            self._slots = []                                     # pipeline: each cell's slot shard on that cell's device
            for k, dev in enumerate(self.devices):
                n = C.c_int64(0)
                _check(lib().gpipe_cell_param_count(self._h, k, C.byref(n)))
                d = self._torch.device("cuda", dev)
                t = self._torch.empty(max(n.value, 1) * 4, dtype=self._torch.uint8, device=d)
                self._slots.append(t)
                with self._torch.cuda.device(self.device):
                    _check(lib().gpipe_attach_optimizer_slots_cell(self._h, k, t.data_ptr(), n.value * 4))
            return
        with self._torch.cuda.device(self.device):
            if getattr(self, "_slots", None) is None:
                n = C.c_size_t(0)
                _check(lib().gpipe_optimizer_slot_bytes(self._h, C.byref(n)))
                self._slots = self._torch.empty(n.value, dtype=self._torch.uint8, device=self.device)
                _check(lib().gpipe_attach_optimizer_slots(self._h, self._slots.data_ptr(), n.value))

    def apply_sgd(self, lr: float):
        with self._torch.cuda.device(self.device):
            _check(lib().gpipe_apply_sgd(self._h, lr))

    def zero_grads(self):
        with self._torch.cuda.device(self.device):
            _check(lib().gpipe_zero_grads(self._h))

    # -- data-parallel replicas ---------------------------------------------------
    @property
    def arena_base(self) -> int:
        """Device address of the (1024-byte aligned) arena this handle carved its memory from."""
        return (self.arena.data_ptr() + 1023) // 1024 * 1024

    def dp_layout(self) -> Dict[str, int]:
        n, mo, go, wo = C.c_int64(), C.c_size_t(), C.c_size_t(), C.c_size_t()
        _check(lib().gpipe_dp_layout(self._h, C.byref(n), C.byref(mo), C.byref(go), C.byref(wo)))
        return {"n_flat": n.value, "master_off": mo.value, "grad_off": go.value, "wlp_off": wo.value}

    def dp_apply_sgd(self, rank: int, peer_arenas: Sequence[int], lr: float, grad_scale: Optional[float] = None):
        """Fused cross-replica gradient sum + SGD + all-gather of the update for this replica's shard.
        peer_arenas[p]: device address of replica p's arena as seen from this process."""
        world = len(peer_arenas)
        arr = (C.c_void_p * world)(*[int(a) for a in peer_arenas])
        with self._torch.cuda.device(self.device):
            _check(lib().gpipe_dp_apply_sgd(self._h, rank, world, arr, lr, 1.0 / world if grad_scale is None else grad_scale))

    def dp_apply_rmsprop(self, rank: int, peer_arenas: Sequence[int], lr: float, rho: float = 0.9, eps: float = 1e-8,
                         grad_scale: Optional[float] = None):
        world = len(peer_arenas)
        arr = (C.c_void_p * world)(*[int(a) for a in peer_arenas])
        with self._torch.cuda.device(self.device):
            self._ensure_slots()
            _check(lib().gpipe_dp_apply_rmsprop(self._h, rank, world, arr, lr, rho, eps,
                                                1.0 / world if grad_scale is None else grad_scale))

    # -- parameters -----------------------------------------------------------------------------
    def _idx(self, key) -> int:
        return key if isinstance(key, int) else self._index[key]

    def _get(self, fn, key) -> np.ndarray:
        i = self._idx(key)
        out = np.empty(self.shapes[self.names[i]], np.float32)
        with self._torch.cuda.device(self.device):
            _check(fn(self._h, i, out.ctypes.data))
        return out

    def get_param(self, key) -> np.ndarray:
        return self._get(lib().gpipe_get_param, key)

    def get_grad(self, key) -> np.ndarray:
        return self._get(lib().gpipe_get_grad, key)

    def get_master(self, key) -> np.ndarray:
        """fp32 master copy, every bit (checkpointing)."""
        return self._get(lib().gpipe_get_master, key)

    def get_optimizer_slot(self, key) -> np.ndarray:
        return self._get(lib().gpipe_get_optimizer_slot, key)

    def _set(self, fn, key, value):
        i = self._idx(key)
        a = np.ascontiguousarray(value, dtype=np.float32)
        if a.size != self.shapes[self.names[i]][0] * self.shapes[self.names[i]][1]:
            raise ValueError("wrong size for %s" % self.names[i])
        with self._torch.cuda.device(self.device):
            _check(fn(self._h, i, a.ctypes.data))

    def set_master(self, key, value):
        self._set(lib().gpipe_set_master, key, value)

    def set_optimizer_slot(self, key, value):
        self._ensure_slots()
        self._set(lib().gpipe_set_optimizer_slot, key, value)

    def state_dict(self) -> Dict[str, Dict[str, np.ndarray]]:
        """Exact training state: fp32 masters (+ RMSProp slots once they exist)."""
        out = {"master": {n: self.get_master(n) for n in self.names}}
        if getattr(self, "_slots", None) is not None:
            out["slot"] = {n: self.get_optimizer_slot(n) for n in self.names}
        return out

    def load_state_dict(self, state):
        for n in self.names:
            self.set_master(n, state["master"][n])
        if "slot" in state:
            for n in self.names:
                self.set_optimizer_slot(n, state["slot"][n])

    def set_param(self, key, value):
        i = self._idx(key)
        a = np.ascontiguousarray(value, dtype=np.float32)
        if a.size != self.shapes[self.names[i]][0] * self.shapes[self.names[i]][1]:
            raise ValueError("wrong size for %s" % self.names[i])
        with self._torch.cuda.device(self.device):
            _check(lib().gpipe_set_param(self._h, i, a.ctypes.data))

    def set_params(self, params: Dict[str, np.ndarray]):
        for n in self.names:
            self.set_param(n, params[n])

    def grads(self) -> Dict[str, np.ndarray]:
        return {n: self.get_grad(n) for n in self.names}

    # -- tracker / trace --------------------------------------------------------------------------
    def peak_bytes(self) -> Dict[str, object]:
        total = C.c_size_t(0)
        cats = (C.c_size_t * len(CATEGORIES))()
        cells = (C.c_size_t * self.K)()
        _check(lib().gpipe_peak_bytes(self._h, C.byref(total), cats, cells))
        return {"total": int(total.value), "by_category": {c: int(cats[i]) for i, c in enumerate(CATEGORIES)},
                "by_cell": [int(cells[k]) for k in range(self.K)]}

    def trace(self, enable: bool):
        _check(lib().gpipe_trace(self._h, int(enable), None, None))

    def trace_events(self) -> List[Tuple[str, int, int, int, float, float]]:
        n = C.c_int64(0)
        _check(lib().gpipe_trace(self._h, 1, None, C.byref(n)))
        buf = (TraceEvent * max(n.value, 1))()
        _check(lib().gpipe_trace(self._h, 1, buf, C.byref(n)))
        return [(chr(e.kind), e.k, e.m, e.enqueue_index, e.start_ms, e.end_ms) for e in buf[:n.value]]

    def kernel_timing(self, enable: bool, serial: bool = False):
        """Per-launch CUDA-event timing; serial=True also runs every cell on stream 0."""
        _check(lib().gpipe_kernel_timing(self._h, (1 if enable else 0) | (2 if serial else 0)))

    def kernel_stats(self) -> Dict[str, Dict[str, float]]:
        out = {}
        for cls in range(10):
            nm, cnt = C.c_char_p(), C.c_int64()
            ms, fl, by = C.c_double(), C.c_double(), C.c_double()
            _check(lib().gpipe_kernel_stats(self._h, cls, C.byref(nm), C.byref(cnt), C.byref(ms), C.byref(fl), C.byref(by)))
            out[nm.value.decode()] = {"launches": cnt.value, "ms": ms.value, "flops": fl.value, "bytes": by.value}
        return out

    def cuda_graph(self, enable: bool):
        """Replay the step as one CUDA graph (default on) or enqueue it eagerly."""
        _check(lib().gpipe_cuda_graph(self._h, int(enable)))

    def cuda_graph_state(self) -> int:
        return int(lib().gpipe_cuda_graph_state(self._h))

    def launch_count(self) -> int:
        return int(lib().gpipe_launch_count(self._h))

    def debug_read(self, what: str, layer: int = -1, max_elems: Optional[int] = None) -> np.ndarray:
        if max_elems is None:
            T_mb = self.n_seqs // self.M * self.seq_len
            s = self.spec
            da = s.n_heads * (s.d_head or s.d_model // s.n_heads)
            max_elems = T_mb * max(s.vocab, s.d_ffn, 3 * da, s.d_model)
        out = np.empty(max_elems, np.float32)
        n = C.c_int64(0)
        with self._torch.cuda.device(self.device):
            self._torch.cuda.synchronize(self.device)
            _check(lib().gpipe_debug_read(self._h, what.encode(), layer, out.ctypes.data, max_elems, C.byref(n)))
        return out[:n.value].copy()


class GPipeEncDec(GPipe):
    """The encoder-decoder Transformer T(L,H,A) of PAPER.md:160 on the same schedule (gpipe_create_encdec /
    gpipe_step_encdec): n_enc encoder layers, then n_dec decoder layers with cross-attention over the
    encoder memory, cut into K cells of consecutive layers.  partition: None or K+1 boundaries over the n_enc + n_dec
    layers.  logit_clip: PAPER.md:174 (0 = off)."""

    def __init__(self, *, n_enc, n_dec, d_model, d_ffn, n_heads, d_head, vocab, seq_len, dtype, K, M, remat=True,
                 n_seqs, ln_eps=1e-5, logit_clip=0.0, device="cuda:0", partition=None, devices=None, staged=False,
                 side_streams=None):
        import torch
        if not torch.cuda.is_available():
            raise GPipeError(-2, "no CUDA device: the GPipe path has no CPU fallback")
        self._torch = torch
        self.device = torch.device(device)
        dt = {"fp32": DTYPE_FP32, "bf16": DTYPE_BF16, 0: 0, 1: 1}[dtype]
        self.spec = EncDecSpec(n_enc, n_dec, d_model, d_ffn, n_heads, d_head, vocab, seq_len, dt, ln_eps, logit_clip)
        self.K, self.M, self.remat, self.n_seqs, self.seq_len = K, M, bool(remat), n_seqs, seq_len
        self._h = C.c_void_p(None)
        self.devices = None if devices is None else [int(d) for d in devices]
        self.side_streams = (K <= 2 if side_streams is None else bool(side_streams)) and devices is None
        if isinstance(partition, str):
            if partition != "cost":
                raise ValueError("partition must be None, 'cost' or a list of K+1 boundaries")
            costs, c_emb, c_head = layer_costs_encdec(self.spec, self.remat)
            partition = partition_min_variance(costs, c_emb, c_head, K)
        lo = (C.c_int32 * (K + 1))(*[int(v) for v in partition]) if partition is not None else None
        if self.devices is not None:                       # gpipe_create_pipeline_encdec: one arena / stream / device per cell
            if len(self.devices) != K:
                raise ValueError("devices must list one CUDA device per cell")
            self.device = torch.device("cuda", self.devices[0])
            need = (C.c_size_t * K)()
            _check(lib().gpipe_plan_bytes_pipeline_encdec(C.byref(self.spec), K, M, int(self.remat), n_seqs, lo, need))
            self.arena, self.arenas, self.streams = None, [], []
            cells = (CellEnv * K)()
            for k, dev in enumerate(self.devices):
                d = torch.device("cuda", dev)
                with torch.cuda.device(d):
                    a = torch.empty(int(need[k]) + 1024, dtype=torch.uint8, device=d)
                    st = torch.cuda.Stream(device=d)
                    torch.cuda.synchronize(d)
                self.arenas.append(a)
                self.streams.append(st)
                cells[k] = CellEnv(dev, (a.data_ptr() + 1023) // 1024 * 1024, int(need[k]), st.cuda_stream)
            with torch.cuda.device(self.device):
                _check(lib().gpipe_create_pipeline_encdec(C.byref(self.spec), K, M, int(self.remat), n_seqs, cells, lo,
                                                          PIPE_STAGED if staged else 0, C.byref(self._h)))
            self._finish_init(K)
            return
        with torch.cuda.device(self.device):
            nbytes = plan_bytes_encdec(self.spec, K, M, remat, n_seqs, partition)
            self.arena = torch.empty(nbytes + 1024, dtype=torch.uint8, device=self.device)
            base = (self.arena.data_ptr() + 1023) // 1024 * 1024
            ns = 2 * K if self.side_streams else K
            self._all_streams = [torch.cuda.Stream(device=self.device) for _ in range(ns)]
            self.streams = self._all_streams[:K]
            self._stream_arr = (C.c_void_p * ns)(*[s.cuda_stream for s in self._all_streams])
            env = Env(base, nbytes, C.cast(self._stream_arr, C.POINTER(C.c_void_p)), ns)
            torch.cuda.synchronize(self.device)
            _check(lib().gpipe_create_encdec(C.byref(self.spec), K, M, int(self.remat), n_seqs, C.byref(env), lo,
                                             C.byref(self._h)))
        self._finish_init(K)

    def step(self, src, tgt, labels) -> float:
        """src / tgt / labels: numpy int32 [N,S] or CPU tensors (gpipe_step_encdec), or CUDA int32 tensors
        (gpipe_step_encdec_device).  Returns the mean loss."""
        torch = self._torch
        loss = C.c_float(0)
        n = self.n_seqs * self.seq_len
        with torch.cuda.device(self.device):
            if isinstance(src, torch.Tensor) and src.is_cuda:
                ts = [t.contiguous() for t in (src, tgt, labels)]
                if any(t.dtype != torch.int32 or t.numel() != n for t in ts):
                    raise ValueError("device ids must be int32 [n_seqs, seq_len]")
                torch.cuda.current_stream(self.device).synchronize()
                _check(lib().gpipe_step_encdec_device(self._h, ts[0].data_ptr(), ts[1].data_ptr(), ts[2].data_ptr(),
                                                      C.byref(loss)))
            else:
                hs = [np.ascontiguousarray(t.numpy() if isinstance(t, torch.Tensor) else t, dtype=np.int32)
                      for t in (src, tgt, labels)]
                if any(h.size != n for h in hs):
                    raise ValueError("src/tgt/labels must be [n_seqs, seq_len]")
                _check(lib().gpipe_step_encdec(self._h, hs[0].ctypes.data, hs[1].ctypes.data, hs[2].ctypes.data,
                                               C.byref(loss)))
        return float(loss.value)

    def debug_read(self, *a, **kw):
        raise GPipeError(-4, "debug taps are not built for the encoder-decoder handle")

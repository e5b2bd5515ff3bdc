"""Thin wrappers of the per-kernel C entry points (include/gpipe_ops.h) on torch CUDA tensors.
Marshalling only: pointers, sizes and the current stream are passed to the library."""
from __future__ import annotations

from typing import Optional

from . import binding as B


def _torch():
    import torch
    return torch


def _dt(t) -> int:
    torch = _torch()
    if t.dtype == torch.bfloat16:
        return B.DTYPE_BF16
    if t.dtype == torch.float32:
        return B.DTYPE_FP32
    raise ValueError("lp tensors must be float32 or bfloat16")


def _p(t):
    return None if t is None else t.data_ptr()


def _stream():
    return _torch().cuda.current_stream().cuda_stream


def gemm(A, B_, C, *, transA=False, transB=False, bias=None, resid=None, mask=None, relu=False,
         accumulate=False, colsum_out=None, bits_out=None, workspace=None, backend=0):
    """C = epilogue(op(A) @ op(B)); shapes follow gpipe_op_gemm.  C is written in place.
    mask / bits_out: int32 [M, N/32] bit-packed ReLU pattern (read / written).
    workspace: None -> a zeroed split-K workspace is allocated when the shape wants one; False -> never
    split; or a uint8 tensor from gemm_workspace() that this stream reuses."""
    torch = _torch()
    M, N = C.shape
    K = A.shape[0] if transA else A.shape[1]
    flags = 0
    if bias is not None: flags |= B.EPI_BIAS
    if relu: flags |= B.EPI_RELU
    if mask is not None: flags |= B.EPI_MASK
    if bits_out is not None:
        assert mask is None
        flags |= B.EPI_BITS_OUT
        mask = bits_out
    if resid is not None: flags |= B.EPI_RESID
    if accumulate: flags |= B.EPI_ACCUM
    if C.dtype == torch.float32: flags |= B.EPI_OUT_F32
    scratch = None
    if colsum_out is not None:
        flags |= B.EPI_COLSUM
        scratch = torch.empty(B.lib().gpipe_op_colsum_scratch_floats(M, N), dtype=torch.float32, device=C.device)
    if workspace is None:
        workspace = gemm_workspace(M, N, K, C.device)
    elif workspace is False:
        workspace = None
    B._check(B.lib().gpipe_op_gemm(_stream(), _dt(A), M, N, K, _p(A), A.stride(0), int(transA), _p(B_),
                                   B_.stride(0), int(transB), _p(C), C.stride(0), _p(bias), _p(resid),
                                   _p(mask), mask.stride(0) if mask is not None else 0, _p(colsum_out),
                                   _p(scratch), _p(workspace), workspace.numel() if workspace is not None else 0,
                                   flags, backend))
    return C


def gemm_workspace(M, N, K, device):
    """Zeroed split-K workspace for a [M,N,K] GEMM (None when the shape is not split)."""
    n = B.lib().gpipe_op_gemm_workspace_bytes(M, N, K)
    return _torch().zeros(n, dtype=_torch().uint8, device=device) if n > 0 else None


def ln_fwd(x, gamma, beta, y, mean, rstd, eps=1e-5, resid_bias=None, resid_out=None):
    """resid_out (optional fp32 [n,d]) = x + resid_bias: the buffer the branch's output GEMM accumulates into."""
    n, d = x.shape
    B._check(B.lib().gpipe_op_ln_fwd(_stream(), _dt(y), _p(x), _p(gamma), _p(beta), _p(y), _p(mean), _p(rstd),
                                     _p(resid_bias), _p(resid_out), n, d, eps))


def ln_bwd(dy, x, mean, rstd, gamma, dres_in, dx_out, dx_out_lp, dgamma, dbeta, colsum_out=None):
    torch = _torch()
    n, d = x.shape
    scratch = torch.empty(B.lib().gpipe_op_ln_bwd_scratch_floats(d), dtype=torch.float32, device=x.device)
    B._check(B.lib().gpipe_op_ln_bwd(_stream(), _dt(dy), _p(dy), _p(x), _p(mean), _p(rstd), _p(gamma), _p(dres_in),
                                     _p(dx_out), _p(dx_out_lp), _p(scratch), _p(dgamma), _p(dbeta), _p(colsum_out), n, d))
    return scratch


def attn_fwd(qkv, o, lse, n_seq, S, A, dh, causal, backend=0):
    B._check(B.lib().gpipe_op_attn_fwd(_stream(), _dt(qkv), _p(qkv), _p(o), _p(lse), n_seq, S, A, dh, int(causal), backend))


def attn_bwd(qkv, o, d_o, lse, dqkv, dvec, n_seq, S, A, dh, causal, backend=0, colpart=None):
    B._check(B.lib().gpipe_op_attn_bwd(_stream(), _dt(qkv), _p(qkv), _p(o), _p(d_o), _p(lse), _p(dqkv), _p(dvec),
                                       n_seq, S, A, dh, int(causal), backend, _p(colpart)))


def softmax_ce(logits, labels, rowloss, inv_T, clip=0.0):
    n, V = logits.shape
    B._check(B.lib().gpipe_op_softmax_ce(_stream(), _dt(logits), _p(logits), _p(labels), _p(rowloss), n, V, inv_T, clip))


def colsum(dy, out):
    torch = _torch()
    n, c = dy.shape
    scratch = torch.empty(B.lib().gpipe_op_colsum_scratch_floats(n, c), dtype=torch.float32, device=dy.device)
    B._check(B.lib().gpipe_op_colsum(_stream(), _dt(dy), _p(dy), dy.stride(0), _p(out), _p(scratch), n, c))


COLSUM_STATIC_MAX_N = 16384


def colsum_static(dy, out):
    """out[n] += sum_t dy[t, n] through gpipe_op_colsum_static: no device allocation anywhere (the scratch is a static
    array inside the library); at most COLSUM_STATIC_MAX_N columns; calls that overlap on the GPU race on it."""
    n, c = dy.shape
    B._check(B.lib().gpipe_op_colsum_static(_stream(), _dt(dy), _p(dy), dy.stride(0), _p(out), n, c))


def embed_fwd(tok, emb, pe, x, S):
    n, d = x.shape
    B._check(B.lib().gpipe_op_embed_fwd(_stream(), _dt(emb), _p(tok), _p(emb), _p(pe), _p(x), n, S, d))


def embed_bwd(tok, dx, gemb):
    n, d = dx.shape
    B._check(B.lib().gpipe_op_embed_bwd(_stream(), _p(tok), _p(dx), _p(gemb), n, d))


def positional(pe):
    S, d = pe.shape
    B._check(B.lib().gpipe_op_positional(_stream(), _p(pe), S, d))


def sgd(master, grad, w_lp, lr):
    B._check(B.lib().gpipe_op_sgd(_stream(), B.DTYPE_BF16 if w_lp is not None else B.DTYPE_FP32, _p(master), _p(grad),
                                  _p(w_lp), master.numel(), lr))


def rmsprop(master, grad, ms, w_lp, lr, rho, eps):
    B._check(B.lib().gpipe_op_rmsprop(_stream(), B.DTYPE_BF16 if w_lp is not None else B.DTYPE_FP32, _p(master), _p(grad),
                                      _p(ms), _p(w_lp), master.numel(), lr, rho, eps))


def dp_apply_sgd(masters, grads, w_lps, rank, lr, grad_scale=None):
    """Fused data-parallel apply on raw arrays: masters / grads / w_lps are lists (one entry per replica)."""
    import ctypes as C
    world = len(masters)
    arr = lambda ts: (C.c_void_p * world)(*[t.data_ptr() for t in ts])
    B._check(B.lib().gpipe_op_dp_apply_sgd(_stream(), B.DTYPE_BF16 if w_lps is not None else B.DTYPE_FP32, world, rank,
                                           arr(masters), arr(grads), arr(w_lps) if w_lps is not None else None,
                                           masters[0].numel(), lr, 1.0 / world if grad_scale is None else grad_scale))

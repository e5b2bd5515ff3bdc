"""Per-kernel ("teacher-forced") parity: each CUDA kernel, called through the C ABI of
include/gpipe_ops.h, against the oracle's operator on identical inputs.  fp32 kernels must agree to
fp32 rounding; bf16 kernels get bf16-representable inputs and must agree to output rounding
(<= 2^-7 max-rel, cosine >= 0.99999)."""
import math

import numpy as np
import pytest
import torch

import gpipe_inputs as gi
from oracle import gpipe_oracle as go
from paper_1811_06965_b200 import ops
from tests.util import cosine, maxrel

pytestmark = pytest.mark.gpu

DEV = "cuda"


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _lp(a, dtype):
    """host fp array -> device lp tensor and the exact fp64 values it holds"""
    if dtype == "bf16":
        a = gi.bf16_round(a.astype(np.float32))
        return torch.tensor(a, device=DEV).to(torch.bfloat16), a.astype(np.float64)
    a = a.astype(np.float32)
    return torch.tensor(a, device=DEV), a.astype(np.float64)


def _np(t):
    return t.detach().float().cpu().numpy().astype(np.float64)


def _tol(dtype):
    return (2e-5, 0.9999999) if dtype == "fp32" else (2 ** -7, 0.99999)


# -------------------------------------------------------------------------------------------------
# GEMM
# -------------------------------------------------------------------------------------------------
GEMM_SHAPES = [(32, 64, 48), (70, 130, 33), (128, 128, 64), (256, 192, 128), (1, 8, 8)]


@pytest.mark.parametrize("dtype", ["fp32", "bf16"])
@pytest.mark.parametrize("transA,transB", [(0, 0), (0, 1), (1, 0), (1, 1)])
def test_gemm_simt_all_layouts(dtype, transA, transB):
    for (M, N, K) in GEMM_SHAPES:
        r = _rng(M * 1000 + N + K)
        A = r.standard_normal((K, M) if transA else (M, K))
        B = r.standard_normal((N, K) if transB else (K, N))
        At, Aq = _lp(A, dtype)
        Bt, Bq = _lp(B, dtype)
        C = torch.empty((M, N), device=DEV, dtype=At.dtype)
        ops.gemm(At, Bt, C, transA=bool(transA), transB=bool(transB), backend=1)
        ref = (Aq.T if transA else Aq) @ (Bq.T if transB else Bq)
        tol, cos = _tol(dtype)
        assert maxrel(_np(C), ref) <= tol, (M, N, K)
        assert cosine(_np(C), ref) >= cos


# tensor-core path: shapes spanning several 256 x 256 pair tiles, a ragged tail in M, N and K, more
# k-blocks than pipeline stages, and small shapes that take the 1-CTA kernel
TC_SHAPES = [(512, 768, 320), (304, 520, 200), (1024, 256, 1088), (128, 136, 72), (264, 1032, 64)]


@pytest.mark.parametrize("transA,transB", [(0, 0), (0, 1), (1, 0), (1, 1)])
def test_gemm_tcgen05_all_layouts(transA, transB):
    for (M, N, K) in TC_SHAPES:
        r = _rng(M * 1000 + N + K)
        At, Aq = _lp(r.standard_normal((K, M) if transA else (M, K)), "bf16")
        Bt, Bq = _lp(r.standard_normal((N, K) if transB else (K, N)), "bf16")
        ref = (Aq.T if transA else Aq) @ (Bq.T if transB else Bq)
        Cf = torch.empty((M, N), device=DEV, dtype=torch.float32)
        ops.gemm(At, Bt, Cf, transA=bool(transA), transB=bool(transB), backend=2)
        assert maxrel(_np(Cf), ref) <= 2e-5, (M, N, K)          # fp32 accumulation of exact bf16 products
        C = torch.empty((M, N), device=DEV, dtype=torch.bfloat16)
        ops.gemm(At, Bt, C, transA=bool(transA), transB=bool(transB), backend=2)
        assert maxrel(_np(C), ref) <= 2 ** -7 and cosine(_np(C), ref) >= 0.99999, (M, N, K)


# 256 x 512 pair tiles (backend 4; backend 3 = 256 x 256 only): several tiles, ragged tails in M, N (a half-empty last
# tile, N % 32 != 0) and K, fewer and more K-blocks than the 4 ring stages, one K-block
WIDE_SHAPES = [(512, 1024, 320), (304, 520, 200), (1024, 512, 1088), (264, 1032, 64), (256, 512, 64), (2048, 2048, 1024),
               (704, 1536, 4160), (136, 3072, 2048)]


@pytest.mark.parametrize("transA,transB", [(0, 0), (0, 1), (1, 0), (1, 1)])
@pytest.mark.parametrize("epi", ["plain", "accum", "bias_relu_bits"])
def test_gemm_tcgen05_wide_tile(transA, transB, epi):
    """The 256 x 512 pair tile (one accumulator in all 512 TMEM columns, two MMAs per K step, accumulator blocks that
    interleave the two CTAs' B halves) against the fp64 product of the same operands, and bit for bit against the
    256 x 256 tile: every output is the same chain of MMAs over K in the same order."""
    for (M, N, K) in WIDE_SHAPES:
        if epi == "bias_relu_bits" and N % 32:
            continue
        r = _rng(M * 1000 + N + K + 7)
        At, Aq = _lp(r.standard_normal((K, M) if transA else (M, K)) * 0.5, "bf16")
        Bt, Bq = _lp(r.standard_normal((N, K) if transB else (K, N)) * 0.5, "bf16")
        ref = (Aq.T if transA else Aq) @ (Bq.T if transB else Bq)
        kw = dict(transA=bool(transA), transB=bool(transB), workspace=False)
        c0 = r.standard_normal((M, N)).astype(np.float32)
        bias = r.standard_normal(N).astype(np.float32)
        out = {}
        for backend in (3, 4):
            if epi == "plain":
                C = torch.empty((M, N), device=DEV, dtype=torch.bfloat16)
                ops.gemm(At, Bt, C, backend=backend, **kw)
                out[backend] = (C,)
                if backend == 4:
                    assert maxrel(_np(C), ref) <= 2 ** -7 and cosine(_np(C), ref) >= 0.99999, (M, N, K)
            elif epi == "accum":
                C = torch.tensor(c0, device=DEV)
                ops.gemm(At, Bt, C, accumulate=True, backend=backend, **kw)
                ops.gemm(At, Bt, C, accumulate=True, backend=backend, **kw)
                out[backend] = (C,)
                if backend == 4:
                    assert maxrel(_np(C), c0 + 2 * ref) <= 2e-5, (M, N, K)
            else:
                C = torch.empty((M, N), device=DEV, dtype=torch.bfloat16)
                bits = torch.zeros((M, N // 32), device=DEV, dtype=torch.int32)
                ops.gemm(At, Bt, C, bias=torch.tensor(bias, device=DEV), relu=True, bits_out=bits, backend=backend, **kw)
                out[backend] = (C, bits)
                if backend == 4:
                    want = np.maximum(ref + bias, 0)
                    assert maxrel(_np(C), want) <= 2 ** -7 and cosine(_np(C), want) >= 0.99999, (M, N, K)
                    assert np.array_equal(_unpack_mask(bits, M, N), _np(C) > 0)
        for a, b in zip(out[3], out[4]):
            assert torch.equal(a, b), (M, N, K, epi)


def test_gemm_tcgen05_wide_tile_refuses_what_it_cannot_take():
    """backend 4 never silently runs another kernel: N < 512 and the epilogues without a 256 x 512 instantiation
    (bias alone, the ReLU-masked dgrad with column sums) are GPIPE_EINVAL."""
    r = _rng(5)
    At, _ = _lp(r.standard_normal((256, 128)), "bf16")
    Bt, _ = _lp(r.standard_normal((128, 256)), "bf16")
    C = torch.empty((256, 256), device=DEV, dtype=torch.bfloat16)
    from paper_1811_06965_b200 import GPipeError
    with pytest.raises(GPipeError):
        ops.gemm(At, Bt, C, backend=4)
    Bt, _ = _lp(r.standard_normal((128, 1024)), "bf16")
    C = torch.empty((256, 1024), device=DEV, dtype=torch.bfloat16)
    with pytest.raises(GPipeError):
        ops.gemm(At, Bt, C, bias=torch.zeros(1024, device=DEV), backend=4)
    ops.gemm(At, Bt, C, backend=4)


def test_gemm_bf16_never_falls_back_silently():
    """A bf16 problem the tcgen05 kernel cannot take (row pitch not a multiple of 16 bytes; a ReLU pattern with
    N % 32 != 0) is GPIPE_EINVAL on the default backend, not a ~50x slower SIMT launch; backend 1 still runs it."""
    from paper_1811_06965_b200 import GPipeError
    r = _rng(9)
    At, Aq = _lp(r.standard_normal((64, 36)), "bf16")        # lda = 36: 72-byte row pitch
    Bt, Bq = _lp(r.standard_normal((36, 64)), "bf16")
    C = torch.empty((64, 64), device=DEV, dtype=torch.bfloat16)
    with pytest.raises(GPipeError) as err:
        ops.gemm(At, Bt, C)
    assert err.value.code == -1
    ops.gemm(At, Bt, C, backend=1)
    assert maxrel(_np(C), Aq @ Bq) <= 2 ** -7
    A2, _ = _lp(r.standard_normal((64, 64)), "bf16")
    B2, _ = _lp(r.standard_normal((64, 48)), "bf16")
    C2 = torch.empty((64, 48), device=DEV, dtype=torch.bfloat16)
    bits = torch.zeros((64, 2), device=DEV, dtype=torch.int32)
    with pytest.raises(GPipeError):
        ops.gemm(A2, B2, C2, relu=True, bits_out=bits)


@pytest.mark.parametrize("dtype,T,d,da", [("fp32", 300, 192, 128), ("bf16", 300, 192, 128), ("bf16", 2048, 1024, 2048)],
                         ids=["fp32-small", "bf16-small", "bf16-config5-microbatch"])
def test_gemm_on_column_views_of_a_packed_buffer(dtype, T, d, da):
    """The cross-attention block of a decoder layer packs q2 | k2 | v2 side by side in ONE [T, 3 da]
    buffer so that the self-attention kernels serve it: GEMMs write column blocks of it (ldc = 3 da), read column
    blocks of its gradient as A (lda = 3 da, dgrad) and as B (ldb = 3 da, wgrad), the memory gradient accumulates in
    fp32 on top of another buffer (EPI_RESID, then EPI_ACCUM), column sums run over a block.  Every launch must touch
    exactly its block: the rest of the buffer is filled with a sentinel and checked bit for bit.  Small case: ragged T
    (two 256-row tiles, the second one partial); large case: the launches of one T(64,16384,32) decoder layer and
    micro-batch (T_mb 2048, d 1024, d_a 2048), compared in full."""
    r = _rng(77)
    lp = torch.bfloat16 if dtype == "bf16" else torch.float32
    tol, cos = _tol(dtype)
    cxt, cxq = _lp(r.standard_normal((T, d)) * 0.5, dtype)
    memt, memq = _lp(r.standard_normal((T, d)) * 0.5, dtype)
    wqt, wqq = _lp(r.standard_normal((d, da)) * 0.1, dtype)
    wkvt, wkvq = _lp(r.standard_normal((d, 2 * da)) * 0.1, dtype)
    bq = torch.tensor(r.standard_normal(da).astype(np.float32), device=DEV)
    bkv = torch.tensor(r.standard_normal(2 * da).astype(np.float32), device=DEV)
    SENT = 7.0
    qkv2 = torch.full((T, 3 * da), SENT, device=DEV, dtype=lp)
    ops.gemm(cxt, wqt, qkv2[:, :da], bias=bq)                 # q2 = cx W_q + b_q -> columns [0, da)
    assert torch.equal(qkv2[:, da:], torch.full((T, 2 * da), SENT, device=DEV, dtype=lp))
    assert maxrel(_np(qkv2[:, :da]), cxq @ wqq + _np(bq)) <= tol
    ops.gemm(memt, wkvt, qkv2[:, da:], bias=bkv)              # k2 | v2 = mem W_kv + b_kv -> columns [da, 3 da)
    assert maxrel(_np(qkv2[:, :da]), cxq @ wqq + _np(bq)) <= tol          # the first block is still there
    assert maxrel(_np(qkv2[:, da:]), memq @ wkvq + _np(bkv)) <= tol
    # backward: the gradient buffer in the same layout
    dqt, dqq = _lp(r.standard_normal((T, 3 * da)) * 0.3, dtype)
    dcx = torch.full((T, d), SENT, device=DEV, dtype=lp)
    ops.gemm(dqt[:, :da], wqt, dcx, transB=True)              # dcx = dq2 W_q^T            (A view, lda = 3 da)
    assert maxrel(_np(dcx), dqq[:, :da] @ wqq.T) <= tol
    gq = torch.tensor(r.standard_normal((d, da)).astype(np.float32), device=DEV)
    gq0 = _np(gq)
    ops.gemm(cxt, dqt[:, :da], gq, transA=True, accumulate=True)          # dW_q += cx^T dq2   (B view, ldb = 3 da)
    assert maxrel(_np(gq), gq0 + cxq.T @ dqq[:, :da]) <= 2e-5 * (1 if dtype == "bf16" else 5)
    gkv = torch.zeros((d, 2 * da), device=DEV)
    ops.gemm(memt, dqt[:, da:], gkv, transA=True, accumulate=True)        # dW_kv += mem^T dkv
    assert maxrel(_np(gkv), memq.T @ dqq[:, da:]) <= 2e-5 * (1 if dtype == "bf16" else 5)
    # memory gradient: first decoder layer of a cell adds to what the next cell handed down, later layers accumulate
    handed = torch.tensor(r.standard_normal((T, d)).astype(np.float32), device=DEV)
    dmem = torch.full((T, d), SENT, device=DEV)
    ops.gemm(dqt[:, da:], wkvt, dmem, transB=True, resid=handed)
    ref = _np(handed) + dqq[:, da:] @ wkvq.T
    assert maxrel(_np(dmem), ref) <= 2e-5 * (1 if dtype == "bf16" else 5)
    ops.gemm(dqt[:, da:], wkvt, dmem, transB=True, accumulate=True)
    assert maxrel(_np(dmem), ref + dqq[:, da:] @ wkvq.T) <= 2e-5 * (1 if dtype == "bf16" else 5)
    # bias gradients over the two blocks
    dbq, dbkv = torch.zeros(da, device=DEV), torch.zeros(2 * da, device=DEV)
    ops.colsum(dqt[:, :da], dbq)
    ops.colsum(dqt[:, da:], dbkv)
    assert maxrel(_np(dbq), dqq[:, :da].sum(0)) <= 2e-5 and maxrel(_np(dbkv), dqq[:, da:].sum(0)) <= 2e-5


def test_gemm_tcgen05_split_k_deep():
    """Few output tiles and a very deep K (the dlogits W_out^T shape class): the launch is split along K,
    partials are reduced in split order, so two runs are bitwise equal and match the unsplit result."""
    r = _rng(123)
    M, N, K = 300, 256, 2 * 192 * 64 + 40                # 2 tiles, 385 K-blocks -> 2 splits, ragged tail
    ws = ops.gemm_workspace(M, N, K, DEV)
    assert ws is not None and ws.numel() > 0, "shape no longer split: pick a deeper K"
    At, Aq = _lp(r.standard_normal((M, K)), "bf16")
    Bt, Bq = _lp(r.standard_normal((N, K)), "bf16")
    ref = Aq @ Bq.T
    bias = torch.tensor(r.standard_normal(N).astype(np.float32), device=DEV)
    C1 = torch.empty((M, N), device=DEV)
    C2 = torch.empty((M, N), device=DEV)
    C0 = torch.empty((M, N), device=DEV)
    ops.gemm(At, Bt, C1, transB=True, bias=bias, workspace=ws, backend=2)
    ops.gemm(At, Bt, C2, transB=True, bias=bias, workspace=ws, backend=2)      # counters reset themselves
    ops.gemm(At, Bt, C0, transB=True, bias=bias, workspace=False, backend=2)   # never split
    assert torch.equal(C1, C2)
    assert maxrel(_np(C1), ref + _np(bias)[None, :]) <= 2e-5
    assert maxrel(_np(C0), ref + _np(bias)[None, :]) <= 1e-4       # one 24 616-deep fp32 accumulation chain
    assert maxrel(_np(C1), _np(C0)) <= 1e-4


def _pack_mask(maskq):
    M, N = maskq.shape
    return torch.tensor(np.packbits(maskq.reshape(M, N // 32, 32), axis=-1, bitorder="little")
                        .view(np.uint32).reshape(M, N // 32).view(np.int32), device=DEV)


def _unpack_mask(bits, M, N):
    return np.unpackbits(bits.cpu().numpy().view(np.uint8).reshape(M, N // 8), axis=-1, bitorder="little").astype(bool)


# Every GEMM launch of one layer + head of the bench workload T(64,16384,32) (T_mb = 2048, d = 1024, d_a = 2048,
# H = 16384, V = 64000), in the compile-time epilogue instantiation engine.cu launches it with:
#   name, M, N, K, transA, transB, epilogue
BENCH_GEMMS = [
    ("qkv_fwd", 2048, 6144, 1024, 0, 0, "bias"),
    ("oproj_fwd", 2048, 1024, 2048, 0, 0, "accum"),
    ("ffn1_fwd", 2048, 16384, 1024, 0, 0, "bias_relu_bits"),
    ("ffn2_fwd", 2048, 1024, 16384, 0, 0, "accum"),
    ("logits_fwd", 2048, 64000, 1024, 0, 0, "plain"),
    ("ffn2_dgrad", 2048, 16384, 1024, 0, 1, "mask_colsum"),
    ("ffn1_dgrad", 2048, 1024, 16384, 0, 1, "plain"),
    ("oproj_dgrad", 2048, 2048, 1024, 0, 1, "plain"),
    ("qkv_dgrad", 2048, 1024, 6144, 0, 1, "plain"),
    ("logits_dgrad", 2048, 1024, 64000, 0, 1, "plain"),
    ("logits_dgrad_unsplit", 2048, 1024, 64000, 0, 1, "plain_nows"),
    ("ffn2_wgrad", 16384, 1024, 2048, 1, 0, "accum2"),
    ("ffn1_wgrad", 1024, 16384, 2048, 1, 0, "accum2"),
    ("oproj_wgrad", 2048, 1024, 2048, 1, 0, "accum2"),
    ("qkv_wgrad", 1024, 6144, 2048, 1, 0, "accum2"),
    ("logits_wgrad", 1024, 64000, 2048, 1, 0, "accum2"),
]


@pytest.mark.parametrize("case", BENCH_GEMMS, ids=[c[0] for c in BENCH_GEMMS])
def test_gemm_tcgen05_bench_shapes_sampled(case):
    """The launch configurations bench.py times: full-size GEMMs of the
    config-5 micro-batch, each with the epilogue the engine fuses into it (>= 7 waves of 256 x 256 tiles on the
    big outputs, 16 to 1000 K-blocks), compared on 24 sampled output rows with the oracle's definition - a plain
    fp64 matmul of the same bf16-representable operands plus the epilogue written out.  fp32 outputs: 2e-5
    (fp32 accumulation of exact products; 1e-4 for the 64000-deep chain); bf16 outputs: one rounding, 2^-7."""
    name, M, N, K, tA, tB, epi = case
    r = _rng(sum(map(ord, name)))
    At, Aq = _lp(r.standard_normal((K, M) if tA else (M, K), dtype=np.float32) * 0.5, "bf16")
    Bt, Bq = _lp(r.standard_normal((N, K) if tB else (K, N), dtype=np.float32) * 0.5, "bf16")
    rows = np.sort(r.choice(M, size=24, replace=False))
    ref = (Aq.T[rows] if tA else Aq[rows]) @ (Bq.T if tB else Bq)          # [24, N] fp64
    f32_tol = 1e-4 if K > 20000 else 2e-5
    # a shallow pipeline (K < 4 cells: config 2) hands every GEMM its cell's split-K workspace: the few-tile, very
    # deep product dlogits W_out^T splits along K (specialised split kernel), the others ignore it.  Split launches
    # are run twice on the same workspace: the partial sums are reduced in split order, so the result is bitwise
    # reproducible and the counters reset themselves.
    ws = None if epi == "plain_nows" else ops.gemm_workspace(M, N, K, DEV)
    if name == "logits_dgrad":
        assert ws is not None and ws.numel() > 0, "%s is no longer split along K" % name
    wsarg = ws if ws is not None else False
    if epi == "plain" or epi == "plain_nows":
        C = torch.empty((M, N), device=DEV, dtype=torch.bfloat16)
        ops.gemm(At, Bt, C, transA=bool(tA), transB=bool(tB), workspace=wsarg, backend=2)
        assert maxrel(_np(C[rows]), ref) <= 2 ** -7 and cosine(_np(C[rows]), ref) >= 0.99999
        if ws is not None:
            C2 = torch.empty_like(C)
            ops.gemm(At, Bt, C2, transA=bool(tA), transB=bool(tB), workspace=ws, backend=2)
            assert torch.equal(C, C2)
    elif epi == "bias":
        bias = r.standard_normal(N).astype(np.float32)
        C = torch.empty((M, N), device=DEV, dtype=torch.bfloat16)
        ops.gemm(At, Bt, C, bias=torch.tensor(bias, device=DEV), workspace=False, backend=2)
        assert maxrel(_np(C[rows]), ref + bias) <= 2 ** -7 and cosine(_np(C[rows]), ref + bias) >= 0.99999
    elif epi == "bias_relu_bits":
        bias = r.standard_normal(N).astype(np.float32)
        C = torch.empty((M, N), device=DEV, dtype=torch.bfloat16)
        bits = torch.zeros((M, N // 32), device=DEV, dtype=torch.int32)
        ops.gemm(At, Bt, C, bias=torch.tensor(bias, device=DEV), relu=True, bits_out=bits, workspace=False, backend=2)
        want = np.maximum(ref + bias, 0)
        assert maxrel(_np(C[rows]), want) <= 2 ** -7 and cosine(_np(C[rows]), want) >= 0.99999
        got_bits = _unpack_mask(bits, M, N)
        assert np.array_equal(got_bits, _np(C) > 0)                        # every row: pattern == [stored h > 0]
        # and the pattern is the oracle's [z > 0] except where |z| is within bf16 rounding of 0
        z = ref + bias
        clear = np.abs(z) > 2 ** -7 * np.abs(z).max()
        assert np.array_equal(got_bits[rows][clear], (z > 0)[clear])
    elif epi == "accum":
        c0 = r.standard_normal((M, N)).astype(np.float32)
        C = torch.tensor(c0, device=DEV)
        ops.gemm(At, Bt, C, accumulate=True, workspace=wsarg, backend=2)    # x += branch (a8, a11)
        assert maxrel(_np(C[rows]), c0[rows] + ref) <= f32_tol
        if ws is not None:
            C2 = torch.tensor(c0, device=DEV)
            ops.gemm(At, Bt, C2, accumulate=True, workspace=ws, backend=2)
            assert torch.equal(C, C2)
    elif epi == "accum2":
        c0 = r.standard_normal((M, N)).astype(np.float32)
        C = torch.tensor(c0, device=DEV)
        ops.gemm(At, Bt, C, transA=True, accumulate=True, workspace=wsarg, backend=2)   # dW += X^T dY, two
        ops.gemm(At, Bt, C, transA=True, accumulate=True, workspace=wsarg, backend=2)   # micro-batches (a18)
        assert maxrel(_np(C[rows]), c0[rows] + 2 * ref) <= f32_tol
    elif epi == "mask_colsum":
        maskq = r.standard_normal((M, N)) > 0
        cs0 = r.standard_normal(N).astype(np.float32)
        cst = torch.tensor(cs0, device=DEV)
        C = torch.empty((M, N), device=DEV, dtype=torch.bfloat16)
        ops.gemm(At, Bt, C, transB=True, mask=_pack_mask(maskq), colsum_out=cst, workspace=False, backend=2)
        want = ref * maskq[rows]
        assert maxrel(_np(C[rows]), want) <= 2 ** -7 and cosine(_np(C[rows]), want) >= 0.99999
        full = _np(C)
        assert not full[~maskq].any()                                      # masked units are exactly zero
        assert maxrel(_np(cst), cs0 + full.sum(0)) <= 2e-5                  # db_1 += column sums of the stored dh
    else:
        raise AssertionError(epi)


# the launches of the list above that a handle with >= 8 cells (the bench workload: 16) sends to the 256 x 512 pair tile
WIDE_BENCH_GEMMS = [c for c in BENCH_GEMMS if c[6] in ("plain_nows", "accum", "accum2") or (c[6] == "plain" and c[0] != "logits_dgrad")]


@pytest.mark.parametrize("case", WIDE_BENCH_GEMMS, ids=[c[0] for c in WIDE_BENCH_GEMMS])
def test_gemm_tcgen05_bench_shapes_wide_tile(case):
    """The same full-size config-5 launches in the tile the 16-cell bench step actually runs them with: the
    256 x 512 pair tile (backend 4) - plain bf16 output (logits, the dgrads of FFN1 / QKV / out-projection, the
    unsplit dlogits W_out^T) and fp32 accumulate (FFN2 / out-projection forward, every wgrad).  24 sampled rows
    against the fp64 product of the same operands, and the whole output bit for bit against the 256 x 256 tiles."""
    name, M, N, K, tA, tB, epi = case
    assert N % 512 == 0
    r = _rng(sum(map(ord, name)) + 1)
    At, Aq = _lp(r.standard_normal((K, M) if tA else (M, K), dtype=np.float32) * 0.5, "bf16")
    Bt, Bq = _lp(r.standard_normal((N, K) if tB else (K, N), dtype=np.float32) * 0.5, "bf16")
    rows = np.sort(r.choice(M, size=24, replace=False))
    ref = (Aq.T[rows] if tA else Aq[rows]) @ (Bq.T if tB else Bq)
    f32_tol = 1e-4 if K > 20000 else 2e-5
    kw = dict(transA=bool(tA), transB=bool(tB), workspace=False)
    out = {}
    for backend in (4, 3):
        if epi in ("plain", "plain_nows"):
            C = torch.empty((M, N), device=DEV, dtype=torch.bfloat16)
            ops.gemm(At, Bt, C, backend=backend, **kw)
            if backend == 4:
                assert maxrel(_np(C[rows]), ref) <= 2 ** -7 and cosine(_np(C[rows]), ref) >= 0.99999
        else:
            n_acc = 2 if epi == "accum2" else 1
            c0 = r.standard_normal((M, N)).astype(np.float32) if backend == 4 else c0
            C = torch.tensor(c0, device=DEV)
            for _ in range(n_acc):
                ops.gemm(At, Bt, C, accumulate=True, backend=backend, **kw)
            if backend == 4:
                assert maxrel(_np(C[rows]), c0[rows] + n_acc * ref) <= f32_tol
        out[backend] = C
    assert torch.equal(out[3], out[4])


@pytest.mark.parametrize("dtype", ["fp32", "bf16"])
@pytest.mark.parametrize("backend", [1, 0])
def test_gemm_epilogues(dtype, backend):
    """bias+ReLU (a10), bias+residual fp32 out (a8/a11), ReLU-mask (a16 dh), fp32 accumulate (a18)."""
    M, N, K = 256, 384, 128
    r = _rng(5)
    At, Aq = _lp(r.standard_normal((M, K)), dtype)
    Bt, Bq = _lp(r.standard_normal((K, N)), dtype)
    bias = r.standard_normal(N).astype(np.float32)
    resid = r.standard_normal((M, N)).astype(np.float32)
    maskq = r.standard_normal((M, N)) > 0                   # bit-packed ReLU pattern, bit n%32 of word n/32
    maskt = torch.tensor(np.packbits(maskq.reshape(M, N // 32, 32), axis=-1, bitorder="little")
                         .view(np.uint32).reshape(M, N // 32).view(np.int32), device=DEV)
    bt, rt = torch.tensor(bias, device=DEV), torch.tensor(resid, device=DEV)
    tol, cos = _tol(dtype)
    ref = Aq @ Bq
    C = torch.empty((M, N), device=DEV, dtype=At.dtype)
    bits = torch.zeros((M, N // 32), device=DEV, dtype=torch.int32)
    ops.gemm(At, Bt, C, bias=bt, relu=True, bits_out=bits, backend=backend)
    assert maxrel(_np(C), np.maximum(ref + bias, 0)) <= tol
    got = np.unpackbits(bits.cpu().numpy().view(np.uint8).reshape(M, N // 8), axis=-1, bitorder="little").astype(bool)
    assert np.array_equal(got, _np(C) > 0)                   # the recorded pattern is [stored h > 0]
    Cf = torch.empty((M, N), device=DEV, dtype=torch.float32)
    ops.gemm(At, Bt, Cf, bias=bt, resid=rt, backend=backend)
    assert maxrel(_np(Cf), ref + bias + resid) <= 2e-5
    ops.gemm(At, Bt, rt, bias=bt, resid=rt, backend=backend)            # residual aliasing the output
    assert maxrel(_np(rt), ref + bias + resid) <= 2e-5
    ops.gemm(At, Bt, C, mask=maskt, backend=backend)
    assert maxrel(_np(C), ref * maskq) <= tol
    # ReLU-mask + fused column sums of the stored output (dh and db_1 of a16 in one kernel)
    cs0 = r.standard_normal(N).astype(np.float32)
    cst = torch.tensor(cs0, device=DEV)
    ops.gemm(At, Bt, C, mask=maskt, colsum_out=cst, backend=backend)
    assert maxrel(_np(C), ref * maskq) <= tol
    assert maxrel(_np(cst), cs0 + _np(C).sum(0)) <= 2e-5
    Mr, Nr = 200, 328                                        # ragged tiles
    Ar, Arq = _lp(r.standard_normal((Mr, K)), dtype)
    Br, Brq = _lp(r.standard_normal((K, Nr)), dtype)
    Cr = torch.empty((Mr, Nr), device=DEV, dtype=At.dtype)
    csr = torch.zeros(Nr, device=DEV)
    ops.gemm(Ar, Br, Cr, colsum_out=csr, backend=backend)
    assert maxrel(_np(Cr), Arq @ Brq) <= tol
    assert maxrel(_np(csr), _np(Cr).sum(0)) <= 2e-5
    acc0 = r.standard_normal((K, N)).astype(np.float32)
    acc = torch.tensor(acc0, device=DEV)
    Xt, Xq = _lp(r.standard_normal((M, K)), dtype)
    Yt, Yq = _lp(r.standard_normal((M, N)), dtype)
    ops.gemm(Xt, Yt, acc, transA=True, accumulate=True, backend=backend)  # dW += X^T dY
    ops.gemm(Xt, Yt, acc, transA=True, accumulate=True, backend=backend)
    assert maxrel(_np(acc), acc0 + 2 * (Xq.T @ Yq)) <= 2e-5


# -------------------------------------------------------------------------------------------------
# LayerNorm
# -------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["fp32", "bf16"])
@pytest.mark.parametrize("n,d", [(7, 64), (130, 1024), (33, 96), (5, 2048)])
def test_layernorm_fwd_bwd(dtype, n, d):
    r = _rng(n * d)
    x = (r.standard_normal((n, d)) * 2 + 0.5).astype(np.float32)
    g = (1 + 0.1 * r.standard_normal((1, d))).astype(np.float32)
    b = (0.1 * r.standard_normal((1, d))).astype(np.float32)
    dyt, dyq = _lp(r.standard_normal((n, d)), dtype)
    dres = r.standard_normal((n, d)).astype(np.float32)
    y_ref, xhat, rstd = go.layernorm_fwd(x.astype(np.float64), g.astype(np.float64), b.astype(np.float64), 1e-5)
    dx_ref, dg_ref, db_ref = go.layernorm_bwd(dyq, xhat, rstd, g.astype(np.float64))
    xt, gt, bt = [torch.tensor(a, device=DEV) for a in (x, g, b)]
    y = torch.empty((n, d), device=DEV, dtype=dyt.dtype)
    mean = torch.empty(n, device=DEV)
    rs = torch.empty(n, device=DEV)
    ops.ln_fwd(xt, gt, bt, y, mean, rs)
    tol, cos = _tol(dtype)
    assert maxrel(_np(y), y_ref) <= tol
    assert maxrel(_np(rs), rstd[:, 0]) <= 1e-5 and maxrel(_np(mean), x.astype(np.float64).mean(1)) <= 1e-5
    # fused residual init: resid_out = x + bias (what the branch's output GEMM accumulates into)
    rb = r.standard_normal(d).astype(np.float32)
    ro, y2 = torch.empty((n, d), device=DEV), torch.empty_like(y)
    ops.ln_fwd(xt, gt, bt, y2, mean, rs, resid_bias=torch.tensor(rb, device=DEV), resid_out=ro)
    assert torch.equal(y2, y)
    assert np.array_equal(_np(ro), x + rb[None, :])
    dx = torch.empty((n, d), device=DEV)
    dx_lp = torch.empty((n, d), device=DEV, dtype=dyt.dtype) if dtype == "bf16" else None
    dg0 = r.standard_normal(d).astype(np.float32)
    dgt, dbt = torch.tensor(dg0, device=DEV), torch.zeros(d, device=DEV)
    ops.ln_bwd(dyt, xt, mean, rs, gt, torch.tensor(dres, device=DEV), dx, dx_lp, dgt, dbt)
    assert maxrel(_np(dx), dx_ref + dres) <= 2e-5
    if dx_lp is not None:
        assert maxrel(_np(dx_lp), dx_ref + dres) <= 2 ** -7
    assert maxrel(_np(dgt), dg0 + dg_ref[0]) <= 2e-5          # accumulates into dgamma
    assert maxrel(_np(dbt), db_ref[0]) <= 2e-5
    ops.ln_bwd(dyt, xt, mean, rs, gt, None, dx, None, dgt, dbt)   # no incoming residual gradient
    assert maxrel(_np(dx), dx_ref) <= 2e-5
    # fused bias gradient: colsum_out += sum_t dx_out (of the lp copy's values when there is one)
    cs0 = r.standard_normal(d).astype(np.float32)
    cst = torch.tensor(cs0, device=DEV)
    ops.ln_bwd(dyt, xt, mean, rs, gt, torch.tensor(dres, device=DEV), dx, dx_lp, dgt, dbt, colsum_out=cst)
    summed = _np(dx_lp) if dx_lp is not None else _np(dx)
    assert maxrel(_np(cst), cs0 + summed.sum(0)) <= 2e-5


# -------------------------------------------------------------------------------------------------
# attention
# -------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["fp32", "bf16"])
@pytest.mark.parametrize("S,A,dh", [(16, 4, 16), (40, 3, 32), (256, 2, 64), (100, 2, 64), (129, 3, 64), (64, 1, 64),
                                    (200, 2, 64), (192, 2, 64), (3, 1, 64)])
@pytest.mark.parametrize("causal", [0, 1])
@pytest.mark.parametrize("backend", [0, 2])       # 0: auto (tcgen05 for bf16, d_head 64, S <= 256); 2: legacy mma.sync
def test_attention_fwd_bwd(dtype, S, A, dh, causal, backend):
    if backend == 2 and (dtype != "bf16" or dh not in (32, 64)):
        pytest.skip("mma.sync attention: bf16, d_head 32 / 64 only")
    n_seq, da = 2, A * dh
    r = _rng(S * A + dh + causal)
    qkvt, qkvq = _lp(r.standard_normal((n_seq * S, 3 * da)), dtype)
    dot, doq = _lp(r.standard_normal((n_seq * S, da)), dtype)
    o = torch.empty((n_seq * S, da), device=DEV, dtype=qkvt.dtype)
    lse = torch.empty((n_seq, A, S), device=DEV)
    ops.attn_fwd(qkvt, o, lse, n_seq, S, A, dh, causal, backend)
    dqkv = torch.empty_like(qkvt)
    dvec = torch.empty((n_seq, A, S), device=DEV)
    ops.attn_bwd(qkvt, o, dot, lse, dqkv, dvec, n_seq, S, A, dh, causal, backend)
    tol, cos = _tol(dtype)
    if dtype == "bf16":
        tol = 2 ** -6                                   # P and dS are rounded to bf16 on tensor cores
    for b in range(n_seq):
        rows = slice(b * S, (b + 1) * S)
        q, k, v = qkvq[rows, :da], qkvq[rows, da:2 * da], qkvq[rows, 2 * da:]
        o_ref, ps = go.attention_fwd(q, k, v, A, dh, causal)
        assert maxrel(_np(o[rows]), o_ref) <= tol
        for h in range(A):
            s = (q[:, h * dh:(h + 1) * dh] @ k[:, h * dh:(h + 1) * dh].T) / math.sqrt(dh)
            if causal:
                s = np.where(np.tril(np.ones((S, S), bool)), s, -np.inf)
            lse_ref = np.log(np.exp(s - s.max(1, keepdims=True)).sum(1)) + s.max(1)
            assert np.abs(_np(lse[b, h]) - lse_ref).max() <= 1e-4
        # backward against the oracle with the kernel's own forward output as O (teacher-forced)
        dq, dk, dv = go.attention_bwd(doq[rows], q, k, v, ps, A, dh)
        got = _np(dqkv[rows])
        for name, ref, blk in (("dq", dq, 0), ("dk", dk, 1), ("dv", dv, 2)):
            assert maxrel(got[:, blk * da:(blk + 1) * da], ref) <= 4 * tol, name
            assert cosine(got[:, blk * da:(blk + 1) * da], ref) >= (cos if dtype == "fp32" else 0.9999), name


@pytest.mark.parametrize("case", ["small", "large", "mixed_rows", "orthogonal_gap", "orthogonal_huge"])
@pytest.mark.parametrize("causal", [0, 1])
@pytest.mark.parametrize("S", [256, 200])
def test_attention_forward_score_range(case, causal, S):
    """softmax is invariant to the shift m in exp(s - m): whatever shift a kernel uses (the exact row maximum today; a
    Cauchy-Schwarz bound |q_row| max_j |k_j| was measured in round 2), output and log-sum-exp
    must match the oracle's plain definition over the whole range of scores: small and large (|s| ~ 100), rows of both
    kinds inside one 128-row block, and q orthogonal to every k with norms far above the scores (where a norm-based
    shift would underflow)."""
    A, dh, n_seq = 2, 64, 2
    da = A * dh
    r = _rng(S + 7 * causal + len(case))
    x = r.standard_normal((n_seq * S, 3 * da))
    if case == "small":
        x[:, :2 * da] *= 0.25
    elif case == "large":
        x[:, :2 * da] *= 3.0                              # |s| up to ~ 100
    elif case == "mixed_rows":
        x[40:72, :da] *= 4.0                              # 32 rows straddling two warps with 16x the scores
        x[S + 130:S + 140, :da] *= 5.0
    else:
        c = 12.5 if case == "orthogonal_gap" else 40.0    # |q| |k| / sqrt(d_head) = 19.5 / 200, scores ~ 0
        x[:, :2 * da] *= 0.01
        for h in range(A):
            x[:, h * dh] += c                             # q along e_0
            x[:, da + h * dh + 1] += c                    # k along e_1
    qkvt, qkvq = _lp(x, "bf16")
    o = torch.empty((n_seq * S, da), device=DEV, dtype=torch.bfloat16)
    lse = torch.empty((n_seq, A, S), device=DEV)
    ops.attn_fwd(qkvt, o, lse, n_seq, S, A, dh, causal)
    for b in range(n_seq):
        rows = slice(b * S, (b + 1) * S)
        q, k, v = qkvq[rows, :da], qkvq[rows, da:2 * da], qkvq[rows, 2 * da:]
        o_ref, _ = go.attention_fwd(q, k, v, A, dh, causal)
        assert maxrel(_np(o[rows]), o_ref) <= 2 ** -6, (case, b)
        for h in range(A):
            sc = (q[:, h * dh:(h + 1) * dh] @ k[:, h * dh:(h + 1) * dh].T) / math.sqrt(dh)
            if causal:
                sc = np.where(np.tril(np.ones((S, S), bool)), sc, -np.inf)
            lse_ref = np.log(np.exp(sc - sc.max(1, keepdims=True)).sum(1)) + sc.max(1)
            assert np.abs(_np(lse[b, h]) - lse_ref).max() <= 1e-4 * max(1.0, np.abs(lse_ref).max()), (case, b, h)


@pytest.mark.parametrize("S,A", [(256, 3), (200, 2), (100, 2), (64, 1)])
@pytest.mark.parametrize("causal", [0, 1])
def test_attention_backward_fused_column_sums(S, A, causal):
    """db_qkv = sum_t dqkv[t]: the tcgen05 backward leaves, per sequence, the column sums of the dqkv
    rows it stores.  They must equal the sums of the stored bf16 values (fp32 summation order aside), leave dqkv
    unchanged bit for bit, and be refused by the backends that do not compute them."""
    from paper_1811_06965_b200 import GPipeError
    n_seq, dh = 3, 64
    da = A * dh
    r = _rng(900 + S + causal)
    qkvt, _ = _lp(r.standard_normal((n_seq * S, 3 * da)), "bf16")
    dot, _ = _lp(r.standard_normal((n_seq * S, da)), "bf16")
    o = torch.empty((n_seq * S, da), device=DEV, dtype=torch.bfloat16)
    lse = torch.empty((n_seq, A, S), device=DEV)
    dvec = torch.empty((n_seq, A, S), device=DEV)
    ops.attn_fwd(qkvt, o, lse, n_seq, S, A, dh, causal)
    d0 = torch.empty((n_seq * S, 3 * da), device=DEV, dtype=torch.bfloat16)
    d1 = torch.empty_like(d0)
    part = torch.full((n_seq, 3 * da), 7.0, device=DEV)
    ops.attn_bwd(qkvt, o, dot, lse, d0, dvec, n_seq, S, A, dh, causal)
    ops.attn_bwd(qkvt, o, dot, lse, d1, dvec, n_seq, S, A, dh, causal, colpart=part)
    assert torch.equal(d0, d1)
    want = _np(d1).reshape(n_seq, S, 3 * da).sum(axis=1)
    got = _np(part)
    assert np.abs(got - want).max() <= 1e-5 * np.abs(want).max(), np.abs(got - want).max()
    with pytest.raises(GPipeError):
        ops.attn_bwd(qkvt, o, dot, lse, d1, dvec, n_seq, S, A, dh, causal, backend=1, colpart=part)


@pytest.mark.parametrize("causal", [0, 1])
def test_attention_bench_shape_sampled(causal):
    """The launch configuration bench.py times at config 5 (8 sequences x 32 heads, S 256, d_head 64: 512 forward
    CTAs, 256 backward CTAs, more than one wave), checked on sampled (sequence, head) pairs the oracle
    computes one by one."""
    n_seq, S, A, dh = 8, 256, 32, 64
    da = A * dh
    r = _rng(4242 + causal)
    qkvt, qkvq = _lp(r.standard_normal((n_seq * S, 3 * da)), "bf16")
    dot, doq = _lp(r.standard_normal((n_seq * S, da)), "bf16")
    o = torch.empty((n_seq * S, da), device=DEV, dtype=torch.bfloat16)
    lse = torch.empty((n_seq, A, S), device=DEV)
    dqkv = torch.empty_like(qkvt)
    dvec = torch.empty((n_seq, A, S), device=DEV)
    ops.attn_fwd(qkvt, o, lse, n_seq, S, A, dh, causal)
    ops.attn_bwd(qkvt, o, dot, lse, dqkv, dvec, n_seq, S, A, dh, causal)
    got_o, got_d = _np(o), _np(dqkv)
    for (b, h) in [(0, 0), (0, 31), (3, 7), (4, 16), (7, 0), (7, 31)]:
        rows, c = slice(b * S, (b + 1) * S), slice(h * dh, (h + 1) * dh)
        q, k, v = qkvq[rows, :da][:, c], qkvq[rows, da:2 * da][:, c], qkvq[rows, 2 * da:][:, c]
        o_ref, ps = go.attention_fwd(q, k, v, 1, dh, causal)
        assert maxrel(got_o[rows, c], o_ref) <= 2 ** -6, (b, h)
        dq, dk, dv = go.attention_bwd(doq[rows, c], q, k, v, ps, 1, dh)
        for name, ref, blk in (("dq", dq, 0), ("dk", dk, 1), ("dv", dv, 2)):
            g = got_d[rows, blk * da + h * dh: blk * da + (h + 1) * dh]
            assert maxrel(g, ref) <= 2 ** -4 and cosine(g, ref) >= 0.9999, (name, b, h)


@pytest.mark.parametrize("S", [100, 129, 256])
@pytest.mark.parametrize("causal", [0, 1])
def test_attention_writes_only_its_outputs(S, causal):
    """Ragged sequence lengths end inside a 128-row block (TMA clipping on loads, predicated direct stores): every
    output lives in the middle of a sentinel-filled buffer whose guard rows must come back untouched, and two
    launches give bitwise equal results (no atomics, fixed accumulation order)."""
    n_seq, A, dh, G = 3, 2, 64, 64
    da = A * dh
    r = _rng(S + causal)
    qkvt, _ = _lp(r.standard_normal((n_seq * S, 3 * da)), "bf16")
    dot, _ = _lp(r.standard_normal((n_seq * S, da)), "bf16")
    sent = float(2.0 ** 100)
    o_big = torch.full((n_seq * S + 2 * G, da), sent, device=DEV, dtype=torch.bfloat16)
    d_big = torch.full((n_seq * S + 2 * G, 3 * da), sent, device=DEV, dtype=torch.bfloat16)
    l_big = torch.full((n_seq * A * S + 2 * G,), sent, device=DEV)
    o, dqkv = o_big[G:G + n_seq * S], d_big[G:G + n_seq * S]
    lse = l_big[G:G + n_seq * A * S].view(n_seq, A, S)
    dvec = torch.empty((n_seq, A, S), device=DEV)
    ops.attn_fwd(qkvt, o, lse, n_seq, S, A, dh, causal)
    ops.attn_bwd(qkvt, o, dot, lse, dqkv, dvec, n_seq, S, A, dh, causal)
    torch.cuda.synchronize()
    for big, inner in ((o_big, o), (d_big, dqkv)):
        assert bool((big[:G] == sent).all()) and bool((big[-G:] == sent).all())
        assert bool(torch.isfinite(inner.float()).all()) and not bool((inner == sent).any())
    assert bool((l_big[:G] == sent).all()) and bool((l_big[-G:] == sent).all()) and bool(torch.isfinite(lse).all())
    o1, d1, l1 = o.clone(), dqkv.clone(), lse.clone()
    ops.attn_fwd(qkvt, o, lse, n_seq, S, A, dh, causal)
    ops.attn_bwd(qkvt, o, dot, lse, dqkv, dvec, n_seq, S, A, dh, causal)
    assert torch.equal(o, o1) and torch.equal(dqkv, d1) and torch.equal(lse, l1)


# -------------------------------------------------------------------------------------------------
# softmax cross-entropy, column sums, embedding, SGD
# -------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["fp32", "bf16"])
@pytest.mark.parametrize("n,V", [(9, 512), (33, 32000), (4, 64000), (3, 1000)])
def test_softmax_ce(dtype, n, V):
    r = _rng(V + n)
    zt, zq = _lp(r.standard_normal((n, V)) * 3, dtype)
    labels = r.integers(0, V, size=n).astype(np.int32)
    rowloss = torch.empty(n, device=DEV)
    inv_T = 1.0 / 77
    loss_ref, dl_ref = go.softmax_ce(zq, labels, 77)
    ops.softmax_ce(zt, torch.tensor(labels, device=DEV), rowloss, inv_T)
    assert abs(float(rowloss.double().sum()) - loss_ref) <= 2e-5 * abs(loss_ref)
    tol, cos = _tol(dtype)
    assert maxrel(_np(zt), dl_ref) <= tol
    assert cosine(_np(zt), dl_ref) >= cos


@pytest.mark.parametrize("dtype", ["fp32", "bf16"])
@pytest.mark.parametrize("n,V", [(9, 512), (5, 32000), (4, 64000), (3, 1000)])
def test_softmax_ce_with_logit_clipping(dtype, n, V):
    """PAPER.md:174 / reading B5: the softmax sees clamp(z, -c, c); dlogits is 0 where the clamp is active.  Both
    sides clamp the SAME stored logits (bf16-representable inputs), so the clamp pattern must agree exactly; a
    label whose logit is clipped makes the case bite (its -1/T would otherwise dominate the row)."""
    from oracle import encdec_oracle as eo
    r = _rng(3 * V + n)
    zt, zq = _lp(r.standard_normal((n, V)) * 3, dtype)
    labels = r.integers(0, V, size=n).astype(np.int32)
    clip = 2.5
    labels[0] = int(np.argmax(zq[0]))                       # a clipped label logit (max of ~N(0,3) draws > 2.5)
    assert zq[0, labels[0]] > clip and (np.abs(zq) > clip).mean() > 0.2
    rowloss = torch.empty(n, device=DEV)
    loss_ref, dl_ref, per_tok = eo.softmax_ce_clipped(zq.astype(np.float64), labels, 77, clip)
    ops.softmax_ce(zt, torch.tensor(labels, device=DEV), rowloss, 1.0 / 77, clip)
    got = _np(zt)
    assert np.array_equal(got == 0, dl_ref == 0)            # the clamp pattern, bit for bit
    assert np.allclose(_np(rowloss), per_tok / 77, rtol=2e-5, atol=0)
    tol, cos = _tol(dtype)
    assert maxrel(got, dl_ref) <= tol
    assert cosine(got, dl_ref) >= cos
    # clip = 0 is "off": identical to the unclipped kernel
    z0, _ = _lp(zq, dtype)
    z1, _ = _lp(zq, dtype)
    ops.softmax_ce(z0, torch.tensor(labels, device=DEV), rowloss, 1.0 / 77)
    ops.softmax_ce(z1, torch.tensor(labels, device=DEV), rowloss, 1.0 / 77, 0.0)
    assert torch.equal(z0, z1)


@pytest.mark.parametrize("clip", [0.0, 2.5])
@pytest.mark.parametrize("dtype,V", [("bf16", 64000), ("fp32", 32000), ("bf16", 32000)])
def test_softmax_ce_label_positions(dtype, V, clip):
    """The row lives on the SM as 16-byte vectors, vector j in slot j // 512 of thread j % 512: slots 0..7 are
    registers, 8..15 shared memory (rows beyond 4096 vectors).  The label's -1/T goes to one element of one vector:
    put it at the first / last element of the first register vector, across the register / shared-memory boundary
    and at the row's last element, with and without the clamp (reading B5)."""
    from oracle import encdec_oracle as eo
    W = 8 if dtype == "bf16" else 4
    nvec = V // W
    pos = [0, W - 1, W, 511 * W + 3, 512 * W, min(4096, nvec) * W - 1, min(4096, nvec - 1) * W, (nvec - 1) * W, V - 1]
    n = len(pos)
    r = _rng(5 * V + n)
    zt, zq = _lp(r.standard_normal((n, V)) * 3, dtype)
    labels = np.asarray(pos, dtype=np.int32)
    rowloss = torch.empty(n, device=DEV)
    if clip > 0:
        loss_ref, dl_ref, per_tok = eo.softmax_ce_clipped(zq.astype(np.float64), labels, 77, clip)
    else:
        loss_ref, dl_ref = go.softmax_ce(zq, labels, 77)
    ops.softmax_ce(zt, torch.tensor(labels, device=DEV), rowloss, 1.0 / 77, clip)
    got = _np(zt)
    assert abs(float(rowloss.double().sum()) - loss_ref) <= 2e-5 * abs(loss_ref)
    tol, cos = _tol(dtype)
    assert maxrel(got, dl_ref) <= tol and cosine(got, dl_ref) >= cos
    for t, v in enumerate(pos):                              # the label's own element, one by one
        assert abs(got[t, v] - dl_ref[t, v]) <= tol * max(abs(dl_ref[t, v]), 1.0 / 77), (t, v)
        if clip > 0:
            assert (got[t, v] == 0) == (abs(zq[t, v]) > clip)


@pytest.mark.parametrize("dtype", ["fp32", "bf16"])
def test_colsum_embedding_sgd(dtype):
    r = _rng(11)
    dyt, dyq = _lp(r.standard_normal((300, 200)), dtype)
    out0 = r.standard_normal(200).astype(np.float32)
    out = torch.tensor(out0, device=DEV)
    ops.colsum(dyt, out)
    assert maxrel(_np(out), out0 + dyq.sum(0)) <= 2e-5
    # embedding forward/backward (reading A6)
    V, d, S, n_seq = 50, 64, 10, 3
    embt, embq = _lp(r.standard_normal((V, d)), dtype)
    tok = r.integers(0, V, size=n_seq * S).astype(np.int32)
    pe = torch.empty((S, d), device=DEV)
    ops.positional(pe)
    assert maxrel(_np(pe), go.positional_table(S, d, np.float64)) <= 1e-6
    x = torch.empty((n_seq * S, d), device=DEV)
    tt = torch.tensor(tok, device=DEV)
    ops.embed_fwd(tt, embt, pe, x, S)
    assert maxrel(_np(x), embq[tok] + np.tile(go.positional_table(S, d, np.float64), (n_seq, 1))) <= 1e-6
    dx = r.standard_normal((n_seq * S, d)).astype(np.float32)
    gemb = torch.zeros((V, d), device=DEV)
    ops.embed_bwd(tt, torch.tensor(dx, device=DEV), gemb)
    ref = np.zeros((V, d))
    np.add.at(ref, tok, dx.astype(np.float64))
    assert maxrel(_np(gemb), ref) <= 1e-5
    # SGD apply
    n = 4096
    m0, g0 = r.standard_normal(n).astype(np.float32), r.standard_normal(n).astype(np.float32)
    m, g = torch.tensor(m0, device=DEV), torch.tensor(g0, device=DEV)
    wl = torch.empty(n, device=DEV, dtype=torch.bfloat16) if dtype == "bf16" else None
    ops.sgd(m, g, wl, 0.25)
    assert np.array_equal(m.cpu().numpy(), m0 - np.float32(0.25) * g0)
    assert not g.any()
    if wl is not None:
        assert torch.equal(wl, m.to(torch.bfloat16))


@pytest.mark.parametrize("dtype", ["fp32", "bf16"])
def test_rmsprop_kernel_matches_library_routine(dtype):
    """gpipe_op_rmsprop against torch.optim.RMSprop on the CPU (alpha = rho, no momentum, not centered) over three
    applications; the bf16 working copy is the RNE rounding of the fp32 master; the gradient is cleared."""
    r = _rng(31)
    n = 4096 + 64
    lr, rho, eps = 0.05, 0.9, 1e-6
    w0 = r.standard_normal(n).astype(np.float32)
    m = torch.tensor(w0, device=DEV)
    ms = torch.zeros(n, device=DEV)
    wl = torch.empty(n, device=DEV, dtype=torch.bfloat16) if dtype == "bf16" else None
    tp = torch.tensor(w0.astype(np.float64), requires_grad=True)
    opt = torch.optim.RMSprop([tp], lr=lr, alpha=rho, eps=eps)
    for step in range(3):
        g0 = (r.standard_normal(n) * 10.0 ** r.integers(-4, 3, size=n)).astype(np.float32)
        g0[::7] = 0.0
        g = torch.tensor(g0, device=DEV)
        ops.rmsprop(m, g, ms, wl, lr, rho, eps)
        tp.grad = torch.tensor(g0.astype(np.float64))
        opt.step()
        assert not _np(g).any()
        assert maxrel(_np(m), tp.detach().numpy()) <= 2e-6, step
        if wl is not None:
            assert torch.equal(wl, m.to(torch.bfloat16))


@pytest.mark.parametrize("n_tok,V,d", [(2048, 64000, 1024), (2048, 7, 1024), (77, 50, 64), (1, 3, 8), (5000, 300, 256)])
def test_embedding_backward_is_exact_and_deterministic(n_tok, V, d):
    """dE[tok[t]] += dx0[t] (a17): every vocabulary row has one owner that adds its tokens in ascending t, so the
    result is the fp32 running sum in token order - reproduced here with a sequential fp32 loop - bitwise, on every
    launch, whatever the multiplicity of an id (V = 7: ~300 tokens per row)."""
    r = _rng(n_tok + V)
    tok = r.integers(0, V, size=n_tok).astype(np.int32)
    dx = r.standard_normal((n_tok, d)).astype(np.float32)
    g0 = r.standard_normal((V, d)).astype(np.float32)
    ref = g0.copy()
    for t in range(n_tok):                                   # the definition, in the kernel's order and precision
        ref[tok[t]] += dx[t]
    tt, dxt = torch.tensor(tok, device=DEV), torch.tensor(dx, device=DEV)
    outs = []
    for _ in range(3):
        gemb = torch.tensor(g0, device=DEV)
        ops.embed_bwd(tt, dxt, gemb)
        outs.append(_np(gemb).astype(np.float32))
    assert np.array_equal(outs[0], ref)
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])

"""gpipe_op_colsum_static (include/gpipe_ops.h): the column sums with their scratch in a static array inside the library,
for callers that cannot allocate device memory.  Collected last on purpose (the suite runs with pytest -x).

Checked against the existing path (gpipe_op_colsum with caller-owned scratch: same kernels, same summation order, so
bit for bit) and against the plain definition (fp64 column sums of the same stored values), on two calls in a row that
share the array - the second with other data and a different shape, so stale partials of the first call would show."""
import numpy as np
import pytest
import torch

from paper_1811_06965_b200 import GPipeError, ops

pytestmark = pytest.mark.gpu

DEV = "cuda"


def _case(seed, n_tok, n, dtype, pad=0):
    r = np.random.default_rng(seed)
    full = torch.tensor(r.standard_normal((n_tok, n + pad)).astype(np.float32), device=DEV)
    if dtype == "bf16":
        full = full.to(torch.bfloat16)
    dy = full[:, :n] if pad else full                     # pad > 0: a column view, row pitch n + pad
    out0 = torch.tensor(r.standard_normal(n).astype(np.float32), device=DEV)
    return dy, out0


@pytest.mark.parametrize("dtype", ["bf16", "fp32"])
def test_colsum_static_matches_the_allocating_path_on_two_calls_in_a_row(dtype):
    # 1: the widest bias of the bench workload (b_1, H = 16384 = the limit) over one micro-batch; 2: ragged rows and
    # columns on a column view, fewer partial rows and columns than call 1 left in the array; 3: call 1's shape again
    shapes = [(2048, ops.COLSUM_STATIC_MAX_N, 0), (301, 1000, 24), (2048, ops.COLSUM_STATIC_MAX_N, 0)]
    for i, (n_tok, n, pad) in enumerate(shapes):
        dy, out0 = _case(100 + i, n_tok, n, dtype, pad)
        got, want = out0.clone(), out0.clone()
        ops.colsum_static(dy, got)
        ops.colsum(dy, want)                              # the existing path, scratch from torch
        torch.cuda.synchronize()
        assert torch.equal(got, want), (i, n_tok, n)
        ref = out0.double().cpu().numpy() + dy.double().cpu().numpy().sum(0)
        err = np.abs(got.cpu().numpy() - ref).max() / np.abs(ref).max()
        assert err <= 2e-5, (i, err)                      # fp32 sums of exactly representable inputs (test_gpu_ops tolerance)


def test_colsum_static_allocates_nothing_and_rejects_sizes_beyond_the_limit():
    dy, out = _case(7, 512, 4096, "bf16")
    ops.colsum_static(dy, out)                            # first use on this device: takes the symbol's address
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        ops.colsum_static(dy, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                 # no device memory taken by the calls
    wide = torch.zeros((8, ops.COLSUM_STATIC_MAX_N + 8), device=DEV, dtype=torch.bfloat16)
    acc = torch.zeros(ops.COLSUM_STATIC_MAX_N + 8, device=DEV)
    with pytest.raises(GPipeError) as err:
        ops.colsum_static(wide, acc)
    assert str(ops.COLSUM_STATIC_MAX_N) in str(err.value)
    assert not acc.any()                                  # rejected before anything ran
    empty = torch.zeros((0, 64), device=DEV, dtype=torch.bfloat16)
    ops.colsum_static(empty, torch.zeros(64, device=DEV))  # empty input: a no-op, not an error

"""CPU-side checks of the boundary: the shared library builds, loads and exports every symbol the
headers declare; the host-only planner and argument validation work without a GPU."""
import os
import re

import pytest

import gpipe_inputs as gi
import paper_1811_06965_b200 as gp
from paper_1811_06965_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    build.build()


def _declared(header):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gpipe_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported():
    lib = gp.lib()
    declared = _declared("gpipe.h") + _declared("gpipe_ops.h")
    assert len(declared) >= 30
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(declared) == sorted(binding.EXPORTED_SYMBOLS)


def test_version_and_error_string():
    assert b"sm_100a" in gp.lib().gpipe_version()


def _spec(w):
    return gp.make_spec(w.n_layers, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len, w.dtype,
                        list(w.causal))


def test_plan_bytes_follows_paper_memory_law():
    """activations ~ N + (L/K)(N/M) with remat; ~ N*L without (tracker, no GPU)."""
    w = gi.CONFIGS["T(12,8192,16)"]
    spec, keep = _spec(w)
    r = {M: gp.plan_bytes(spec, w.K, M, True, w.n_seqs) for M in (1, 4, 8, 16, 32)}
    s = {M: gp.plan_bytes(spec, w.K, M, False, w.n_seqs) for M in (1, 4, 8, 16, 32)}
    # a + b/M: successive differences are proportional to differences of 1/M
    b1 = (r[1] - r[4]) / (1 - 1 / 4)
    b2 = (r[8] - r[16]) / (1 / 8 - 1 / 16)
    assert abs(b1 - b2) / b1 < 0.02
    assert r[32] < r[1] / 5
    assert max(s.values()) / min(s.values()) < 1.4          # ~ independent of M
    assert s[32] > 5 * r[32]


def test_per_accelerator_plan_follows_table1():
    """PAPER.md:65 / :103 (Table 1): with cell k on accelerator k the parameters, gradients and activations are
    spread over the K devices - the per-device need falls roughly as 1/K, which is what lets a larger model fit.
    Host-only planner of the pipeline handle (gpipe_plan_bytes_pipeline)."""
    from paper_1811_06965_b200.binding import plan_bytes_pipeline
    w = gi.CONFIGS["T(64,16384,32)"]
    spec, keep = _spec(w)
    one = gp.plan_bytes(spec, 16, w.M, True, w.n_seqs)
    per = {K: plan_bytes_pipeline(spec, K, w.M, True, w.n_seqs) for K in (2, 4, 8, 16)}
    for K, need in per.items():
        assert len(need) == K
        # the split adds only the staging copies of the boundary tensors
        assert abs(sum(need) - gp.plan_bytes(spec, K, w.M, True, w.n_seqs)) <= 0.02 * one
        assert max(need[1:-1] or need) <= 1.15 * min(need[1:-1] or need)   # interior cells are balanced
    assert max(per[16]) < 0.09 * one and max(per[16]) < 16e9               # the 6 B model on 16 small accelerators
    assert max(per[2]) > 6 * max(per[16])
    uneven = plan_bytes_pipeline(spec, 4, w.M, True, w.n_seqs, cell_lo=[0, 10, 40, 100, 128])
    assert uneven[2] > 1.8 * uneven[1] > 3 * uneven[0]


def test_config5_fits_180GB_with_remat():
    w = gi.CONFIGS["T(64,16384,32)"]
    spec, keep = _spec(w)
    assert gp.plan_bytes(spec, w.K, w.M, True, w.n_seqs) < 180e9


def test_invalid_arguments_are_rejected():
    w = gi.CONFIGS["tiny"]
    spec, keep = _spec(w)
    with pytest.raises(gp.GPipeError) as e:
        gp.plan_bytes(spec, 3, 4, True, 8)              # K > L
    assert e.value.code == -1
    with pytest.raises(gp.GPipeError):
        gp.plan_bytes(spec, 2, 3, True, 8)              # 8 % 3 != 0: micro-batches must be equal
    with pytest.raises(gp.GPipeError):
        gp.plan_bytes(spec, 2, 0, True, 8)
    bad, keep2 = gp.make_spec(2, 64, 256, 4, 24, 512, 16, "fp32")
    with pytest.raises(gp.GPipeError):
        gp.plan_bytes(bad, 2, 4, True, 8)               # unsupported d_head


def test_product_does_not_import_oracle():
    """The CUDA package must not reach into oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1811_06965_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "oracle" not in txt.replace("no oracle code", ""), fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith(".py"):
            assert "paper_1811_06965_b200" not in open(os.path.join(ROOT, "oracle", fn)).read().replace(
                "CUDA path (paper_1811_06965_b200/)", "")


def test_encdec_planner_and_argument_checks():
    """gpipe_plan_bytes_encdec (host only): the 6.04 B T(64,16384,32) of PAPER.md:158 fits one 180 GB B200 with
    remat, K = M = 16; the activation law of PAPER.md:87 holds for the pair boundary too; bad arguments are refused."""
    from paper_1811_06965_b200.binding import EncDecSpec, plan_bytes_encdec
    s6 = EncDecSpec(64, 64, 1024, 16384, 32, 64, 64000, 256, 1, 1e-5, 0.0)
    need = plan_bytes_encdec(s6, 16, 16, True, 128)
    n_param = 6.04e9
    assert 10 * n_param < need < 180e9                      # 10 B / parameter (bf16 copy + fp32 master + fp32 grad) + activations
    r = {M: plan_bytes_encdec(s6, 16, M, True, 128) for M in (1, 4, 16)}
    assert r[1] > r[4] > r[16]
    assert plan_bytes_encdec(s6, 16, 16, False, 128) > 1.5 * need
    # explicit boundaries over the 128 layers: same parameters, so nearly the same bytes
    lo = [0] + [8 * k + 4 for k in range(1, 16)] + [128]
    assert abs(plan_bytes_encdec(s6, 16, 16, True, 128, lo) - need) < 0.05 * need
    tiny = EncDecSpec(2, 2, 64, 256, 4, 16, 512, 16, 0, 1e-5, 0.0)
    assert plan_bytes_encdec(tiny, 4, 4, True, 8) > 0
    for bad in (dict(K=5), dict(M=3), dict(lo=[0, 2, 2, 4], K=3)):
        with pytest.raises(gp.GPipeError):
            plan_bytes_encdec(tiny, bad.get("K", 2), bad.get("M", 4), True, 8, bad.get("lo"))
    for spec in (EncDecSpec(0, 2, 64, 256, 4, 16, 512, 16, 0, 1e-5, 0.0),
                 EncDecSpec(2, 0, 64, 256, 4, 16, 512, 16, 0, 1e-5, 0.0),
                 EncDecSpec(2, 2, 64, 256, 4, 16, 512, 16, 0, 1e-5, -0.5)):
        with pytest.raises(gp.GPipeError):
            plan_bytes_encdec(spec, 2, 4, True, 8)

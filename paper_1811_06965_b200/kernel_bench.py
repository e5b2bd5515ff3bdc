"""Per-kernel roofline microbenchmark: times every kernel class of the hot path ALONE, at the
shapes one micro-batch of a workload produces (T_mb tokens), through the C ABI of
include/gpipe_ops.h.

    python -m paper_1811_06965_b200.kernel_bench [--workload NAME] [--only gemm|ln|attn|ce|all]
                                                 [--reps R] [--json PATH] [--compare]

Each case runs on R rotating operand sets whose total footprint exceeds the 126 MB L2 (so no
launch finds its inputs cached from its own previous run), is timed with CUDA events on the
launching stream after 3 warm-up launches, and is reported as algorithmic FLOP/s or bytes/s
(2MNK per GEMM; every operand and output counted once) against the
measured peaks in MEASURED_PEAKS.json.  `--compare` adds torch.matmul on the same GEMM shape as a
comparator column (never part of the product path).  This is also the command the ncu captures
under profiles/ were taken with.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import gpipe_inputs as gi  # noqa: E402


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        j = json.load(open(p))
        return j["bf16_tflops"], j["hbm_gbs"], "measured"
    return 1590.0, 6650.0, "fallback"


def gemm_cases(w, T):
    d, H, da, V = w.d_model, w.d_ffn, w.d_attn, w.vocab
    # name, M, N, K, transA, transB, epilogue kwargs (as the engine launches them)
    return [
        ("qkv_fwd", T, 3 * da, d, 0, 0, dict(bias=1)),
        ("oproj_fwd", T, d, da, 0, 0, dict(accum=1)),
        ("ffn1_fwd", T, H, d, 0, 0, dict(bias=1, relu=1, bits=1)),
        ("ffn2_fwd", T, d, H, 0, 0, dict(accum=1)),
        ("logits_fwd", T, V, d, 0, 0, dict()),
        ("ffn2_dgrad", T, H, d, 0, 1, dict(mask=1, colsum=1)),
        ("ffn1_dgrad", T, d, H, 0, 1, dict()),
        ("oproj_dgrad", T, da, d, 0, 1, dict()),
        ("qkv_dgrad", T, d, 3 * da, 0, 1, dict()),
        ("logits_dgrad", T, d, V, 0, 1, dict()),
        ("ffn2_wgrad", H, d, T, 1, 0, dict(accum=1)),
        ("ffn1_wgrad", d, H, T, 1, 0, dict(accum=1)),
        ("oproj_wgrad", da, d, T, 1, 0, dict(accum=1)),
        ("qkv_wgrad", d, 3 * da, T, 1, 0, dict(accum=1)),
        ("logits_wgrad", d, V, T, 1, 0, dict(accum=1)),
    ]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="T(64,16384,32)", choices=gi.CONFIG_ORDER)
    ap.add_argument("--only", default="all")
    ap.add_argument("--case", default=None, help="substring filter on the case name")
    ap.add_argument("--reps", type=int, default=10)
    ap.add_argument("--json", default=None)
    ap.add_argument("--compare", action="store_true")
    ap.add_argument("--gemm-backend", type=int, default=0,
                    help="0: the launcher's own tile choice; 3: 256 x 256 pair tiles only; 4: 256 x 512 pair tiles only "
                         "(shapes / epilogues the wide tile does not take are skipped)")
    args = ap.parse_args()

    import torch
    from paper_1811_06965_b200 import ops, build
    build.build()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    w = gi.CONFIGS[args.workload]
    T = w.n_seqs // w.M * w.seq_len
    bf = torch.bfloat16
    tf_peak, hbm_peak, src = _peaks()
    rows = []
    want = lambda kind, name: (args.only in ("all", kind)) and (args.case is None or args.case in name)

    def time_it(fns, reps):
        for f in fns[:3]:
            f()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n = 0
        e0.record()
        for _ in range(reps):
            for f in fns:
                f()
                n += 1
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n

    def nsets(bytes_per_set):
        return max(2, min(8, int(256e6 // max(bytes_per_set, 1)) + 1))

    def report(kind, name, ms, flops, byts, extra=None):
        r = {"kind": kind, "case": name, "us": ms * 1e3, "tflops": flops / ms / 1e9 if flops else None,
             "gbs": byts / ms / 1e6, "frac_tensor": (flops / ms / 1e9 / tf_peak) if flops else None,
             "frac_hbm": byts / ms / 1e6 / hbm_peak}
        if extra:
            r.update(extra)
        rows.append(r)
        print("%-6s %-14s %9.1f us  %8s TF/s  %8.0f GB/s  tensor %5s  hbm %5.2f %s" % (
            kind, name, r["us"], "%.0f" % r["tflops"] if flops else "-", r["gbs"],
            "%.2f" % r["frac_tensor"] if flops else "-", r["frac_hbm"],
            ("cmp %.1f us" % extra["cmp_us"]) if extra and "cmp_us" in extra else ""), flush=True)

    # ------------------------------------------------------------------ GEMMs
    for name, M, N, K, tA, tB, ep in gemm_cases(w, T):
        if not want("gemm", name):
            continue
        out_f32 = bool(ep.get("resid") or ep.get("accum"))
        per = (M * K + K * N) * 2 + M * N * (4 if out_f32 else 2)
        ns = nsets(per)
        sets = []
        for _ in range(ns):
            A = torch.randn((K, M) if tA else (M, K), device=dev, dtype=torch.float32).mul_(0.05).to(bf)
            Bm = torch.randn((N, K) if tB else (K, N), device=dev, dtype=torch.float32).mul_(0.05).to(bf)
            Cm = torch.zeros((M, N), device=dev, dtype=torch.float32 if out_f32 else bf)
            kw = {}
            if ep.get("bias"): kw["bias"] = torch.randn(N, device=dev)
            if ep.get("relu"): kw["relu"] = True
            if ep.get("bits"): kw["bits_out"] = torch.zeros((M, N // 32), device=dev, dtype=torch.int32)
            if ep.get("resid"): kw["resid"] = torch.randn((M, N), device=dev)
            if ep.get("mask"): kw["mask"] = torch.randint(-2 ** 31, 2 ** 31 - 1, (M, N // 32), device=dev, dtype=torch.int32)
            if ep.get("accum"): kw["accumulate"] = True
            if ep.get("colsum"): kw["colsum_out"] = torch.zeros(N, device=dev)
            kw["workspace"] = ops.gemm_workspace(M, N, K, dev)
            if kw["workspace"] is None: kw["workspace"] = False
            sets.append((A, Bm, Cm, kw))
        fns = [(lambda s=s: ops.gemm(s[0], s[1], s[2], transA=bool(tA), transB=bool(tB), backend=args.gemm_backend, **s[3]))
               for s in sets]
        try:
            ms = time_it(fns, args.reps)
        except Exception as e:                                 # backend 4 on a shape the wide tile does not take
            if args.gemm_backend == 0:
                raise
            print("gemm   %-14s skipped (%s)" % (name, str(e).splitlines()[0][:60]), flush=True)
            continue
        byts = per + (M * N * 4 if ep.get("resid") else 0) + (M * N * 4 if ep.get("accum") else 0) + \
            (M * N // 8 if ep.get("mask") or ep.get("bits") else 0)
        extra = {"M": M, "N": N, "K": K, "transA": tA, "transB": tB}
        if args.compare:
            cf = [(lambda s=s: torch.matmul(s[0].t() if tA else s[0], s[1].t() if tB else s[1])) for s in sets]
            extra["cmp_us"] = time_it(cf, args.reps) * 1e3
        report("gemm", name, ms, 2.0 * M * N * K, byts, extra)
        del sets, fns

    d, H, da, V, S, A_, dh = w.d_model, w.d_ffn, w.d_attn, w.vocab, w.seq_len, w.n_heads, w.d_head
    nb = T // S
    # ------------------------------------------------------------------ LayerNorm
    if want("ln", "ln_fwd"):
        ns = nsets(T * d * 6)
        sets = [(torch.randn((T, d), device=dev), torch.empty((T, d), device=dev, dtype=bf),
                 torch.empty(T, device=dev), torch.empty(T, device=dev)) for _ in range(ns)]
        g, b = torch.ones(d, device=dev), torch.zeros(d, device=dev)
        ms = time_it([(lambda s=s: ops.ln_fwd(s[0], g, b, s[1], s[2], s[3])) for s in sets], args.reps)
        extra = None
        if args.compare:
            # comparators (never on the product path): the vendor LayerNorm on the same rows, and a plain fp32 -> bf16
            # copy with exactly this kernel's traffic - what a launch of this size can reach at all
            extra = {"cmp_us": time_it([(lambda s=s: torch.nn.functional.layer_norm(s[0], (d,), g, b)) for s in sets], args.reps) * 1e3}
            cp = time_it([(lambda s=s: s[1].copy_(s[0])) for s in sets], args.reps)
        report("ln", "ln_fwd", ms, 0, T * d * 6.0, extra)
        if args.compare:
            report("ln", "copy_floor", cp, 0, T * d * 6.0)
    if want("ln", "ln_bwd"):
        ns = nsets(T * d * 18)
        g = torch.ones(d, device=dev)
        sets = []
        for _ in range(ns):
            x = torch.randn((T, d), device=dev)
            sets.append((torch.randn((T, d), device=dev).to(bf), x, x.mean(1), 1.0 / x.std(1), torch.randn((T, d), device=dev),
                         torch.empty((T, d), device=dev), torch.empty((T, d), device=dev, dtype=bf),
                         torch.zeros(d, device=dev), torch.zeros(d, device=dev), torch.zeros(d, device=dev)))
        ms = time_it([(lambda s=s: ops.ln_bwd(s[0], s[1], s[2], s[3], g, s[4], s[5], s[6], s[7], s[8], s[9])) for s in sets],
                     args.reps)
        report("ln", "ln_bwd", ms, 0, T * d * (2 + 4 + 4 + 4 + 2.0))
    # ------------------------------------------------------------------ attention
    for causal in (0, 1):
        if want("attn", "attn_fwd"):
            ns = nsets(T * da * 8)
            sets = [(torch.randn((T, 3 * da), device=dev).to(bf), torch.empty((T, da), device=dev, dtype=bf),
                     torch.empty((nb, A_, S), device=dev)) for _ in range(ns)]
            ms = time_it([(lambda s=s: ops.attn_fwd(s[0], s[1], s[2], nb, S, A_, dh, causal)) for s in sets], args.reps)
            f = 4.0 * T * S * da * ((S + 1.0) / (2 * S) if causal else 1.0)
            report("attn", "attn_fwd_c%d" % causal, ms, f, T * da * 8.0)
        if want("attn", "attn_bwd"):
            ns = nsets(T * da * 16)
            sets = []
            for _ in range(ns):
                qkv = torch.randn((T, 3 * da), device=dev).to(bf)
                o = torch.empty((T, da), device=dev, dtype=bf)
                lse = torch.empty((nb, A_, S), device=dev)
                ops.attn_fwd(qkv, o, lse, nb, S, A_, dh, causal)
                sets.append((qkv, o, torch.randn((T, da), device=dev).to(bf), lse,
                             torch.empty((T, 3 * da), device=dev, dtype=bf), torch.empty((nb, A_, S), device=dev)))
            ms = time_it([(lambda s=s: ops.attn_bwd(s[0], s[1], s[2], s[3], s[4], s[5], nb, S, A_, dh, causal)) for s in sets],
                         args.reps)
            f = 10.0 * T * S * da * ((S + 1.0) / (2 * S) if causal else 1.0)
            report("attn", "attn_bwd_c%d" % causal, ms, f, T * da * 16.0)
    # ------------------------------------------------------------------ softmax cross-entropy
    if want("ce", "softmax_ce"):
        ns = nsets(T * V * 2)
        lab = torch.randint(0, V, (T,), device=dev, dtype=torch.int32)
        sets = [(torch.randn((T, V), device=dev, dtype=bf), torch.empty(T, device=dev)) for _ in range(ns)]
        ms = time_it([(lambda s=s: ops.softmax_ce(s[0], lab, s[1], 1.0 / T)) for s in sets], max(2, args.reps // 2))
        report("ce", "softmax_ce", ms, 0, T * V * 4.0)
    # ------------------------------------------------------------------ SGD apply
    if want("sgd", "sgd_apply"):
        n = 64 * 1024 * 1024
        sets = [(torch.randn(n, device=dev), torch.randn(n, device=dev), torch.empty(n, device=dev, dtype=bf))
                for _ in range(2)]
        ms = time_it([(lambda s=s: ops.sgd(s[0], s[1], s[2], 1e-3)) for s in sets], max(2, args.reps // 2))
        report("sgd", "sgd_apply", ms, 0, n * 18.0)
        sets = [s + (torch.rand(n, device=dev),) for s in sets]
        ms = time_it([(lambda s=s: ops.rmsprop(s[0], s[1], s[3], s[2], 1e-3, 0.9, 1e-6)) for s in sets], max(2, args.reps // 2))
        report("sgd", "rmsprop_apply", ms, 0, n * 26.0)          # g r+w, ms r+w, master r+w, bf16 copy w

    # ------------------------------------------------------------------ fused data-parallel apply (f3), R replicas
    # emulated on this one device: the NVLink hop is absent, so this is the HBM roofline of the kernel -
    # per parameter of the shard: R x 4 B gradient reads, 4 B master read, R x (4 + 4 + 2) B stores
    if want("sgd", "dp_apply"):
        n = 32 * 1024 * 1024
        for R in (1, 2, 4):
            ms_ = [torch.randn(n, device=dev) for _ in range(R)]
            gs_ = [torch.randn(n, device=dev) for _ in range(R)]
            ws_ = [torch.empty(n, device=dev, dtype=bf) for _ in range(R)]
            fns = [(lambda r=r: ops.dp_apply_sgd(ms_, gs_, ws_, r, 1e-3)) for r in range(R)]
            ms = time_it(fns, max(2, args.reps // 2)) * R          # all R shards = one whole update of n parameters
            report("sgd", "dp_apply_R%d" % R, ms, 0, n * (4.0 * R + 4.0 + 10.0 * R))
            del ms_, gs_, ws_

    if args.json:
        os.makedirs(os.path.dirname(os.path.abspath(args.json)), exist_ok=True)
        with open(args.json, "w") as f:
            json.dump({"workload": w.name, "T_mb": T, "peak_tflops": tf_peak, "peak_hbm_gbs": hbm_peak,
                       "peaks": src, "rows": rows}, f, indent=1)


if __name__ == "__main__":
    main()

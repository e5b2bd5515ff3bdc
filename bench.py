#!/usr/bin/env python
"""bench.py - tokens/s of one GPipe mini-batch step (forward + re-materialized backward, fp32
gradient accumulation) on B200, through the C ABI of libgpipe_b200.so.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]

One "step" is one pass of the whole hot path (every row of SURVEY.md 8(a): micro-batch split,
all forward ticks, all replay + backward ticks, gradient accumulation) over one synthetic
mini-batch.  `value` is measured with the token ids already resident in HBM
(gpipe_step_device); `e2e` is the same step called with HOST id buffers (gpipe_step: H2D of
the ids and D2H of the loss partials inside the timed region).  The default workload is
BASELINE.json's T(64,16384,32) configuration - the one its target is quoted on; it fits one GPU.
Prints ONE JSON line on rank 0.  `--impl reference` times the CPU oracle on a bounded sample
(see DESIGN.md "Measurement").  N > 1: independent replicas, no collective (the
north star fixes "no sharding across GPUs and no collectives"); launched under torchrun, or by plain
`python bench.py --gpus N`, which starts the N ranks itself.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import gpipe_inputs as gi  # noqa: E402

METRIC = "tokens_per_sec_fwd_bwd"
UNIT = "tokens/s"
DEFAULT_WORKLOAD = "T(64,16384,32)"


# ---------------------------------------------------------------------------------------------
# FLOP model
# ---------------------------------------------------------------------------------------------
def flops_per_step(w, every_task=False):
    """model: forward + backward of the whole model; executed: what the engine runs - with re-materialization the
    replays too, minus the work it elides (readings A15, A15b, A15c; every_task=True: none elided)."""
    d, H, da, V, S = w.d_model, w.d_ffn, w.d_attn, w.vocab, w.seq_len
    T = w.tokens_per_step
    f_qkv, f_o, f_1, f_2 = 2 * d * 3 * da, 2 * da * d, 2 * d * H, 2 * H * d
    f_v = 2 * d * V
    n_dec = getattr(w, "n_dec", 0)
    # per layer and token: GEMM FLOPs f_g[l], attention FLOPs f_a[l] (causal: the unmasked half).  A decoder layer of
    # the encoder-decoder model adds the cross-attention block: q (d x da), k|v (d x 2 da) and
    # output (da x d) projections and one unmasked attention over the S memory positions.
    f_g, f_a = [], []
    for l, c in enumerate(w.causal):
        dec = n_dec > 0 and l >= w.n_layers - n_dec
        f_g.append(f_qkv + f_o + f_1 + f_2 + (2 * d * da + 2 * d * 2 * da + 2 * da * d if dec else 0))
        f_a.append(4 * S * da * ((S + 1) / (2 * S) if c else 1.0) + (4 * S * da if dec else 0))
    fwd_l = [g + a for g, a in zip(f_g, f_a)]
    model = (sum(fwd_l) + f_v + 2 * sum(f_g) + 2.5 * sum(f_a) + 2 * f_v) * T
    if not w.remat:
        return {"model": model, "executed": model}
    # cells of the equal split (the first L mod K cells get one more layer)
    L, K, M = w.n_layers, w.K, w.M
    base, extra = L // K, L % K
    lo = [k * base + min(k, extra) for k in range(K + 1)]
    executed = (2 * sum(f_g) + 2.5 * sum(f_a) + 2 * f_v) * T            # every backward task
    for k in range(K):
        cell = sum(fwd_l[lo[k]:lo[k + 1]]) + (f_v if k == K - 1 else 0.0)
        if every_task:
            executed += 2 * cell * T                                    # F(k, m) and R(k, m) for every m
        elif k == K - 1:
            executed += cell * T                                        # A15c: F(K-1, m) elided, R(K-1, m) runs (head included)
        else:
            # F(k, m) for every m; R(k, m) without the cell's last FFN2 (A15), and not for m = M-1 (A15b)
            executed += cell * T + (cell - (f_2 if lo[k + 1] > lo[k] else 0.0)) * T * (M - 1) / M
    return {"model": model, "executed": executed}


# ---------------------------------------------------------------------------------------------
# clocks
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()                      # the exact PID we started
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w": float(np.median(pw)) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


_T0 = time.perf_counter()


def progress(msg):
    """Phase marker on stderr (stdout carries only the JSON line)."""
    if int(os.environ.get("RANK", "0")) == 0:
        print("[bench %7.1fs] %s" % (time.perf_counter() - _T0, msg), file=sys.stderr, flush=True)


def ncu_traffic(kernel_key):
    """DRAM read+write bytes per launch of the dominant kernel from the committed ncu --set full capture
    (profiles/ncu_traffic.json, written by `python -m paper_1811_06965_b200.ncu_summary`); None when absent."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if not os.path.exists(p):
        return None, "absent: no profiles/ncu_traffic.json"
    try:
        j = json.load(open(p))
    except Exception as ex:                                   # a damaged file must not take the bench down
        return None, "absent: %s" % ex
    rec = j.get(kernel_key)
    if not rec:
        return None, "absent: no entry %r in profiles/ncu_traffic.json" % kernel_key
    return float(rec["dram_bytes_per_launch"]), "profiles/ncu_traffic.json[%s] (%s)" % (kernel_key, rec.get("source", "?"))


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        j = json.load(open(p))
        return {"burst": j["bf16_tflops"], "sustained": j.get("bf16_tflops_sustained", j["bf16_tflops"]),
                "hbm": j["hbm_gbs"], "src": "measured"}
    return {"burst": 1590.0, "sustained": 1400.0, "hbm": 6650.0, "src": "fallback"}


# ---------------------------------------------------------------------------------------------
# the oracle arm (cpu_baseline and --impl reference)
# ---------------------------------------------------------------------------------------------
def oracle_sample(w, repeats=2):
    """Times the CPU oracle, as it stands, on a bounded sample of the workload: ONE sequence
    through a 2-layer / 2-cell model of the same d, H, A, d_head, V, S (forward, replay,
    backward, head), and through the 0-layer model (embedding + head only); per-layer and head
    costs are separated and extrapolated linearly to the full depth (gradients are sums of
    independent per-sequence terms, so cost is linear in sequences and layers)."""
    from oracle import gpipe_oracle as go
    try:
        from threadpoolctl import threadpool_info
        cores = max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
    except Exception:
        cores = os.cpu_count() or 1

    def run(L):
        causal = tuple(w.causal[i * len(w.causal) // L] for i in range(L)) if L else ()
        ww = w.replace(n_layers=L, causal=causal, n_seqs=1, M=1, K=max(1, min(L, 2)))
        params = gi.make_params(ww, 1, parity=False, round_bf16=False)
        tok, lab = gi.make_tokens(ww, 2)
        o = go.GPipeOracle(go.Spec(ww.n_layers, ww.d_model, ww.d_ffn, ww.n_heads, ww.d_head, ww.vocab,
                                   ww.seq_len, ww.causal, ww.ln_eps), ww.K, 1, ww.remat, dtype=np.float32)
        o.set_params(params)
        o.step(tok, lab)                                    # BLAS thread pool / page-fault warm-up
        best = 1e30
        for _ in range(repeats):
            t0 = time.perf_counter()
            o.step(tok, lab)
            best = min(best, time.perf_counter() - t0)
        return best

    nl = min(4, w.n_layers)
    t_head = run(0)
    t_some = run(nl) if nl else t_head
    t_layer = max(t_some - t_head, 0.0) / max(nl, 1)
    t_seq = t_head + w.n_layers * t_layer                   # one sequence through the full depth
    value = w.seq_len / t_seq
    return {"value": value, "unit": UNIT, "cores": int(cores), "kind": "oracle",
            "sample": "fp32 numpy oracle step (forward, replay, backward) on 1 sequence of %d tokens: 0-layer model "
                      "(embedding+head) %.3fs, %d-layer/2-cell model %.3fs; per-layer cost extrapolated linearly to "
                      "%d layers" % (w.seq_len, t_head, nl, t_some, w.n_layers),
            "seconds": t_head + t_some}


def oracle_sample_encdec(w, repeats=2):
    """The bounded oracle sample for the encoder-decoder model (oracle/encdec_oracle.py as it stands): ONE source /
    target sequence pair through the (1 + 1)-layer and the (2 + 2)-layer model of the same widths; the cost of one
    encoder + decoder layer pair and the cost of embedding + head are separated and extrapolated linearly."""
    from oracle import encdec_oracle as eo
    try:
        from threadpoolctl import threadpool_info
        cores = max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
    except Exception:
        cores = os.cpu_count() or 1

    def run(L):
        ww = w.replace(n_layers=2 * L, n_dec=L, causal=(0,) * L + (1,) * L, n_seqs=1, M=1, K=2)
        params = gi.make_params(ww, 1, parity=False, round_bf16=False)
        ids = gi.make_tokens_encdec(ww, 2)
        o = eo.GPipeEncDecOracle(eo.EncDecSpec(L, L, ww.d_model, ww.d_ffn, ww.n_heads, ww.d_head, ww.vocab, ww.seq_len,
                                               ww.ln_eps, ww.logit_clip), 2, 1, ww.remat, dtype=np.float32)
        o.set_params(params)
        o.step(*ids)
        best = 1e30
        for _ in range(repeats):
            t0 = time.perf_counter()
            o.step(*ids)
            best = min(best, time.perf_counter() - t0)
        return best

    t1, t2 = run(1), run(2)
    t_pair = max(t2 - t1, 0.0)
    t_head = max(t1 - t_pair, 0.0)
    t_seq = t_head + (w.n_dec) * t_pair
    return {"value": w.seq_len / t_seq, "unit": UNIT, "cores": int(cores), "kind": "oracle",
            "sample": "fp32 numpy encoder-decoder oracle step on 1 sequence pair of %d tokens: (1+1)-layer model %.3fs, "
                      "(2+2)-layer model %.3fs; per-pair cost extrapolated linearly to %d+%d layers"
                      % (w.seq_len, t1, t2, w.n_enc, w.n_dec),
            "seconds": t1 + t2}


def oracle_full(w):
    """One WHOLE oracle step of the full workload (all N sequences, all L layers, the K/M schedule with replay),
    fp32, timed once after a one-sequence warm-up of the BLAS pool.  Minutes for config 2; do not use on 4/5."""
    from oracle import gpipe_oracle as go
    try:
        from threadpoolctl import threadpool_info
        cores = max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
    except Exception:
        cores = os.cpu_count() or 1
    params = gi.make_params(w, 1, parity=False, round_bf16=False)
    tok, lab = gi.make_tokens(w, 2)
    spec = go.Spec(w.n_layers, w.d_model, w.d_ffn, w.n_heads, w.d_head, w.vocab, w.seq_len, w.causal, w.ln_eps)
    warm = go.GPipeOracle(spec, w.K, 1, w.remat, dtype=np.float32)
    warm.set_params(params)
    warm.step(tok[:1], lab[:1])
    o = go.GPipeOracle(spec, w.K, w.M, w.remat, dtype=np.float32)
    o.set_params(params)
    t0 = time.perf_counter()
    loss = o.step(tok, lab)
    dt = time.perf_counter() - t0
    return {"value": w.tokens_per_step / dt, "unit": UNIT, "cores": int(cores), "kind": "oracle",
            "sample": "one full fp32 numpy oracle step of %s (%d sequences x %d tokens, K %d, M %d, remat %s): %.1f s, "
                      "loss %.4f" % (w.name, w.n_seqs, w.seq_len, w.K, w.M, w.remat, dt, loss),
            "seconds": dt}


def run_reference(args, w, rank, world):
    if rank != 0:
        return
    times = []
    res = None
    for i in range(args.warmup + args.steps):
        res = oracle_sample_encdec(w) if w.n_dec else (oracle_full(w) if args.oracle_full else oracle_sample(w))
        if i >= args.warmup:
            times.append(res["value"])
        if args.oracle_full:
            times = [res["value"]]                          # one full step is the measurement
            break
    value = float(np.mean(times))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * w.tokens_per_step / value,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "K": w.K, "M": w.M, "remat": w.remat, "n_seqs": w.n_seqs,
                       "seq_len": w.seq_len},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": res["cores"], "kind": "oracle",
                             "sample": res["sample"]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
def run_ours(args, w, rank, world, local_rank):
    import torch
    import paper_1811_06965_b200 as gp
    from paper_1811_06965_b200 import build
    from paper_1811_06965_b200.dist_util import max_over_ranks, barrier

    torch.cuda.set_device(local_rank)                    # before the first (NCCL) barrier
    dev = torch.device("cuda", local_rank)
    if rank == 0:
        build.build()
    barrier(world)
    peaks = measured_peaks()
    progress("library built and loaded; creating engine for %s" % w.name)
    torch.cuda.synchronize(dev)
    free_before, _ = torch.cuda.mem_get_info(dev)
    torch.cuda.reset_peak_memory_stats(dev)
    pipe_devices = [int(x) for x in args.pipeline_devices.split(",")] if args.pipeline_devices else None
    if w.n_dec:          # the encoder-decoder T(L,H,A): equal split, depth-scaled FFN init
        eng = gp.from_workload(w, device=dev, side_streams={'auto': None, 'on': True, 'off': False}[args.side_streams])
        eng.init_params(seed=1000 + rank, std=0.02, parity=False, ffn_scale=1.0 / w.n_layers)
        ids = gi.make_tokens_encdec(w, 2000 + rank)
    else:
        eng = gp.from_workload(w, device=dev, partition=None if args.partition == "equal" else args.partition,
                               devices=pipe_devices, staged=bool(pipe_devices) and args.pipeline_staged,
                               side_streams={'auto': None, 'on': True, 'off': False}[args.side_streams])
        eng.init_params(seed=1000 + rank, std=0.02, parity=False)
        ids = gi.make_tokens(w, 2000 + rank)
    progress("engine ready (%.1f GB arena)" % (eng.peak_bytes()["total"] / 1e9))
    ids_d = [torch.tensor(a, device=dev) for a in ids]
    ids_h = [torch.tensor(a).pin_memory().numpy() for a in ids]
    s0 = eng.streams[0]

    per_step = []

    def timed(fn, steps):
        barrier(world)
        torch.cuda.synchronize(dev)
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        evs[0].record(s0)                   # the engine starts and joins every step on stream 0
        for i in range(steps):
            fn()                            # gradients keep accumulating (no apply in fwd+bwd)
            evs[i + 1].record(s0)           # also the end of step i: min / median / max over the K steps
        torch.cuda.synchronize(dev)
        barrier(world)
        per_step[:] = [evs[i].elapsed_time(evs[i + 1]) for i in range(steps)]
        return max_over_ranks(evs[0].elapsed_time(evs[steps]), world)

    loss = None
    for i in range(args.warmup):
        loss = eng.step(*ids_d)
        eng.zero_grads()
        progress("warm-up step %d done, loss %.4f" % (i, loss))
    sampler = ClockSampler(local_rank) if rank == 0 else None
    l0 = eng.launch_count()
    ms = timed(lambda: eng.step(*ids_d), args.steps)
    launches = (eng.launch_count() - l0)
    clocks = sampler.stop() if sampler else None
    step_ms = sorted(per_step)
    progress("timed region done: %.1f ms/step" % (ms / args.steps))
    ms_e2e = timed(lambda: eng.step(*ids_h), args.steps)
    # two extra steps with per-launch CUDA events for the roofline of the dominant kernel class:
    # (1) "isolated": every cell on stream 0, each launch alone on the GPU (standalone durations);
    # (2) "in-step": the K-stream schedule as timed above, each launch bracketed on its own stream (durations
    #     then include the SMs it shares with the other cells' kernels)
    progress("e2e region done: %.1f ms/step; per-launch timing steps" % (ms_e2e / args.steps))
    eng.kernel_timing(True, serial=True)
    eng.step(*ids_d)
    stats = eng.kernel_stats()
    eng.kernel_timing(True, serial=False)
    eng.step(*ids_d)
    stats_conc = eng.kernel_stats()
    progress("per-launch timing steps done")
    eng.kernel_timing(False)
    # gpipe_apply_sgd, timed separately (the metric is forward + backward): 18 B of traffic per parameter
    ea0, ea1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_param_flat = sum(r * c for r, c in eng.shapes.values())
    if pipe_devices is None:
        torch.cuda.synchronize(dev)
        ea0.record(s0)
        eng.apply_sgd(0.0)                   # lr = 0: same traffic, parameters unchanged
        ea1.record(s0)
        torch.cuda.synchronize(dev)
        apply_ms = ea0.elapsed_time(ea1)
    else:
        apply_ms = None
    eng.zero_grads()
    peak_hbm = eng.peak_bytes()
    torch.cuda.synchronize(dev)
    free_after, _ = torch.cuda.mem_get_info(dev)
    hbm_check = {"gpipe_peak_bytes": peak_hbm["total"],
                 "torch_max_memory_allocated": int(torch.cuda.max_memory_allocated(dev)),
                 "cudaMemGetInfo_delta": int(free_before - free_after),
                 "note": "the arena is one torch allocation of gpipe_plan_bytes; the deltas also hold the id tensors "
                         "and the caching allocator's rounding"}

    tokens = w.tokens_per_step * world
    value = tokens * args.steps / (ms / 1e3)
    fl = flops_per_step(w, every_task=bool(int(os.environ.get("GPIPE_REPLAY_FULL", "0"))))
    step_s = ms / 1e3 / args.steps
    gem = {k: stats[k] for k in ("gemm_fwd", "gemm_dgrad", "gemm_wgrad")}
    gem_ms = sum(v["ms"] for v in gem.values())
    gem_fl = sum(v["flops"] for v in gem.values())
    tot_ms = sum(v["ms"] for v in stats.values())
    achieved = gem_fl / (gem_ms / 1e3) / 1e12 if gem_ms > 0 else 0.0
    traffic, traffic_src = ncu_traffic("gemm_tcgen05:ffn1_fwd")

    def per_class(st):
        return {k: {"launches": int(v["launches"]), "ms": round(v["ms"], 3),
                    "tflops": (v["flops"] / v["ms"] / 1e9) if v["ms"] > 0 and v["flops"] > 0 else None,
                    "gbs": (v["bytes"] / v["ms"] / 1e6) if v["ms"] > 0 else None}
                for k, v in st.items()}

    n_gemm = int(sum(v["launches"] for v in gem.values()))
    # in-step regime: what the timed step achieves on the tensor cores - all GEMM + attention FLOPs it executes,
    # over the step's device time (K streams co-running; HBM-bound kernels share the same clock)
    tens_fl = sum(v["flops"] for v in stats.values())
    gem_c_ms = sum(stats_conc[k]["ms"] for k in gem)
    # The headline `roofline` is the regime that is TIMED: the K-stream step.  Its launches overlap on the SMs, so a
    # per-launch duration there is not a standalone kernel time; achieved = all tensor FLOPs the step executes (GEMM +
    # attention, counted per launch by the library) / the step's device time, against the sustained bf16 peak.  The
    # nested "isolated" regime times every launch alone (one extra step serialised on one stream) - with the tile
    # selection of the 16-cell step (256 x 512 tiles wherever eligible), which is tuned for SM-time under co-running
    # cells, not for single-launch latency: a 16-tile launch then runs on 32 SMs.
    in_step_achieved = tens_fl / step_s / 1e12
    roofline = {"bound": "tensor", "kernel": "gemm_tcgen05_pair_kernel (fwd + dgrad + wgrad launches; %.0f %% of the "
                                             "step's tensor FLOPs, the rest is the tcgen05 attention)" % (100.0 * gem_fl / tens_fl),
                "regime": "in-step",
                "regime_note": "the timed K-stream schedule: executed tensor FLOPs (GEMM + attention) / step device "
                               "time; per_class durations are per-launch events on the launch's own stream while the "
                               "other cells' kernels share the SMs",
                "achieved": in_step_achieved, "peak": peaks["sustained"], "unit": "TFLOP/s",
                "frac": in_step_achieved / peaks["sustained"],
                "peak_src": peaks["src"] + " sustained bf16 (kernel timed inside a long step)",
                "frac_of_burst": in_step_achieved / peaks["burst"],
                "traffic": traffic, "traffic_src": traffic_src,
                "launches": n_gemm,
                "gemm_share_of_stream_time": gem_c_ms / sum(v["ms"] for v in stats_conc.values()) if stats_conc else None,
                "per_class": per_class(stats_conc),
                "isolated": {"regime": "isolated",
                             "regime_note": "each launch timed alone on the GPU (all cells serialised on one stream, one "
                                            "extra step, same tile selection as the 16-cell step); achieved = sum of "
                                            "2MNK / sum of GEMM launch durations",
                             "achieved": achieved, "peak": peaks["sustained"], "unit": "TFLOP/s",
                             "frac": achieved / peaks["sustained"], "frac_of_burst": achieved / peaks["burst"],
                             "avg_launch_us": 1e3 * gem_ms / n_gemm if n_gemm else None,
                             "share_of_kernel_time": gem_ms / tot_ms if tot_ms else None,
                             "per_class": per_class(stats)}}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "ms_per_step_min_median_max": [step_ms[0], step_ms[len(step_ms) // 2], step_ms[-1]] if step_ms else None,
            "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16" if w.dtype == "bf16" else "f32", "data": "synthetic",
            "config": {"workload": w.name, "L": w.n_layers, "n_enc": w.n_enc if w.n_dec else None, "n_dec": w.n_dec or None,
                       "d_model": w.d_model, "d_ffn": w.d_ffn,
                       "n_heads": w.n_heads, "d_head": w.d_head, "vocab": w.vocab, "seq_len": w.seq_len,
                       "n_seqs": w.n_seqs, "K": w.K, "M": w.M, "remat": w.remat, "partition": args.partition,
                       "layers_per_cell": [hi - lo for lo, hi in eng.cells],
                       "parallelism": ("pipeline over devices %s%s" % (pipe_devices, " (staged boundary copies)" if args.pipeline_staged else ""))
                       if pipe_devices else ("replicas" if world > 1 else "1 GPU, K streams"),
                       "side_streams": bool(getattr(eng, "side_streams", False)),
                       "l2": "inputs larger than L2 (activations+weights per step >> 126 MB)"},
            "loss": loss,
            "tflops_executed": fl["executed"] / step_s / 1e12, "tflops_model": fl["model"] / step_s / 1e12,
            "executed_flops_per_step": {"formula": fl["executed"], "engine_count": tens_fl,
                                        "note": "formula: flops_per_step (DESIGN.md section 9); engine_count: sum of 2MNK / attention "
                                                "FLOPs over every launch of one step, counted by the library (gpipe_kernel_stats)"},
            "frac_of_bf16_peak_executed": fl["executed"] / step_s / 1e12 / peaks["burst"],
            "frac_of_sustained_executed": fl["executed"] / step_s / 1e12 / peaks["sustained"],
            "frac_of_nominal_2250_executed": fl["executed"] / step_s / 1e12 / 2250.0,
            "apply_sgd": {"ms": apply_ms, "gbs": (18.0 * n_param_flat / apply_ms / 1e6) if apply_ms else None,
                          "note": "gpipe_apply_sgd timed separately (not part of tokens/s): 18 B per parameter"},
            "mfu_model_flops": fl["model"] / step_s / 1e12 / peaks["burst"],
            "peak_tflops_burst": peaks["burst"], "peak_tflops_sustained": peaks["sustained"],
            "peak_hbm_bytes": peak_hbm["total"], "peak_hbm_by_category": peak_hbm["by_category"],
            "peak_hbm_cross_check": hbm_check,
            "clocks": clocks, "roofline": roofline,
            "e2e": {"value": tokens * args.steps / (ms_e2e / 1e3), "unit": UNIT,
                    "h2d_bytes_per_step": int(sum(a.nbytes for a in ids)), "d2h_bytes_per_step": 4 * w.M},
            "gpu_launches": int(launches)}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        progress("timing the CPU oracle sample")
        res = oracle_sample_encdec(w) if w.n_dec else (oracle_full(w) if args.oracle_full else oracle_sample(w))
        line["cpu_baseline"] = {k: v for k, v in res.items() if k != "seconds"}
    eng.close()
    if rank == 0:
        print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=gi.CONFIG_ORDER + list(gi.ENCDEC_CONFIGS),
                    help="a BASELINE.json config, or the paper's own encoder-decoder T(64,16384,32) (PAPER.md:158-160)")
    ap.add_argument("--M", type=int, default=None)
    ap.add_argument("--K", type=int, default=None)
    ap.add_argument("--no-remat", action="store_true")
    ap.add_argument("--d-head", type=int, default=None,
                    help="variant row of reading A3: d_head = d_model / n_heads = 32 for the 32-head configs (d_attn 1024)")
    ap.add_argument("--partition", default="equal", choices=["equal", "cost"],
                    help="equal: L/K consecutive layers per cell; cost: minimum variance of the estimated cell costs (PAPER.md:65)")
    ap.add_argument("--pipeline-devices", default=None,
                    help="comma-separated CUDA device ordinals, one per cell: run the step on the pipeline handle "
                         "(gpipe_create_pipeline; PAPER.md:65) from THIS process; ordinals may repeat")
    ap.add_argument("--pipeline-staged", action="store_true", help="force staged boundary copies when cells share a device")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--side-streams", choices=("auto", "on", "off"), default="auto",
                    help="a second stream per cell for the weight-gradient GEMMs (gpipe_env.n_streams = 2K); auto: the "
                         "binding's default (on for K <= 2)")
    ap.add_argument("--oracle-full", action="store_true",
                    help="cpu_baseline / --impl reference: one WHOLE oracle step of the workload instead of the bounded "
                         "sample (config 2: minutes; BASELINE.md section 3)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    w = gi.CONFIGS[args.workload] if args.workload in gi.CONFIGS else gi.ENCDEC_CONFIGS[args.workload]
    if args.M:
        w = w.replace(M=args.M)
    if args.K:
        w = w.replace(K=args.K)
    if args.no_remat:
        w = w.replace(remat=False)
    if args.d_head:
        w = w.replace(d_head=args.d_head, name="%s d_head=%d" % (w.name, args.d_head))
    if args.impl == "reference":
        run_reference(args, w, rank, world)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: start the N replica ranks ourselves, one per GPU, over NCCL
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE is %d" % (args.gpus, world))
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl")
    try:
        run_ours(args, w, rank, world, local_rank)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()

"""Writes tests/golden/bf16_floor.json: the bf16 noise floor of the reduced parity cases of
BASELINE.json configs 2-5, computed by the CPU oracle ALONE (this script imports nothing from the
CUDA package and needs no GPU).

    python tests/golden/make_bf16_floor.py ["T(6,4096,16)" ...]        # default: all four

What it stores (reading A14 (iii)): for each case the oracle is run twice on the same
seeded inputs - plain, and with `round_operands=True` (RNE-bf16 rounding at the points where the
CUDA path stores a tensor in bf16) - and for every tensor of the canonical list
the cosine between the two gradients is recorded, plus both losses and, per layer, the fraction of
ReLU units of micro-batch 0 whose sign differs between the two runs.  `tests/test_gpu_configs.py`
reads these values as the floor a bf16 implementation can be held to: a GPU gradient passes with
cosine >= 0.999, or >= floor - 5e-4 where the floor itself is below 0.999.
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from tests.util import REDUCED_CASES, cosine, reduced_case, run_oracle  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "bf16_floor.json")


def floor_of(name):
    w, params, tok, lab, dt = reduced_case(name)
    res = {}
    masks = {}
    grads = {}
    for tag, rnd in (("plain", False), ("rounded", True)):
        t0 = time.time()
        from oracle import gpipe_oracle as go
        from tests.util import oracle_spec
        o = go.GPipeOracle(oracle_spec(w), w.K, w.M, w.remat, dtype=dt, round_operands=rnd)
        o.keep_relu_masks = True
        o.set_params(params)
        res["loss_" + tag] = o.step(tok, lab)
        masks[tag] = {l: o.relu_masks[(l, 0)] for l in range(w.n_layers)}
        o.relu_masks = {}
        grads[tag] = o.g
        print("%s %s: %.1f s, loss %.6f" % (name, tag, time.time() - t0, res["loss_" + tag]), flush=True)
    cos = {n: cosine(grads["rounded"][n], grads["plain"][n]) for n in grads["plain"]}
    res["floor_cosine"] = cos
    res["min"] = min(cos.values())
    res["median"] = float(np.median(list(cos.values())))
    res["relu_mismatch_m0"] = {str(l): float((masks["plain"][l] != masks["rounded"][l]).mean())
                               for l in range(w.n_layers)}
    res["oracle_dtype"] = REDUCED_CASES[name]["oracle_dtype"]
    res["workload"] = {k: getattr(w, k) for k in ("n_layers", "d_model", "d_ffn", "n_heads", "d_head", "vocab",
                                                   "seq_len", "n_seqs", "M", "K")}
    res["workload"]["causal"] = list(w.causal)
    res["seeds"] = {k: REDUCED_CASES[name][k] for k in ("seed_p", "seed_t")}
    return res


def main():
    names = sys.argv[1:] or list(REDUCED_CASES)
    out = json.load(open(OUT)) if os.path.exists(OUT) else {}
    for name in names:
        out[name] = floor_of(name)
        with open(OUT, "w") as f:
            json.dump(out, f, indent=1, sort_keys=True)
            f.write("\n")
        print("%s: floor min cosine %.6f, median %.6f" % (name, out[name]["min"], out[name]["median"]), flush=True)


if __name__ == "__main__":
    main()

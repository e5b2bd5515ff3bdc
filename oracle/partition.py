"""Oracle for GPipe's cell partitioning - TEST INFRASTRUCTURE ONLY (imported by tests/, never by the
product path; shares no code with the CUDA library).

PAPER.md:59 (2.1): a cell is a run of "consecutive layers between layers i and j", its cost is the sum of its
layers' costs c_i.  PAPER.md:65 (2.2): "the partitioning algorithm minimizes the variance in the estimated cost
of all cells in order to maximize the efficiency of the pipeline by syncing the computation time across all
partitions".  The paper gives no algorithm, so the oracle is the definition written out: enumerate EVERY way to
cut L layers into K consecutive non-empty cells, compute the population variance of the K cell costs, keep
the smallest (brute force: fine for the L <= 14 the tests use).  SURVEY.md 8(f) f2: the embedding adds its cost
to the first cell and the head (final LayerNorm + logits + loss) to the last.

layer_costs() restates the per-token FLOP model of SURVEY.md 8(d):
    F_g = 2 (4 d d_a + 2 d H)   the four linear layers        F_a = 4 S d_a  (x (S+1)/(2S) if causal)
    F_v = 2 d V                 the vocabulary head
    forward = F_g + F_a,  backward = 2 F_g + 2.5 F_a,  replay (remat) = forward again
"""
from itertools import combinations
from typing import List, Sequence, Tuple


def cell_costs(layer_cost: Sequence[float], bounds: Sequence[int], first_extra: float, last_extra: float) -> List[float]:
    K = len(bounds) - 1
    out = []
    for k in range(K):
        c = 0.0
        for l in range(bounds[k], bounds[k + 1]):
            c += layer_cost[l]
        if k == 0:
            c += first_extra
        if k == K - 1:
            c += last_extra
        out.append(c)
    return out


def variance(xs: Sequence[float]) -> float:
    mean = sum(xs) / len(xs)
    return sum((x - mean) * (x - mean) for x in xs) / len(xs)


def all_partitions(L: int, K: int):
    """Every boundary vector [0, b_1 < ... < b_{K-1}, L] with non-empty consecutive cells, in lexicographic order."""
    for cuts in combinations(range(1, L), K - 1):
        yield [0] + list(cuts) + [L]


def min_variance_partition(layer_cost: Sequence[float], K: int, first_extra: float = 0.0,
                           last_extra: float = 0.0) -> Tuple[List[int], float]:
    """Brute force over all consecutive partitions; the first (lexicographically smallest) minimiser wins."""
    best, best_var = None, None
    for b in all_partitions(len(layer_cost), K):
        v = variance(cell_costs(layer_cost, b, first_extra, last_extra))
        if best_var is None or v < best_var:
            best, best_var = b, v
    return best, best_var


def layer_costs(n_layers, d_model, d_ffn, n_heads, d_head, vocab, seq_len, causal, remat) -> Tuple[List[float], float, float]:
    d, H, da, V, S = float(d_model), float(d_ffn), float(n_heads * d_head), float(vocab), float(seq_len)
    f_g = 2.0 * (4.0 * d * da + 2.0 * d * H)
    f_v = 2.0 * d * V
    costs = []
    for l in range(n_layers):
        f_a = 4.0 * S * da * ((S + 1.0) / (2.0 * S) if causal[l] else 1.0)
        fwd, bwd = f_g + f_a, 2.0 * f_g + 2.5 * f_a
        costs.append(fwd + bwd + (fwd if remat else 0.0))
    head = f_v + 2.0 * f_v + (f_v if remat else 0.0)
    return costs, 0.0, head


def layer_costs_encdec(n_enc, n_dec, d_model, d_ffn, n_heads, d_head, vocab, seq_len, remat) -> Tuple[List[float], float, float]:
    """The same per-token FLOP model for the encoder-decoder T(L,H,A) (oracle/encdec_oracle.py, reading B1):
    an encoder layer is the unmasked layer above; a decoder layer is the causal layer plus the cross-attention block -
    q (d x d_a), k | v (d x 2 d_a) and output (d_a x d) projections, 2 * 4 d d_a FLOPs, and one unmasked attention over
    the S memory positions, 4 S d_a."""
    d, H, da, V, S = float(d_model), float(d_ffn), float(n_heads * d_head), float(vocab), float(seq_len)
    f_g = 2.0 * (4.0 * d * da + 2.0 * d * H)
    f_x = 2.0 * (4.0 * d * da)
    f_v = 2.0 * d * V
    costs = []
    for l in range(n_enc + n_dec):
        dec = l >= n_enc
        g = f_g + (f_x if dec else 0.0)
        a = 4.0 * S * da * ((S + 1.0) / (2.0 * S) if dec else 1.0) + (4.0 * S * da if dec else 0.0)
        fwd, bwd = g + a, 2.0 * g + 2.5 * a
        costs.append(fwd + bwd + (fwd if remat else 0.0))
    head = f_v + 2.0 * f_v + (f_v if remat else 0.0)
    return costs, 0.0, head

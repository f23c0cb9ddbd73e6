"""Token sampling for the oracle (TEST INFRASTRUCTURE).

The paper gives only the settings (train: T=0.6, top-p 1.0, top-k -1; eval: T=0.7, top-p 0.8,
top-k 20 - PAPER.md L295-301, Table 3). BASELINE.json north_star (g) fixes the mechanism:
"temperature/top-p, Gumbel-max on seeded uniforms supplied as inputs". Reading R10:

  greedy (T == 0):  y = lowest-index argmax_v z_v
  otherwise:        score_v = z_v / T + g_v,  g_v = -ln(-log1p(-u_v));
                    y = lowest-index argmax of score over the kept set;
                    kept set = all ids if top_p >= 1, else the shortest prefix of ids sorted by
                    descending softmax(z/T) (ties: lower id first) whose cumulative probability
                    reaches top_p (never empty).
  top-k (R18):      PAPER.md Table 3 (L299-301) evaluates with top-k 20 next to top-p 0.8 and trains with top-k -1. The
                    paper does not say how the two filters compose; reading R18 takes the usual order of its
                    generation engine: top-k first (the k ids of largest z / T, ties: lower id first; k <= 0 or
                    k >= V: no filter), then top-p on the distribution renormalised over those k ids.
  log-prob:         log softmax(z / T')[y], T' = T (1 if greedy) - the distribution actually sampled
                    from, before any top-p / top-k truncation (R11).
"""
import numpy as np

from .rng import gumbel_from_uniform


def log_softmax(z):
    z = np.asarray(z, dtype=np.float64)
    m = np.max(z)
    return z - (m + np.log(np.sum(np.exp(z - m))))


def log_prob(z, y, temperature):
    """log softmax(z/T')[y] with T' = T, or 1 when greedy (T == 0)."""
    t = float(temperature) if temperature > 0 else 1.0
    return float(log_softmax(np.asarray(z, dtype=np.float64) / t)[int(y)])


def kept_set_top_p(z, temperature, top_p):
    """Boolean mask of ids kept by nucleus filtering (all True if top_p >= 1)."""
    z = np.asarray(z, dtype=np.float64)
    V = z.shape[0]
    if top_p >= 1.0:
        return np.ones(V, dtype=bool)
    t = float(temperature) if temperature > 0 else 1.0
    p = np.exp(log_softmax(z / t))
    order = np.lexsort((np.arange(V), -p))          # descending p, ties: lower id first
    cum = np.cumsum(p[order])
    n_keep = int(np.searchsorted(cum, top_p, side="left")) + 1   # shortest prefix with cum >= top_p
    n_keep = min(max(n_keep, 1), V)
    keep = np.zeros(V, dtype=bool)
    keep[order[:n_keep]] = True
    return keep


def kept_set(z, temperature, top_p=1.0, top_k=0):
    """Boolean mask of the ids the Gumbel argmax runs over: top-k first, then top-p on the renormalised rest (R18)."""
    z = np.asarray(z, dtype=np.float64)
    V = z.shape[0]
    keep = np.ones(V, dtype=bool)
    if 0 < top_k < V:
        order = np.lexsort((np.arange(V), -z))        # descending z (the order of z / T for T > 0), ties: lower id first
        keep = np.zeros(V, dtype=bool)
        keep[order[:top_k]] = True
    if top_p < 1.0:
        zz = np.where(keep, z, -np.inf)               # softmax over the kept ids only
        keep = keep & kept_set_top_p(zz, temperature, top_p)
    return keep


def sample_token(z, temperature, top_p, u, top_k=0):
    """One token from logits z. `u`: float32 uniforms [V] (ignored when greedy)."""
    z = np.asarray(z, dtype=np.float64)
    if temperature <= 0:
        return int(np.argmax(z))                    # np.argmax returns the lowest index among ties
    score = z / float(temperature) + gumbel_from_uniform(u)
    if top_p < 1.0 or top_k > 0:
        score = np.where(kept_set(z, temperature, top_p, top_k), score, -np.inf)
    return int(np.argmax(score))

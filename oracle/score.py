"""Teacher-forced scoring with the oracle (TEST INFRASTRUCTURE).

Used to compare a token stream produced elsewhere (the CUDA path's own sampling, bf16 configs)
with what the definition gives on that same stream: PAPER.md L61 - every y_t is drawn from
pi_{a_t}(. | x.y_<t), so given (x, y_1..y_n, a_1..a_n) the owner's logits at every step are fixed
by one causal full-recompute forward per model (DESIGN.md §5 procedure VII.3).
"""
import numpy as np


def teacher_forced_logits(model, prompt, tokens):
    """Logits z_t (t = 1..n) predicting y_t from x.y_<t, for one model: [n, V]."""
    prompt = [int(x) for x in prompt]
    tokens = [int(x) for x in tokens]
    ctx = prompt + tokens[:-1]
    P = len(prompt)
    positions = np.arange(P - 1, P - 1 + len(tokens))
    return model.forward_full(ctx, positions=positions)


def replay_owner_logits(models, prompt, tokens, owners):
    """The *owner's* logits at each generated position: row t-1 comes from models[owners[t-1]]."""
    per_model = [None, None]
    owners = np.asarray(owners)
    out = None
    for m in (0, 1):
        if np.any(owners == m):
            per_model[m] = teacher_forced_logits(models[m], prompt, tokens)
            if out is None:
                out = np.empty_like(per_model[m])
            out[owners == m] = per_model[m][owners == m]
    return out


def overlap_from_logits(z_sen, z_jun, temperature=1.0):
    """alpha = sum_v min(p_sen(v), p_jun(v)) with p = softmax(z / T') - PAPER.md L134 (section 4.4.2, after
    Leviathan et al. 2023): "the probability mass both models assign to the same tokens", 0 = disjoint, 1 = identical."""
    from .sampler import log_softmax
    t = float(temperature) if temperature > 0 else 1.0
    ps = np.exp(log_softmax(np.asarray(z_sen, dtype=np.float64) / t))
    pj = np.exp(log_softmax(np.asarray(z_jun, dtype=np.float64) / t))
    return float(np.sum(np.minimum(ps, pj)))


def dual_score(models, tokens, temperature=1.0):
    """Teacher-forced dual scoring of one finished token stream y_0..y_{L-1} (prompt and response alike) under both
    models (reading R17 in DESIGN.md section 3). For every position i >= 1:

      sen_logp[i] = log p_sen(y_i | y_<i)                      (the senior's log-prob at *all* positions)
      jun_logp[i] = log p_jun(y_i | y_<i)                      (the junior's per-token cross-entropy on
                                                                a stream is the mean of -jun_logp over its positions)
      overlap[i]  = sum_v min(p_sen(v | y_<i), p_jun(v | y_<i))  (the token-level overlap alpha)

    with p = softmax(z / T'), T' = temperature (1.0: the models' own distributions). Entry 0 of each array is 0:
    the first token has no prediction. One causal full-recompute forward per model."""
    from .sampler import log_softmax
    tokens = [int(x) for x in tokens]
    L = len(tokens)
    out = {k: np.zeros(L, dtype=np.float64) for k in ("sen_logp", "jun_logp", "overlap")}
    if L < 2:
        return out
    t = float(temperature) if temperature > 0 else 1.0
    z = [m.forward_full(tokens[:-1]) for m in models]            # row i-1 predicts y_i
    for i in range(1, L):
        ls = log_softmax(z[0][i - 1] / t)
        lj = log_softmax(z[1][i - 1] / t)
        out["sen_logp"][i] = ls[tokens[i]]
        out["jun_logp"][i] = lj[tokens[i]]
        out["overlap"][i] = np.sum(np.minimum(np.exp(ls), np.exp(lj)))
    return out

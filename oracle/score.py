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

"""Seeded generators. Random data only - no arithmetic of the method."""
import numpy as np
import torch

_LAYER_TENSORS = ("attn_norm", "wq", "wk", "wv", "wo", "mlp_norm", "w_gate", "w_up", "w_down")


def _layer_shapes(s):
    qd, kd = s.n_q_heads * s.head_dim, s.n_kv_heads * s.head_dim
    return dict(attn_norm=(s.hidden,), wq=(qd, s.hidden), wk=(kd, s.hidden), wv=(kd, s.hidden),
                wo=(s.hidden, qd), mlp_norm=(s.hidden,), w_gate=(s.intermediate, s.hidden),
                w_up=(s.intermediate, s.hidden), w_down=(s.hidden, s.intermediate))


def make_weights(shape, seed, device="cpu", std=0.02, gain_jitter=0.0):
    """Random-init weights, row-major [out_features, in_features]: matrices N(0, std^2), norm gains
    1 (+ gain_jitter * N(0,1) when asked, to make a dropped gain visible in tests). dtype follows
    shape.dtype (bf16: drawn in float32 then rounded). One generator per tensor, so a tensor's
    values depend only on (seed, its index), not on generation order."""
    dt = torch.float32 if shape.dtype == "f32" else torch.bfloat16
    dev = torch.device(device)
    counter = [0]

    def draw(shp, is_gain):
        g = torch.Generator(device=dev)
        g.manual_seed(int(seed) * 1000003 + counter[0])
        counter[0] += 1
        if is_gain:
            t = torch.ones(shp, dtype=torch.float32, device=dev)
            if gain_jitter:
                t += gain_jitter * torch.randn(shp, generator=g, dtype=torch.float32, device=dev)
        else:
            t = torch.randn(shp, generator=g, dtype=torch.float32, device=dev) * std
        return t.to(dt).contiguous()

    w = dict(embed=draw((shape.vocab, shape.hidden), False),
             lm_head=draw((shape.vocab, shape.hidden), False),
             final_norm=draw((shape.hidden,), True), layers=[])
    ls = _layer_shapes(shape)
    for _ in range(shape.n_layers):
        w["layers"].append({n: draw(ls[n], n.endswith("norm")) for n in _LAYER_TENSORS})
    return w


def make_word_start(vocab, frac, seed):
    """uint8[vocab], 1 = the id begins a new word. Stand-in for the leading-space-marker set of the
    tokenizer (~53k of 151k ids); i.i.d. Bernoulli(frac)."""
    return (np.random.default_rng(seed).random(vocab) < frac).astype(np.uint8)


def make_prompts(workload, seed=None):
    """List of int32 id arrays, one per sequence; each of the n_prompts prompts is repeated `group`
    times consecutively (the G rollouts of a prompt)."""
    w = workload
    rng = np.random.default_rng(w.seeds["prompts"] if seed is None else seed)
    out = []
    for _ in range(w.n_prompts):
        n = int(rng.integers(w.prompt_len[0], w.prompt_len[1] + 1))
        ids = rng.integers(0, w.shape.vocab, size=n, dtype=np.int64).astype(np.int32)
        out.extend([ids.copy() for _ in range(w.group)])
    return out


def make_max_new(workload, seed=None):
    """int32[B]: the cap, or min(Geometric(1/geom_mean), cap) for the ragged-termination configs."""
    w = workload
    if w.geom_mean <= 0:
        return np.full(w.batch, w.max_new, dtype=np.int32)
    rng = np.random.default_rng(w.seeds["lengths"] if seed is None else seed)
    return np.minimum(rng.geometric(1.0 / w.geom_mean, size=w.batch), w.max_new).astype(np.int32)


def make_explicit_uniforms(batch, max_new, vocab, seed):
    """Explicit position-addressed uniforms in (0,1) as float32:
    u_switch [B, max_new + 1] (index t, t = 0 is the a_1 draw), u_sample [B, max_new, vocab] (index t-1)."""
    rng = np.random.default_rng(seed)
    lo, hi = np.float32(2.0 ** -30), np.float32(1.0 - 2.0 ** -24)
    usw = np.clip(rng.random((batch, max_new + 1), dtype=np.float32), lo, hi)
    usa = np.clip(rng.random((batch, max_new, vocab), dtype=np.float32), lo, hi)
    return usw, usa


def flatten_prompts(prompts):
    """CSR form: (int32 tokens, int64 offsets[B+1])."""
    off = np.zeros(len(prompts) + 1, dtype=np.int64)
    off[1:] = np.cumsum([len(p) for p in prompts])
    return np.concatenate(prompts).astype(np.int32), off

"""Decoder-only transformer forward in float64 NumPy (TEST INFRASTRUCTURE).

The paper names only the checkpoint family and says the two policies are
"decoder-only transformers with the same architecture" in BASELINE.json's wording; the
dimensions come from BASELINE.json's configs. Architecture reading R12:
pre-norm residual blocks, RMSNorm with learned gain, rotary embedding with half-split
pairing (j, j + d/2) over the full head_dim, scale 1/sqrt(d), causal softmax, grouped-query
attention (q-head a reads kv-head a // (n_q/n_kv)), SwiGLU MLP, no biases, untied LM head.

For ids x_0..x_{n-1} (position of prompt token 0 is 0):
    h_i = E[x_i]
    per layer:  u = RMSNorm(h; g_attn),  u_j = h_j g_j / sqrt(mean_j h_j^2 + eps)
                q = W_q u, k = W_k u, v = W_v u;  RoPE on q, k at position i:
                   phi = i * theta^(-2j/d);  (z_j, z_{j+d/2}) <- (z_j cos - z_{j+d/2} sin, z_{j+d/2} cos + z_j sin)
                s_ij = q_i . k_j / sqrt(d) (j <= i), softmax over j, o_i = sum_j p_ij v_j
                h <- h + W_o concat(o);  u = RMSNorm(h; g_mlp)
                h <- h + W_down( silu(W_gate u) * (W_up u) ),  silu(a) = a / (1 + exp(-a))
    logits z = W_head RMSNorm(h_{n-1}; g_final)

Two evaluation orders of the same definition, which must agree (pin 4, tests/test_oracle_model.py):
  * `forward_full`   - recompute everything on the whole prefix ("both states
                       condition on the same history" - the history *is* the definition);
  * `KVState.extend` - incremental: append K/V of new positions (any chunk length, which is what
                       a model does when it catches up on its partner's tokens) and attend.

`round_bf16=True` is the rounding-point-faithful mode (DESIGN.md §3 R-V): float64 arithmetic with
round-to-nearest-even bf16 applied at exactly the points where the bf16 CUDA path stores bf16
(GEMM A-operands and the KV cache). It is used only for the sharp kernel-correctness check.
`round_qp=True` (only with `round_bf16`) adds the two rounding points of the tensor-core attention path
that R-V names: the RoPE'd queries are stored as bf16, and the softmax numerators exp(s - max) enter
the P.V product as bf16 while the denominator is summed from the unrounded values:
o_i = sum_j bf16(e_ij) v_j / sum_j e_ij. (A tiled online softmax rounds e relative to its running
maximum, which is the same relative rounding, not the same bits; so this mode is statistically, not
bitwise, faithful for P.)
"""
import numpy as np


def _to_f64(a):
    """Any array-like (NumPy array, or a torch tensor incl. bfloat16) -> float64 ndarray, exactly."""
    if isinstance(a, np.ndarray):
        return a.astype(np.float64, copy=False)
    if hasattr(a, "detach"):                      # torch tensor, without importing torch here
        t = a.detach().cpu()
        try:
            import torch
            return t.to(torch.float64).numpy()
        except Exception:                         # pragma: no cover
            return np.asarray(t.tolist(), dtype=np.float64)
    return np.asarray(a, dtype=np.float64)


def round_to_bf16(x):
    """float64 -> float32 (RNE) -> bf16 (RNE on the dropped 16 bits) -> float64. The intermediate
    float32 step is deliberate: the bf16 CUDA path holds these values in float32 before it stores
    bf16, so this is the same two-step rounding (it differs from a direct float64->bf16 rounding
    only when the float32 value lands exactly on a bf16 tie)."""
    f = np.asarray(x, dtype=np.float64).astype(np.float32)
    b = f.view(np.uint32).astype(np.uint64)
    lsb = (b >> np.uint64(16)) & np.uint64(1)
    b = (b + np.uint64(0x7FFF) + lsb) & np.uint64(0xFFFF0000)
    return b.astype(np.uint32).view(np.float32).astype(np.float64)


def rms_norm(h, g, eps):
    """u_j = h_j g_j / sqrt(mean_j h_j^2 + eps), rows of h."""
    ms = np.mean(h * h, axis=-1, keepdims=True)
    return h * g / np.sqrt(ms + eps)


def rope(z, positions, theta):
    """z: [n, heads, d]; rotate pairs (j, j + d/2) by phi = pos * theta^(-2j/d)."""
    d = z.shape[-1]
    half = d // 2
    j = np.arange(half, dtype=np.float64)
    inv_freq = theta ** (-2.0 * j / d)
    phi = np.asarray(positions, dtype=np.float64)[:, None] * inv_freq[None, :]      # [n, half]
    c = np.cos(phi)[:, None, :]
    s = np.sin(phi)[:, None, :]
    a = z[..., :half]
    b = z[..., half:]
    return np.concatenate([a * c - b * s, b * c + a * s], axis=-1)


def silu(a):
    return a / (1.0 + np.exp(-a))


def softmax_rows(s):
    m = np.max(s, axis=-1, keepdims=True)
    e = np.exp(s - m)
    return e / np.sum(e, axis=-1, keepdims=True)


class KVState:
    """Per-model cache of post-RoPE keys and values for one sequence: k[l], v[l] are [n, n_kv, d]."""

    def __init__(self, n_layers):
        self.k = [None] * n_layers
        self.v = [None] * n_layers
        self.n = 0              # number of context positions ingested ("ing[M]" in DESIGN.md §2)


class OracleModel:
    def __init__(self, cfg, weights, round_bf16=False, cache=True, round_qp=False):
        self.cfg = cfg
        self.w = weights
        self.round_bf16 = bool(round_bf16)
        self.round_qp = bool(round_qp) and self.round_bf16
        self._cache = {} if cache else None

    # -- weight access: float64 view of the values as given ------------------------------------
    def _W(self, name, layer=None):
        key = (name, layer)
        if self._cache is not None and key in self._cache:
            return self._cache[key]
        a = self.w[name] if layer is None else self.w["layers"][layer][name]
        a = _to_f64(a)
        if self._cache is not None:
            self._cache[key] = a
        return a

    def _rb(self, x):
        return round_to_bf16(x) if self.round_bf16 else x

    # -- one pass over `tokens` placed at absolute positions pos0.., on top of an optional cache -----
    def _blocks(self, tokens, pos0, state):
        c = self.cfg
        tokens = np.asarray(tokens, dtype=np.int64)
        n_new = tokens.shape[0]
        nq, nkv, d = c.n_q_heads, c.n_kv_heads, c.head_dim
        group = nq // nkv
        positions = np.arange(pos0, pos0 + n_new)
        h = self._W("embed")[tokens]                                   # [n_new, H]
        for l in range(c.n_layers):
            u = self._rb(rms_norm(h, self._W("attn_norm", l), c.rms_eps))
            q = (u @ self._W("wq", l).T).reshape(n_new, nq, d)
            k = (u @ self._W("wk", l).T).reshape(n_new, nkv, d)
            v = (u @ self._W("wv", l).T).reshape(n_new, nkv, d)
            q = rope(q, positions, c.rope_theta)
            if self.round_qp:
                q = round_to_bf16(q)
            k = self._rb(rope(k, positions, c.rope_theta))
            v = self._rb(v)
            if state is not None:
                if state.k[l] is None:
                    kk, vv = k, v
                else:
                    kk = np.concatenate([state.k[l], k], axis=0)
                    vv = np.concatenate([state.v[l], v], axis=0)
                state.k[l], state.v[l] = kk, vv
            else:
                kk, vv = k, v
            n_ctx = kk.shape[0]                                        # keys end at position pos0 + n_new - 1
            o = np.empty((n_new, nq, d), dtype=np.float64)
            kpos = np.arange(n_ctx) + (pos0 + n_new - n_ctx)           # absolute key positions
            causal = kpos[None, :] <= positions[:, None]               # [n_new, n_ctx]
            for a in range(nq):
                g = a // group
                s = (q[:, a, :] @ kk[:, g, :].T) / np.sqrt(d)          # [n_new, n_ctx]
                s = np.where(causal, s, -np.inf)
                if self.round_qp:                                      # bf16 numerators, unrounded denominator (R-V)
                    e = np.exp(s - np.max(s, axis=-1, keepdims=True))
                    o[:, a, :] = (round_to_bf16(e) @ vv[:, g, :]) / np.sum(e, axis=-1, keepdims=True)
                else:
                    p = softmax_rows(s)
                    o[:, a, :] = p @ vv[:, g, :]
            o = self._rb(o.reshape(n_new, nq * d))
            h = h + o @ self._W("wo", l).T
            u = self._rb(rms_norm(h, self._W("mlp_norm", l), c.rms_eps))
            act = self._rb(silu(u @ self._W("w_gate", l).T) * (u @ self._W("w_up", l).T))
            h = h + act @ self._W("w_down", l).T
        return h

    def _head(self, h_rows):
        c = self.cfg
        u = self._rb(rms_norm(h_rows, self._W("final_norm"), c.rms_eps))
        return u @ self._W("lm_head").T

    # -- public ------------------------------------------------------------------------------------
    def forward_full(self, tokens, positions=None):
        """Logits [len(positions), V] predicting the token after each listed position (default: all),
        by full recompute on `tokens`."""
        h = self._blocks(tokens, 0, None)
        if positions is None:
            return self._head(h)
        return self._head(h[np.asarray(positions, dtype=np.int64)])

    def next_logits_full(self, tokens):
        """Logits for position len(tokens) given the whole context, full recompute."""
        return self.forward_full(tokens, positions=[len(tokens) - 1])[0]

    def new_state(self):
        return KVState(self.cfg.n_layers)

    def extend(self, state, new_tokens):
        """Ingest `new_tokens` at positions state.n.. (any chunk length >= 1); returns the logits
        after the last of them. This is the incremental / catch-up evaluation order."""
        new_tokens = np.asarray(new_tokens, dtype=np.int64)
        assert new_tokens.shape[0] >= 1
        h = self._blocks(new_tokens, state.n, state)
        state.n += new_tokens.shape[0]
        return self._head(h[-1:])[0]

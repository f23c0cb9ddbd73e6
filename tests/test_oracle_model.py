"""Pins for oracle/model.py: library-routine cross-check (pin 7), closed forms (pin 8), incremental ==
full recompute (pin 4), log-softmax identities (pin 10), scalar brute force on a micro model."""
import math

import numpy as np
import torch
import torch.nn.functional as F

from oracle import OracleModel
from oracle.model import rms_norm, rope, silu, softmax_rows, round_to_bf16
from oracle.sampler import log_softmax, log_prob
from workloads import ModelShape, make_weights, get_workload

MICRO = ModelShape(2, 16, 4, 2, 8, 24, 40, 1e-6, 1e4, "f32")


def _model(shape, seed, **kw):
    return OracleModel(shape, make_weights(shape, seed, gain_jitter=0.2, std=0.3 if shape is MICRO else 0.02), **kw)


# ---------------------------------------------------------------------------------------------- pin 7
def _torch_library_forward(shape, w, tokens):
    """Independent composition of library routines in float64: F.rms_norm, F.scaled_dot_product_attention
    (causal, GQA), F.silu, RoPE as a complex rotation (torch.polar)."""
    s = shape
    T = len(tokens)
    d, nq, nkv = s.head_dim, s.n_q_heads, s.n_kv_heads
    f = lambda t: t.to(torch.float64)
    h = f(w["embed"])[torch.as_tensor(tokens)]
    pos = torch.arange(T, dtype=torch.float64)
    inv = torch.as_tensor([s.rope_theta ** (-2.0 * j / d) for j in range(d // 2)], dtype=torch.float64)
    rot = torch.polar(torch.ones(T, d // 2, dtype=torch.float64), pos[:, None] * inv[None, :])   # e^{i phi}

    def rope_c(x):                                   # x [T, heads, d]; pairs (j, j+d/2) as complex numbers
        z = torch.complex(x[..., : d // 2], x[..., d // 2:]) * rot[:, None, :]
        return torch.cat([z.real, z.imag], dim=-1)

    for L in w["layers"]:
        u = F.rms_norm(h, (s.hidden,), f(L["attn_norm"]), s.rms_eps)
        q = rope_c(F.linear(u, f(L["wq"])).view(T, nq, d))
        k = rope_c(F.linear(u, f(L["wk"])).view(T, nkv, d))
        v = F.linear(u, f(L["wv"])).view(T, nkv, d)
        o = F.scaled_dot_product_attention(q.transpose(0, 1)[None], k.transpose(0, 1)[None], v.transpose(0, 1)[None],
                                           is_causal=True, enable_gqa=True)[0].transpose(0, 1).reshape(T, nq * d)
        h = h + F.linear(o, f(L["wo"]))
        u = F.rms_norm(h, (s.hidden,), f(L["mlp_norm"]), s.rms_eps)
        h = h + F.linear(F.silu(F.linear(u, f(L["w_gate"]))) * F.linear(u, f(L["w_up"])), f(L["w_down"]))
    return F.linear(F.rms_norm(h, (s.hidden,), f(w["final_norm"]), s.rms_eps), f(w["lm_head"])).numpy()


def test_forward_matches_library_routines_cfg1_shape():
    shape = get_workload("cfg1_tiny_f32").shape
    w = make_weights(shape, 1, gain_jitter=0.1)
    tokens = np.random.default_rng(0).integers(0, shape.vocab, size=23)
    z = OracleModel(shape, w).forward_full(tokens)
    zl = _torch_library_forward(shape, w, tokens)
    assert z.shape == zl.shape == (23, shape.vocab)
    assert np.max(np.abs(z - zl)) <= 1e-9 * max(1.0, np.max(np.abs(zl)))


def test_forward_matches_library_routines_micro_big_weights():
    w = make_weights(MICRO, 5, std=0.4, gain_jitter=0.3)
    tokens = np.random.default_rng(1).integers(0, MICRO.vocab, size=11)
    z = OracleModel(MICRO, w).forward_full(tokens)
    zl = _torch_library_forward(MICRO, w, tokens)
    assert np.max(np.abs(z - zl)) <= 1e-9 * np.max(np.abs(zl))


# ------------------------------------------------------------------------- scalar brute force, micro
def _scalar_forward(shape, w, tokens):
    """Pure-Python scalar loops with explicit indices (no array ops): catches transposed operands,
    wrong head mapping, wrong RoPE pairing."""
    s = shape
    H, d, nq, nkv, I = s.hidden, s.head_dim, s.n_q_heads, s.n_kv_heads, s.intermediate
    g = nq // nkv
    W = lambda t: t.to(torch.float64).tolist()
    emb, head, fn = W(w["embed"]), W(w["lm_head"]), W(w["final_norm"])
    T = len(tokens)
    h = [[emb[tok][j] for j in range(H)] for tok in tokens]

    def norm(x, gain):
        ms = sum(v * v for v in x) / len(x)
        return [x[j] * gain[j] / math.sqrt(ms + s.rms_eps) for j in range(len(x))]

    def matvec(M, x):
        return [sum(M[o][i] * x[i] for i in range(len(x))) for o in range(len(M))]

    def rot(vec, pos):
        out = list(vec)
        for j in range(d // 2):
            phi = pos * s.rope_theta ** (-2.0 * j / d)
            a, b = vec[j], vec[j + d // 2]
            out[j] = a * math.cos(phi) - b * math.sin(phi)
            out[j + d // 2] = b * math.cos(phi) + a * math.sin(phi)
        return out

    for L in w["layers"]:
        an, mn = W(L["attn_norm"]), W(L["mlp_norm"])
        wq, wk, wv, wo = W(L["wq"]), W(L["wk"]), W(L["wv"]), W(L["wo"])
        wg, wu, wd = W(L["w_gate"]), W(L["w_up"]), W(L["w_down"])
        qs, ks, vs = [], [], []
        for i in range(T):
            u = norm(h[i], an)
            q, k, v = matvec(wq, u), matvec(wk, u), matvec(wv, u)
            qs.append([rot(q[a * d:(a + 1) * d], i) for a in range(nq)])
            ks.append([rot(k[a * d:(a + 1) * d], i) for a in range(nkv)])
            vs.append([v[a * d:(a + 1) * d] for a in range(nkv)])
        for i in range(T):
            o = []
            for a in range(nq):
                kvh = a // g
                sc = [sum(qs[i][a][e] * ks[j][kvh][e] for e in range(d)) / math.sqrt(d) for j in range(i + 1)]
                m = max(sc)
                ex = [math.exp(x - m) for x in sc]
                Z = sum(ex)
                o.extend(sum(ex[j] / Z * vs[j][kvh][e] for j in range(i + 1)) for e in range(d))
            att = matvec(wo, o)
            h[i] = [h[i][j] + att[j] for j in range(H)]
        for i in range(T):
            u = norm(h[i], mn)
            gt, up = matvec(wg, u), matvec(wu, u)
            act = [gt[j] / (1.0 + math.exp(-gt[j])) * up[j] for j in range(I)]
            dn = matvec(wd, act)
            h[i] = [h[i][j] + dn[j] for j in range(H)]
    return [matvec(head, norm(h[i], fn)) for i in range(T)]


def test_forward_matches_scalar_loops_micro():
    w = make_weights(MICRO, 9, std=0.3, gain_jitter=0.2)
    tokens = [3, 17, 17, 39, 0]
    z = OracleModel(MICRO, w).forward_full(tokens)
    zs = np.asarray(_scalar_forward(MICRO, w, tokens))
    assert np.max(np.abs(z - zs)) <= 1e-10 * max(1.0, np.max(np.abs(zs)))


# ---------------------------------------------------------------------------------------------- pin 4
def test_incremental_equals_full_recompute_any_chunking():
    m = _model(MICRO, 3)
    tokens = np.random.default_rng(2).integers(0, MICRO.vocab, size=20)
    zf = m.forward_full(tokens)
    for chunks in ([20], [1] * 20, [7, 1, 1, 5, 6], [16, 4], [1, 19]):
        st = m.new_state()
        off = 0
        for c in chunks:
            z = m.extend(st, tokens[off:off + c])
            off += c
            assert np.max(np.abs(z - zf[off - 1])) <= 1e-9 * np.max(np.abs(zf))
        assert st.n == 20


def test_incremental_equals_full_cfg1_shape():
    shape = get_workload("cfg1_tiny_f32").shape
    m = OracleModel(shape, make_weights(shape, 2))
    tokens = np.random.default_rng(3).integers(0, shape.vocab, size=40)
    st = m.new_state()
    m.extend(st, tokens[:16])
    for i in range(16, 40):
        z = m.extend(st, tokens[i:i + 1])
        assert np.max(np.abs(z - m.next_logits_full(tokens[:i + 1]))) <= 1e-10


# ---------------------------------------------------------------------------------------------- pin 8
def test_rope_closed_forms():
    rng = np.random.default_rng(0)
    z = rng.standard_normal((5, 3, 8))
    assert np.allclose(rope(z, np.zeros(5), 1e4), z, atol=0)                       # position 0 = identity
    r = rope(z, np.arange(5) * 37, 1e4)
    assert np.allclose(np.linalg.norm(r, axis=-1), np.linalg.norm(z, axis=-1))     # rotation preserves norms
    # q.k depends on the position difference only
    q, k = rng.standard_normal((1, 1, 8)), rng.standard_normal((1, 1, 8))
    d0 = np.sum(rope(q, [9], 1e4) * rope(k, [4], 1e4))
    d1 = np.sum(rope(q, [109], 1e4) * rope(k, [104], 1e4))
    assert abs(d0 - d1) < 1e-12
    # the pair is (j, j + d/2), rotated by pos * theta^(-2j/d): check one coordinate by hand
    e = np.zeros((1, 1, 8)); e[0, 0, 1] = 1.0                                      # unit vector on j = 1
    out = rope(e, [3], 1e4)[0, 0]
    phi = 3 * 1e4 ** (-2 * 1 / 8)
    assert abs(out[1] - math.cos(phi)) < 1e-15 and abs(out[5] - math.sin(phi)) < 1e-15
    assert np.count_nonzero(np.abs(out) > 1e-15) == 2


def test_shift_invariance_of_logits():
    """RoPE makes attention depend on relative positions only: evaluating the same tokens at
    positions shifted by a constant leaves the logits unchanged."""
    m = _model(MICRO, 4)
    tokens = np.random.default_rng(5).integers(0, MICRO.vocab, size=9)
    h0 = m._blocks(tokens, 0, None)
    h1 = m._blocks(tokens, 1234, None)
    assert np.max(np.abs(m._head(h0) - m._head(h1))) < 1e-9


def test_norm_softmax_silu_closed_forms():
    g = np.array([1.0, 2.0, 3.0, 4.0])
    assert np.allclose(rms_norm(np.full((1, 4), 2.0), g, 0.0), g)                   # constant vector -> gains
    assert np.allclose(rms_norm(np.full((1, 4), -3.0), g, 7.0), -3.0 * g / 4.0)      # sqrt(9 + 7) = 4
    x = np.array([[3.0, 4.0]])
    assert np.allclose(rms_norm(x, np.ones(2), 0.0), x / math.sqrt(12.5))
    p = softmax_rows(np.random.default_rng(0).standard_normal((6, 11)) * 5)
    assert np.allclose(p.sum(-1), 1.0) and np.all(p > 0)
    assert np.allclose(softmax_rows(np.array([[0.0, math.log(3.0)]])), [[0.25, 0.75]])
    assert silu(0.0) == 0.0 and abs(silu(1.0) - 1.0 / (1.0 + math.exp(-1.0))) < 1e-15
    assert abs(silu(-2.0) + 2.0 / (1.0 + math.exp(2.0))) < 1e-15


def test_single_token_attention_returns_v_and_hand_swiglu():
    """One layer, one token: softmax over a single key is 1, so the attention output is v itself:
    h1 = h0 + W_o W_v u. With W_o = 0 the block reduces to the SwiGLU MLP, checked by hand."""
    s = ModelShape(1, 2, 1, 1, 2, 2, 3, 0.0, 1e4, "f32")
    w = make_weights(s, 0)
    L = w["layers"][0]
    w["embed"] = torch.tensor([[3.0, 4.0], [1.0, 0.0], [0.0, 2.0]])
    L["attn_norm"] = torch.tensor([1.0, 1.0]); L["mlp_norm"] = torch.tensor([1.0, 1.0]); w["final_norm"] = torch.tensor([1.0, 1.0])
    L["wq"] = torch.eye(2); L["wk"] = torch.eye(2)
    L["wv"] = torch.tensor([[0.0, 1.0], [1.0, 0.0]])                     # swaps coordinates
    L["wo"] = torch.tensor([[2.0, 0.0], [0.0, 2.0]])
    L["w_gate"] = torch.zeros(2, 2); L["w_up"] = torch.zeros(2, 2); L["w_down"] = torch.zeros(2, 2)
    w["lm_head"] = torch.tensor([[1.0, 0.0], [0.0, 1.0], [1.0, 1.0]])
    z = OracleModel(s, w).forward_full([0])[0]
    u = np.array([3.0, 4.0]) / math.sqrt(12.5)
    h1 = np.array([3.0, 4.0]) + 2.0 * u[::-1]                            # v = swap(u); W_o doubles
    f = h1 / math.sqrt(np.mean(h1 * h1))
    assert np.allclose(z, [f[0], f[1], f[0] + f[1]], atol=1e-14)
    # MLP only
    L["wo"] = torch.zeros(2, 2)
    L["w_gate"] = torch.tensor([[1.0, 0.0], [0.0, -1.0]]); L["w_up"] = torch.tensor([[0.0, 1.0], [1.0, 1.0]])
    L["w_down"] = torch.tensor([[1.0, 2.0], [0.0, -1.0]])
    z = OracleModel(s, w).forward_full([0])[0]
    gate = np.array([u[0], -u[1]]); up = np.array([u[1], u[0] + u[1]])
    act = gate / (1 + np.exp(-gate)) * up
    h1 = np.array([3.0, 4.0]) + np.array([act[0] + 2 * act[1], -act[1]])
    f = h1 / math.sqrt(np.mean(h1 * h1))
    assert np.allclose(z, [f[0], f[1], f[0] + f[1]], atol=1e-14)


# --------------------------------------------------------------------------------------------- pin 10
def test_log_softmax_identities():
    z = np.random.default_rng(0).standard_normal(512) * 3
    lp = log_softmax(z)
    assert abs(np.sum(np.exp(lp)) - 1.0) < 1e-12
    assert np.allclose(lp, torch.log_softmax(torch.as_tensor(z), -1).numpy(), atol=1e-12)
    assert abs(log_prob(z, 17, 0.6) - torch.log_softmax(torch.as_tensor(z) / 0.6, -1)[17].item()) < 1e-12
    assert abs(log_prob(z, 17, 0.0) - lp[17]) < 1e-15                              # greedy => T' = 1


def test_round_to_bf16_matches_torch():
    x = np.random.default_rng(0).standard_normal(10000) * np.exp(np.random.default_rng(1).uniform(-20, 20, 10000))
    ref = torch.as_tensor(x).to(torch.float32).to(torch.bfloat16).to(torch.float64).numpy()
    assert np.array_equal(round_to_bf16(x), ref)
    m = OracleModel(MICRO, make_weights(MICRO, 3), round_bf16=True)
    t = np.arange(6)
    assert 0 < np.max(np.abs(m.forward_full(t) - OracleModel(MICRO, m.w).forward_full(t))) < 0.05


def test_round_qp_mode_pins():
    """`round_qp` (DESIGN.md section 3 R-V: bf16 queries, bf16 softmax numerators over an unrounded denominator).
    (a) a single key has softmax 1 whatever the query, and 1 is a bf16 number: identical to `round_bf16` alone;
    (b) with an independent torch composition of one attention head (bf16 casts by torch) on values chosen so
        that nothing else rounds; (c) the perturbation of the logits is of the size of a bf16 ulp, not zero."""
    m0 = OracleModel(MICRO, make_weights(MICRO, 3), round_bf16=True)
    m1 = OracleModel(MICRO, m0.w, round_bf16=True, round_qp=True)
    assert np.array_equal(m0.forward_full([5]), m1.forward_full([5]))
    assert not OracleModel(MICRO, m0.w, round_qp=True).round_qp                      # needs round_bf16
    t = np.arange(9)
    d = np.max(np.abs(m0.forward_full(t) - m1.forward_full(t)))
    assert 0 < d < 0.05
    # (b) one layer, one head, identity projections except W_v; W_o = W_down = 0 would hide the head, so read the
    # attention output through W_o = I and a zero MLP: h1 = h0 + o.
    s = ModelShape(1, 4, 1, 1, 4, 4, 4, 0.0, 1e4, "f32")
    w = make_weights(s, 0)
    L = w["layers"][0]
    rng = np.random.default_rng(5)
    E = torch.as_tensor(rng.standard_normal((4, 4)))
    w["embed"] = E.clone()
    for n in ("attn_norm", "mlp_norm"):
        L[n] = torch.ones(4, dtype=torch.float64)
    w["final_norm"] = torch.ones(4, dtype=torch.float64)
    L["wq"] = torch.eye(4, dtype=torch.float64); L["wk"] = torch.eye(4, dtype=torch.float64); L["wv"] = torch.eye(4, dtype=torch.float64)
    L["wo"] = torch.eye(4, dtype=torch.float64)
    L["w_gate"] = torch.zeros(4, 4, dtype=torch.float64); L["w_up"] = torch.zeros(4, 4, dtype=torch.float64); L["w_down"] = torch.zeros(4, 4, dtype=torch.float64)
    w["lm_head"] = torch.eye(4, dtype=torch.float64)
    toks = [0, 1, 2, 3]
    z = OracleModel(s, w, round_bf16=True, round_qp=True).forward_full(toks)
    bf = lambda x: x.to(torch.float32).to(torch.bfloat16).to(torch.float64)
    h = E[toks]
    u = bf(h / torch.sqrt((h * h).mean(-1, keepdim=True)))
    pos = torch.arange(4, dtype=torch.float64)
    inv = torch.as_tensor([1e4 ** (-2.0 * j / 4) for j in range(2)], dtype=torch.float64)
    ang = pos[:, None] * inv[None, :]
    rot = lambda x: torch.cat([x[:, :2] * torch.cos(ang) - x[:, 2:] * torch.sin(ang), x[:, 2:] * torch.cos(ang) + x[:, :2] * torch.sin(ang)], -1)
    q, k, v = bf(rot(u)), bf(rot(u)), bf(u)
    sc = (q @ k.T) / 2.0
    sc = sc.masked_fill(torch.triu(torch.ones(4, 4, dtype=torch.bool), 1), float("-inf"))
    e = torch.exp(sc - sc.max(-1, keepdim=True).values)
    o = bf((bf(e) @ v) / e.sum(-1, keepdim=True))
    h1 = h + o
    f = bf(h1 / torch.sqrt((h1 * h1).mean(-1, keepdim=True)))        # MLP is zero; final norm, then the identity head
    assert np.allclose(z, f.numpy(), atol=1e-12)

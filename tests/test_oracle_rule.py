"""Pins for oracle/rule.py: closed form at p=1 (pin 2), change-only-after-word-start invariant and cap
(pin 3), role swap (pin 5), brute force over coin outcomes vs a hand-written transition table (pin 12),
run-length and senior-share laws (pins 11, 13), DRAW start, EOS stop, both modes."""
import itertools

import numpy as np
import pytest

from oracle import (SENIOR, JUNIOR, DRAW, TOGGLE, REDRAW, TandemParams, OracleModel, owners_from_tokens,
                    tandem_generate)
from oracle.rule import Uniforms
from workloads import ModelShape, make_weights, make_word_start

S, J = SENIOR, JUNIOR

# PAPER.md L61 written out as a table: NEXT[mode][(a_t, y_t begins a word, coin u<p)] = a_{t+1}
NEXT = {
    TOGGLE: {(S, 0, 0): S, (S, 0, 1): S, (J, 0, 0): J, (J, 0, 1): J,
             (S, 1, 0): S, (S, 1, 1): J, (J, 1, 0): J, (J, 1, 1): S},
    REDRAW: {(S, 0, 0): S, (S, 0, 1): S, (J, 0, 0): J, (J, 0, 1): J,      # "if y_t does not begin a new word, a_{t+1} = a_t"
             (S, 1, 0): J, (S, 1, 1): S, (J, 1, 0): J, (J, 1, 1): S},     # "set to the senior with probability p and to the junior otherwise"
}


def _uni_from_coins(coins, p=0.5):
    """u_switch row with u < p exactly where coins[t] == 1 (index t = 0..n)."""
    return Uniforms(u_switch=[np.where(np.asarray(coins) == 1, np.float32(p / 2), np.float32((1 + p) / 2))])


@pytest.mark.parametrize("mode", [TOGGLE, REDRAW])
@pytest.mark.parametrize("start", [S, J])
def test_brute_force_all_coin_outcomes(mode, start):
    ws = np.array([0, 1, 0, 1, 1, 0, 0, 1], dtype=np.uint8)
    tokens = [1, 0, 3, 4, 2, 7, 5, 6]                       # flags: 1 0 1 1 0 1 0 0
    n = len(tokens)
    for coins in itertools.product([0, 1], repeat=n + 1):
        params = TandemParams(p=0.5, switch_mode=mode, start_owner=start)
        got = owners_from_tokens(tokens, ws, params, _uni_from_coins(coins))
        a, exp = start, []
        for t in range(1, n + 1):
            exp.append(a)
            a = NEXT[mode][(a, int(ws[tokens[t - 1]]), coins[t])]
        assert got.tolist() == exp


def test_toggle_p1_closed_form_and_p0_constant():
    rng = np.random.default_rng(0)
    ws = make_word_start(100, 0.3, 1)
    tokens = rng.integers(0, 100, size=500)
    uni = Uniforms(seed=5)
    o = owners_from_tokens(tokens, ws, TandemParams(p=1.0, switch_mode=TOGGLE, start_owner=S), uni)
    exp = np.zeros(500, dtype=np.uint8)
    for t in range(1, 500):
        exp[t] = exp[t - 1] ^ ws[tokens[t - 1]]             # owner[t+1] = owner[t] XOR word_start[y_t]
    assert np.array_equal(o, exp)
    assert not owners_from_tokens(tokens, ws, TandemParams(p=0.0, switch_mode=TOGGLE, start_owner=S), uni).any()
    assert owners_from_tokens(tokens, ws, TandemParams(p=0.0, switch_mode=TOGGLE, start_owner=J), uni).all()
    # REDRAW: p=1 => senior from the first redraw on (all senior if started senior); p=0 => junior after it
    assert not owners_from_tokens(tokens, ws, TandemParams(p=1.0, switch_mode=REDRAW, start_owner=S), uni).any()
    o = owners_from_tokens(tokens, ws, TandemParams(p=0.0, switch_mode=REDRAW, start_owner=S), uni)
    first = int(np.argmax(ws[tokens] == 1))
    assert not o[:first + 1].any() and o[first + 1:].all()


@pytest.mark.parametrize("mode", [TOGGLE, REDRAW])
@pytest.mark.parametrize("p", [0.1, 0.5, 0.9])
def test_owner_changes_only_after_word_start(mode, p):
    rng = np.random.default_rng(1)
    ws = make_word_start(1000, 0.3, 2)
    for b in range(8):
        tokens = rng.integers(0, 1000, size=400)
        o = owners_from_tokens(tokens, ws, TandemParams(p=p, switch_mode=mode), Uniforms(seed=9), b=b)
        changed = np.nonzero(o[1:] != o[:-1])[0]           # index t-1 such that a_{t+1} != a_t
        assert len(changed) > 0
        assert np.all(ws[tokens[changed]] == 1)


def test_cap_bounds_runs_without_redraw():
    ws = np.zeros(50, dtype=np.uint8)                       # no boundary token at all
    tokens = np.random.default_rng(0).integers(0, 50, size=300)
    K = 32
    p = TandemParams(p=1.0, switch_mode=TOGGLE, cap_k=K)
    o = owners_from_tokens(tokens, ws, p, Uniforms(seed=1))
    # p=1 TOGGLE flips at every redraw position; with no boundaries those are exactly every K tokens
    exp = (np.arange(300) // K) % 2
    assert np.array_equal(o, exp)
    # cap off: never changes
    assert not owners_from_tokens(tokens, ws, TandemParams(p=1.0, cap_k=0), Uniforms(seed=1)).any()
    # a boundary resets the counter: boundary at t=10 => flips after 10, then every K after that
    ws2 = ws.copy(); ws2[7] = 1
    tok2 = np.where(np.arange(300) == 9, 7, np.where(tokens == 7, 8, tokens))
    o2 = owners_from_tokens(tok2, ws2, p, Uniforms(seed=1))
    exp2 = np.zeros(300, dtype=int); a = 0; c = 0
    for t in range(1, 301):
        exp2[t - 1] = a
        b = t == 10
        c = 0 if b else c + 1
        if b or c >= K:
            a ^= 1; c = 0
    assert np.array_equal(o2, exp2)
    # maximum run between owner changes is K
    runs = np.diff(np.nonzero(np.diff(o2))[0])
    assert runs.max() <= K


def test_draw_start_and_eos():
    ws = make_word_start(64, 0.5, 0)
    tokens = [5, 9, 13, 2, 40, 41]
    for b in range(20):
        uni = Uniforms(seed=3)
        u0 = uni.switch(b, 0)
        for mode in (TOGGLE, REDRAW):
            o = owners_from_tokens(tokens, ws, TandemParams(p=0.5, switch_mode=mode, start_owner=DRAW), uni, b=b)
            assert o[0] == (S if u0 < np.float32(0.5) else J)
    # p extremes with DRAW: u is never 0 or 1
    assert owners_from_tokens(tokens, ws, TandemParams(p=0.0, start_owner=DRAW), Uniforms(seed=3))[0] == J
    assert owners_from_tokens(tokens, ws, TandemParams(p=1.0, start_owner=DRAW, switch_mode=REDRAW), Uniforms(seed=3))[0] == S
    # EOS: emitted, flagged, no entry after it
    o = owners_from_tokens(tokens, ws, TandemParams(p=1.0, eos_id=13), Uniforms(seed=3))
    assert o[3:].tolist() == [0, 0, 0] and len(o) == 6      # positions after the EOS are left untouched (zero)


def test_senior_share_and_run_length_laws():
    """TOGGLE, i.i.d. boundary flags at rate f: switch rate per token = f p, mean run = 1/(f p);
    senior share ~ 0.5 (PAPER.md L494 reports mean 50.0% for Bernoulli(0.5) handoffs)."""
    f, p, n, B = 0.3, 0.5, 2048, 128
    rng = np.random.default_rng(0)
    ws = make_word_start(5000, f, 7)
    f_emp = ws.mean()
    shares, switches = [], 0
    for b in range(B):
        tokens = rng.integers(0, 5000, size=n)
        o = owners_from_tokens(tokens, ws, TandemParams(p=p), Uniforms(seed=21), b=b)
        shares.append(1.0 - o.mean())
        switches += int(np.count_nonzero(o[1:] != o[:-1]))
    rate = switches / (B * (n - 1))
    assert abs(rate - f_emp * p) < 0.004                    # 0.150 expected
    assert abs(np.mean(shares) - 0.5) < 0.01
    assert 0.015 < np.std(shares) < 0.045                   # ~2.7% predicted for f=0.3, 2048 tokens
    # REDRAW: senior share = p
    sh = []
    for b in range(32):
        tokens = rng.integers(0, 5000, size=n)
        o = owners_from_tokens(tokens, ws, TandemParams(p=0.9, switch_mode=REDRAW), Uniforms(seed=22), b=b)
        sh.append(1.0 - o.mean())
    assert abs(np.mean(sh) - 0.9) < 0.01


# ---- rollouts with models --------------------------------------------------------------------------
MICRO = ModelShape(2, 16, 4, 2, 8, 24, 40, 1e-6, 1e4, "f32")


def _pair():
    return (OracleModel(MICRO, make_weights(MICRO, 1, std=0.3, gain_jitter=0.2)),
            OracleModel(MICRO, make_weights(MICRO, 2, std=0.3, gain_jitter=0.2)))


def _prompts(n=3):
    rng = np.random.default_rng(4)
    return [rng.integers(0, MICRO.vocab, size=int(rng.integers(3, 9))) for _ in range(n)]


@pytest.mark.parametrize("temperature", [0.0, 1.0])
def test_generate_consistent_with_integer_replay_and_full_recompute(temperature):
    sen, jun = _pair()
    ws = make_word_start(MICRO.vocab, 0.4, 3)
    prm = TandemParams(p=0.5, temperature=temperature, seed=17)
    prompts = _prompts()
    inc = tandem_generate((sen, jun), prm, prompts, [12] * 3, ws, want_logits=True)
    full = tandem_generate((sen, jun), prm, prompts, [12] * 3, ws, mode="full", want_logits=True)
    for b in range(3):
        assert np.array_equal(inc["tokens"][b], full["tokens"][b])                  # pin 4 on whole rollouts
        assert np.array_equal(inc["owner"][b], full["owner"][b])
        assert np.allclose(inc["sen_logp"][b], full["sen_logp"][b], atol=1e-9)
        for z0, z1 in zip(inc["logits"][b], full["logits"][b]):
            assert np.max(np.abs(z0 - z1)) < 1e-9
        o = owners_from_tokens(inc["tokens"][b], ws, prm, Uniforms(seed=17), b=b)
        assert np.array_equal(o, inc["owner"][b])
        assert np.array_equal(inc["mask"][b], 1 - inc["owner"][b])                  # m_t = 1[a_t = sen]
        assert np.all(inc["sen_logp"][b][inc["owner"][b] == J] == 0)
        assert np.all(inc["sen_logp"][b][inc["owner"][b] == S] < 0)
    assert len(set(np.concatenate(inc["owner"]).tolist())) == 2                      # both models did emit


def test_role_swap_symmetry():
    sen, jun = _pair()
    ws = make_word_start(MICRO.vocab, 0.4, 3)
    prompts = _prompts()
    a = tandem_generate((sen, jun), TandemParams(p=0.5, start_owner=S, seed=5), prompts, [10] * 3, ws)
    b = tandem_generate((jun, sen), TandemParams(p=0.5, start_owner=J, seed=5), prompts, [10] * 3, ws)
    for i in range(3):
        assert np.array_equal(a["tokens"][i], b["tokens"][i])
        assert np.array_equal(a["owner"][i], 1 - b["owner"][i])


def test_eos_stops_and_forced_tokens():
    sen, jun = _pair()
    ws = make_word_start(MICRO.vocab, 0.4, 3)
    prompts = _prompts(1)
    forced = [np.array([4, 7, 9, 11, 13, 2])]
    out = tandem_generate((sen, jun), TandemParams(p=0.5, eos_id=11, seed=1), prompts, [6], ws, forced=forced)
    assert out["tokens"][0].tolist() == [4, 7, 9, 11]                               # EOS recorded, then stop
    assert len(out["owner"][0]) == 4

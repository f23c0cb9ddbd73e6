"""Pins 1 and 6: the tandem rollout degenerates to solo decoding where the paper/BASELINE.json say it must."""
import numpy as np
import pytest

from oracle import (SENIOR, JUNIOR, TOGGLE, REDRAW, TandemParams, OracleModel, tandem_generate, solo_generate)
from workloads import ModelShape, make_weights, make_word_start, get_workload, make_prompts, make_explicit_uniforms
from oracle.rule import Uniforms

MICRO = ModelShape(2, 16, 4, 2, 8, 24, 40, 1e-6, 1e4, "f32")


def _mk(seed):
    return OracleModel(MICRO, make_weights(MICRO, seed, std=0.3, gain_jitter=0.2))


def _prompts():
    rng = np.random.default_rng(8)
    return [rng.integers(0, MICRO.vocab, size=int(rng.integers(2, 7))) for _ in range(3)]


@pytest.mark.parametrize("temperature,top_p", [(0.0, 1.0), (1.0, 1.0), (0.8, 0.7)])
def test_p0_toggle_and_p1_redraw_reproduce_solo_senior(temperature, top_p):
    """BASELINE.json north_star: 'With p=0 it must reproduce solo senior decoding token for token'."""
    sen, jun = _mk(1), _mk(2)
    ws = make_word_start(MICRO.vocab, 0.4, 3)
    prompts = _prompts()
    for mode, p in ((TOGGLE, 0.0), (REDRAW, 1.0)):
        prm = TandemParams(p=p, switch_mode=mode, start_owner=SENIOR, temperature=temperature, top_p=top_p, seed=3)
        t = tandem_generate((sen, jun), prm, prompts, [14] * 3, ws)
        s = solo_generate(sen, prm, prompts, [14] * 3)
        for b in range(3):
            assert np.array_equal(t["tokens"][b], s[b])
            assert not t["owner"][b].any() and t["mask"][b].all()
    # and the junior alone when started junior with p = 0
    prm = TandemParams(p=0.0, start_owner=JUNIOR, temperature=temperature, top_p=top_p, seed=3)
    t = tandem_generate((sen, jun), prm, prompts, [14] * 3, ws)
    s = solo_generate(jun, prm, prompts, [14] * 3)
    for b in range(3):
        assert np.array_equal(t["tokens"][b], s[b]) and t["owner"][b].all()
        assert np.all(t["sen_logp"][b] == 0)


@pytest.mark.parametrize("p,mode", [(0.1, TOGGLE), (0.5, TOGGLE), (1.0, TOGGLE), (0.5, REDRAW)])
def test_identical_weights_make_tokens_schedule_independent(p, mode):
    """senior and junior start as identical copies. Then who is active cannot matter:
    the token stream equals solo decoding for every p / mode / table; only the flags vary."""
    m = _mk(1)
    m2 = OracleModel(MICRO, m.w)                    # same weights, separate caches
    ws = make_word_start(MICRO.vocab, 0.5, 11)
    prompts = _prompts()
    prm = TandemParams(p=p, switch_mode=mode, temperature=1.0, seed=12)
    t = tandem_generate((m, m2), prm, prompts, [16] * 3, ws)
    s = solo_generate(m, prm, prompts, [16] * 3)
    for b in range(3):
        assert np.array_equal(t["tokens"][b], s[b])
    assert np.concatenate(t["owner"]).any()        # the junior did take turns


def test_cfg1_recipe_runs_and_margin_is_recorded():
    """configs[0] end to end with the oracle: B=4, prompts of 16 ids, 32 greedy tokens, p=0.5,
    explicit uniforms. Incremental and full-recompute modes agree; the minimum top-1/top-2 margin is
    reported so the GPU free-running comparison (R16) knows how much slack it has."""
    wl = get_workload("cfg1_tiny_f32")
    sen = OracleModel(wl.shape, make_weights(wl.shape, wl.seeds["senior"]))
    jun = OracleModel(wl.shape, make_weights(wl.shape, wl.seeds["junior"]))
    ws = make_word_start(wl.shape.vocab, wl.word_start_frac, wl.seeds["table"])
    prompts = make_prompts(wl)
    usw, usa = make_explicit_uniforms(wl.batch, wl.max_new, wl.shape.vocab, wl.seeds["uniforms"])
    prm = TandemParams(p=wl.p, temperature=wl.temperature)
    a = tandem_generate((sen, jun), prm, prompts, [wl.max_new] * wl.batch, ws, uni=Uniforms(u_switch=usw, u_sample=usa),
                        want_logits=True)
    b = tandem_generate((sen, jun), prm, prompts, [wl.max_new] * wl.batch, ws, uni=Uniforms(u_switch=usw, u_sample=usa),
                        mode="full")
    for i in range(wl.batch):
        assert len(a["tokens"][i]) == 32
        assert np.array_equal(a["tokens"][i], b["tokens"][i]) and np.array_equal(a["owner"][i], b["owner"][i])
    own = np.concatenate(a["owner"])
    assert 0.2 < own.mean() < 0.8
    assert a["min_margin"] > 1e-4, a["min_margin"]

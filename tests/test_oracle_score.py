"""Pins for oracle.score.dual_score / overlap_from_logits."""
import numpy as np
import torch

from oracle import SENIOR, TandemParams, OracleModel, tandem_generate, dual_score, overlap_from_logits
from workloads import ModelShape, make_weights, make_word_start

MICRO = ModelShape(2, 16, 4, 2, 8, 24, 40, 1e-6, 1e4, "f32")


def _mk(seed):
    return OracleModel(MICRO, make_weights(MICRO, seed, std=0.3, gain_jitter=0.2))


def test_overlap_hand_examples():
    """alpha on distributions worked by hand (L134: 0 = disjoint, 1 = identical)."""
    p = np.array([0.5, 0.3, 0.2]); q = np.array([0.2, 0.3, 0.5])
    assert abs(overlap_from_logits(np.log(p), np.log(q)) - 0.7) < 1e-12            # 0.2 + 0.3 + 0.2
    assert abs(overlap_from_logits(np.log(p), np.log(p) + 3.0) - 1.0) < 1e-12      # softmax ignores a shift
    a = np.array([0.0, 0.0, -800.0, -800.0]); b = np.array([-800.0, -800.0, 0.0, 0.0])
    assert overlap_from_logits(a, b) < 1e-300                                      # disjoint supports
    # temperature: T -> infinity flattens both to uniform => alpha -> 1
    assert overlap_from_logits(np.log(p), np.log(q), temperature=1e9) > 1 - 1e-8


def test_overlap_is_one_minus_total_variation():
    """The textbook identity sum min(p, q) = 1 - (1/2) sum |p - q| on random logits."""
    rng = np.random.default_rng(0)
    for _ in range(20):
        zs, zj = rng.standard_normal(40) * 2, rng.standard_normal(40) * 2
        p = torch.softmax(torch.tensor(zs, dtype=torch.float64) / 0.7, 0).numpy()
        q = torch.softmax(torch.tensor(zj, dtype=torch.float64) / 0.7, 0).numpy()
        assert abs(overlap_from_logits(zs, zj, 0.7) - (1.0 - 0.5 * np.abs(p - q).sum())) < 1e-12


def test_dual_score_against_library_cross_entropy_and_symmetry():
    sen, jun = _mk(1), _mk(2)
    rng = np.random.default_rng(3)
    toks = rng.integers(0, MICRO.vocab, size=23)
    r = dual_score((sen, jun), toks)
    assert r["sen_logp"][0] == 0 and r["jun_logp"][0] == 0 and r["overlap"][0] == 0
    # the junior's per-token cross-entropy (L126) is the library's cross_entropy of its logits against the next tokens
    zj = torch.tensor(jun.forward_full(list(toks[:-1])), dtype=torch.float64)
    ce = torch.nn.functional.cross_entropy(zj, torch.tensor(toks[1:], dtype=torch.long), reduction="none").numpy()
    assert np.max(np.abs(-r["jun_logp"][1:] - ce)) < 1e-10
    assert np.all(r["overlap"][1:] > 0) and np.all(r["overlap"][1:] <= 1 + 1e-12)
    # swapping the roles swaps the two log-prob streams and leaves alpha unchanged
    s = dual_score((jun, sen), toks)
    assert np.allclose(s["sen_logp"], r["jun_logp"], atol=1e-12) and np.allclose(s["jun_logp"], r["sen_logp"], atol=1e-12)
    assert np.allclose(s["overlap"], r["overlap"], atol=1e-12)
    # the same model twice: alpha = 1 and equal log-probs at every position
    t = dual_score((sen, sen), toks)
    assert np.allclose(t["overlap"][1:], 1.0, atol=1e-12) and np.array_equal(t["sen_logp"], t["jun_logp"])
    # a one-token stream has nothing to score
    assert not dual_score((sen, jun), toks[:1])["overlap"].any()


def test_dual_score_reproduces_the_rollouts_senior_log_probs():
    """On a stream the senior sampled alone (p = 0) at temperature T, the senior log-probs the rollout recorded (incremental KV
    path, L69) equal dual_score's at the generated positions, scored at the same T."""
    sen, jun = _mk(1), _mk(2)
    ws = make_word_start(MICRO.vocab, 0.4, 3)
    prompt = np.array([3, 9, 27, 1])
    prm = TandemParams(p=0.0, start_owner=SENIOR, temperature=0.8, seed=5)
    out = tandem_generate((sen, jun), prm, [prompt], [12], ws)
    stream = np.concatenate([prompt, out["tokens"][0]])
    r = dual_score((sen, jun), stream, temperature=0.8)
    assert np.max(np.abs(r["sen_logp"][len(prompt):] - out["sen_logp"][0])) < 1e-9
    # under the tandem rule the recorded values are dual_score's senior stream masked by authorship (L263 mask)
    prm = TandemParams(p=0.5, start_owner=SENIOR, temperature=0.8, seed=6)
    out = tandem_generate((sen, jun), prm, [prompt], [16], ws)
    stream = np.concatenate([prompt, out["tokens"][0]])
    r = dual_score((sen, jun), stream, temperature=0.8)
    want = np.where(out["mask"][0], r["sen_logp"][len(prompt):], 0.0)
    assert np.max(np.abs(want - out["sen_logp"][0])) < 1e-9 and 0 < out["mask"][0].sum() < 16

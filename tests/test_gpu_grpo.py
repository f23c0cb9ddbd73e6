"""-m gpu: tandem_grpo_objective (senior-masked GRPO forward) against oracle.grpo.
PAPER.md Eq. 1 (L69), Table 3 (L277-292), Alg. 1; reading R19."""
import numpy as np
import pytest
import torch

import paper_2606_28166_b200 as T
from oracle import grpo_objective as oracle_grpo, TandemParams as OParams
from workloads import get_workload, make_word_start
from gpu_util import make_pair, dev

pytestmark = pytest.mark.gpu


def _inputs(n_groups, G, L, seed, ragged=True):
    rng = np.random.default_rng(seed)
    B = n_groups * G
    rewards = rng.integers(0, 2, size=B).astype(np.float32)
    lengths = (rng.integers(1, L + 1, size=B) if ragged else np.full(B, L)).astype(np.int32)
    owner = rng.integers(0, 2, size=(B, L)).astype(np.uint8)
    old = (-rng.random((B, L)) * 3).astype(np.float32)
    new = (old + rng.standard_normal((B, L)).astype(np.float32) * 0.3).astype(np.float32)
    ref = (old + rng.standard_normal((B, L)).astype(np.float32) * 0.2).astype(np.float32)
    return rewards, lengths, owner, new, old, ref


def _check(got, ref, rtol=2e-5):
    assert np.allclose(got["advantages"].cpu().numpy(), ref["advantages"], rtol=rtol, atol=1e-6)
    assert np.allclose(got["seq_obj"].cpu().numpy(), ref["seq_obj"], rtol=rtol, atol=2e-6)
    if got["token_obj"] is not None:
        assert np.allclose(got["token_obj"].cpu().numpy(), ref["token_obj"], rtol=rtol, atol=2e-6)
    assert abs(got["loss"] - ref["loss"]) <= 2e-6 + rtol * abs(ref["loss"])
    assert got["n_senior"] == ref["n_senior"]
    assert abs(got["clip_frac"] - ref["clip_frac"]) <= 2.0 / max(1, ref["n_senior"])      # a ratio within rounding of the clip edge


@pytest.mark.parametrize("n_groups,G,L,kl", [(1, 2, 3, 0.0), (3, 4, 17, 0.04), (16, 8, 700, 0.0), (16, 8, 3000, 0.001), (5, 1, 40, 0.0)])
def test_grpo_objective_matches_oracle(n_groups, G, L, kl):
    rewards, lengths, owner, new, old, ref_lp = _inputs(n_groups, G, L, 100 + L)
    if n_groups >= 3:
        owner[2, :] = 1                                             # a rollout the junior wrote alone
        rewards[G * (n_groups - 1):] = 1.0                          # a group with equal rewards: advantage 0
    want = oracle_grpo(rewards, G, lengths, owner, new, old, ref_lp if kl else None, clip_eps=0.2, kl_beta=kl)
    got = T.grpo_objective(dev(rewards), G, dev(lengths), dev(owner), dev(new), dev(old), dev(ref_lp) if kl else None, clip_eps=0.2, kl_beta=kl)
    _check(got, want)
    if n_groups >= 3:
        assert got["seq_obj"][2].item() == 0.0 and torch.all(got["advantages"][G * (n_groups - 1):] == 0)
    again = T.grpo_objective(dev(rewards), G, dev(lengths), dev(owner), dev(new), dev(old), dev(ref_lp) if kl else None, clip_eps=0.2, kl_beta=kl,
                             want_tokens=False)
    assert again["loss"] == got["loss"] and again["token_obj"] is None          # deterministic, bit for bit


def test_grpo_hand_example_and_errors():
    owner = np.array([[0, 1, 0], [0, 0, 1]], np.uint8)
    old = np.array([[-1.0, -2.0, -1.5], [-0.7, -0.2, -9.0]], np.float32)
    new = (old + np.array([[0.1, 5.0, 0.3], [-0.5, 0.0, 7.0]], np.float32)).astype(np.float32)
    got = T.grpo_objective(dev(np.array([1.0, 0.0], np.float32)), 2, dev(np.array([3, 2], np.int32)), dev(owner), dev(new), dev(old), adv_eps=0.0)
    assert np.allclose(got["token_obj"].cpu().numpy(), [[np.exp(0.1), 0.0, 1.2], [-0.8, -1.0, 0.0]], atol=1e-6)   # worked by hand, tests/test_oracle_grpo.py
    assert abs(got["loss"] + ((np.exp(0.1) + 1.2) / 2 - 0.9) / 2) < 1e-6 and got["n_senior"] == 4 and abs(got["clip_frac"] - 0.5) < 1e-6
    with pytest.raises(T.TandemError):
        T.grpo_objective(dev(np.zeros(2, np.float32)), 2, dev(np.array([3, 2], np.int32)), dev(owner), dev(new), dev(old), kl_beta=0.1)   # no ref


def test_rollout_then_score_then_objective():
    """The chain the paper's Alg. 1 runs per step, on the tiny fp32 pair: tandem rollout (G rollouts per prompt, mask and senior
    log-probs recorded), a changed senior scores the same streams (tandem_score), and the objective consumes both. Checked against
    the oracle's objective fed with the oracle's own rollout log-probs and scores of the same streams."""
    from oracle import dual_score, OracleModel
    from workloads import make_weights
    shape = get_workload("cfg1_tiny_f32").shape
    ws = make_word_start(shape.vocab, 0.3, 11)
    rng = np.random.default_rng(41)
    n_groups, G, L = 2, 4, 24
    prompts = [rng.integers(0, shape.vocab, size=int(n)).astype(np.int32) for n in (7, 12)]
    prompts = [p for p in prompts for _ in range(G)]
    B = len(prompts)
    eng, orc, _ = make_pair(shape, (1, 2), max_seqs=B, max_seq_len=64, gain_jitter=0.1, std=0.08)
    gen = eng.generate(T.TandemParams(ws, p=0.5, temperature=1.0, eos_id=3, seed=5), prompts, [L] * B)
    streams = [np.concatenate([prompts[b], gen["tokens"][b, :gen["len"][b]]]) for b in range(B)]
    w_new = make_weights(shape, 7, gain_jitter=0.1, std=0.08)                   # the senior after an update (stand-in: other weights)
    eng.load_weights(0, w_new)
    sc = eng.score(streams, temperature=1.0)
    new = np.zeros((B, L), np.float32)
    for b in range(B):
        n = gen["len"][b]
        new[b, :n] = sc["sen_logp"][b][len(prompts[b]):]
    rewards = (gen["tokens"][:, 0] % 2).astype(np.float32)                       # a stand-in verifier
    got = T.grpo_objective(dev(rewards), G, dev(gen["len"].astype(np.int32)), dev(gen["owner"]), dev(new), dev(gen["sen_logp"]))
    o_new = OracleModel(shape, w_new)
    new_ref = np.zeros((B, L))
    for b in range(B):
        n = gen["len"][b]
        new_ref[b, :n] = dual_score((o_new, orc[1]), streams[b])["sen_logp"][len(prompts[b]):]
    want = oracle_grpo(rewards, G, gen["len"], gen["owner"], new_ref, gen["sen_logp"].astype(np.float64))
    assert abs(got["loss"] - want["loss"]) < 5e-4 * max(1.0, abs(want["loss"])) and got["n_senior"] == want["n_senior"] == int(gen["mask"].sum())
    assert np.allclose(got["seq_obj"].cpu().numpy(), want["seq_obj"], rtol=2e-3, atol=2e-4)
    eng.free()

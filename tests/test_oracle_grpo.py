"""Pins for oracle.grpo (Eq. 1, Table 3, Alg. 1; reading R19)."""
import numpy as np
import torch

from oracle import group_advantages, grpo_objective


def test_advantages_closed_form_for_binary_rewards():
    """The paper's reward is binary (L67). With k successes out of G: mean = k/G =: q, population std = sqrt(q(1-q)), so a success
    gets sqrt((1-q)/q) and a failure -sqrt(q/(1-q)); a group with equal rewards gets 0."""
    G = 8
    for k in range(0, G + 1):
        r = np.array([1.0] * k + [0.0] * (G - k))
        A = group_advantages(r, G, adv_eps=0.0) if 0 < k < G else group_advantages(r, G)
        if k in (0, G):
            assert np.all(A == 0)
            continue
        q = k / G
        assert np.allclose(A[:k], np.sqrt((1 - q) / q), atol=1e-12) and np.allclose(A[k:], -np.sqrt(q / (1 - q)), atol=1e-12)
        assert abs(A.mean()) < 1e-12 and abs((A ** 2).mean() - 1) < 1e-12
    # groups are independent and contiguous
    r = np.array([1, 0, 0, 0, 1, 1, 1, 0], dtype=float)
    A = group_advantages(r, 4, adv_eps=0.0)
    assert np.allclose(A[:4], group_advantages(r[:4], 4, adv_eps=0.0)) and np.allclose(A[4:], group_advantages(r[4:], 4, adv_eps=0.0))


def test_objective_hand_example():
    """Two rollouts of one prompt, worked by hand. rewards (1, 0): A = (+1, -1) (adv_eps = 0).
    rollout 0: positions senior, junior, senior; ratios e^{0.1}, -, e^{0.3} -> min(rho, clip) * 1 = e^{0.1} = 1.10517, 1.2
    rollout 1: positions senior, senior (length 2); ratios e^{-0.5} = 0.60653, 1 with A = -1: min(-rho, -clip(rho)) = -0.8, -1."""
    owner = np.array([[0, 1, 0], [0, 0, 1]])
    old = np.array([[-1.0, -2.0, -1.5], [-0.7, -0.2, -9.0]])
    new = old + np.array([[0.1, 5.0, 0.3], [-0.5, 0.0, 7.0]])
    r = grpo_objective([1.0, 0.0], 2, [3, 2], owner, new, old, adv_eps=0.0)
    assert np.allclose(r["advantages"], [1.0, -1.0])
    assert np.allclose(r["token_obj"], [[np.exp(0.1), 0.0, 1.2], [-0.8, -1.0, 0.0]], atol=1e-12)
    assert np.allclose(r["seq_obj"], [(np.exp(0.1) + 1.2) / 2, -0.9], atol=1e-12)
    assert abs(r["loss"] + ((np.exp(0.1) + 1.2) / 2 - 0.9) / 2) < 1e-12
    assert r["n_senior"] == 4 and abs(r["clip_frac"] - 0.5) < 1e-12          # e^{0.3} > 1.2 and e^{-0.5} < 0.8 are clipped
    # junior-emitted positions and positions past the length carry no weight (Eq. 1: the sum runs over a_t = sen)
    new2 = new.copy(); new2[0, 1] = -30.0; new2[1, 2] = 3.0
    assert grpo_objective([1.0, 0.0], 2, [3, 2], owner, new2, old, adv_eps=0.0)["loss"] == r["loss"]


def test_objective_against_torch_ops():
    """The same formula through library routines (torch.clamp / torch.minimum / masked means) on random inputs, KL term included."""
    rng = np.random.default_rng(1)
    n_groups, G, L = 3, 4, 17
    B = n_groups * G
    rewards = rng.integers(0, 2, size=B).astype(float)
    lengths = rng.integers(1, L + 1, size=B)
    owner = rng.integers(0, 2, size=(B, L))
    old = -rng.random((B, L)) * 3; new = old + rng.standard_normal((B, L)) * 0.3; ref = old + rng.standard_normal((B, L)) * 0.2
    r = grpo_objective(rewards, G, lengths, owner, new, old, ref, clip_eps=0.2, kl_beta=0.04)
    tr = torch.tensor(rewards, dtype=torch.float64).view(n_groups, G)
    A = ((tr - tr.mean(1, keepdim=True)) / (tr.std(1, unbiased=False, keepdim=True) + 1e-6)).view(B, 1)
    tn, to, tf = (torch.tensor(x, dtype=torch.float64) for x in (new, old, ref))
    rho = torch.exp(tn - to)
    s = torch.minimum(rho * A, torch.clamp(rho, 0.8, 1.2) * A) - 0.04 * (torch.exp(tf - tn) - (tf - tn) - 1)
    mask = (torch.tensor(owner) == 0) & (torch.arange(L)[None, :] < torch.tensor(lengths)[:, None])
    n = mask.sum(1)
    seq = torch.where(n > 0, (s * mask).sum(1) / n.clamp(min=1), torch.zeros(B, dtype=torch.float64))
    assert np.allclose(r["seq_obj"], seq.numpy(), atol=1e-12) and abs(r["loss"] + seq.mean().item()) < 1e-12
    assert np.allclose(r["advantages"], A.view(-1).numpy(), atol=1e-12)


def test_on_policy_special_cases():
    """logp_new == logp_old (the first update after a rollout): every ratio is 1, nothing is clipped, J_i = A_i wherever rollout i has
    a senior token, so with senior tokens everywhere the loss is -mean(A) = 0 group by group; a rollout written by the junior alone
    contributes 0 (lambda_jun = 0, Table 3)."""
    rng = np.random.default_rng(2)
    G, L = 8, 9
    rewards = np.array([1, 0, 0, 1, 1, 0, 0, 0], dtype=float)
    old = -rng.random((G, L))
    owner = rng.integers(0, 2, size=(G, L)); owner[:, 0] = 0
    r = grpo_objective(rewards, G, [L] * G, owner, old, old)
    assert r["clip_frac"] == 0 and np.allclose(r["seq_obj"], r["advantages"], atol=1e-12) and abs(r["loss"]) < 1e-12
    owner[3, :] = 1
    r2 = grpo_objective(rewards, G, [L] * G, owner, old, old)
    assert r2["seq_obj"][3] == 0 and abs(r2["loss"] - r["advantages"][3] / G) < 1e-12


def test_clip_frac_counts_only_positions_where_the_clipped_branch_is_taken():
    """R19: for A > 0 and rho < 1 - eps (or A < 0 and rho > 1 + eps) the min selects the UNCLIPPED branch: the ratio left the
    interval but the gradient is not cut, so the position does not count. Hand case, one group of two rollouts (A = +1, -1),
    one senior position each: rho = e^{-0.5} = 0.607 with A = +1 -> min(0.607, 0.8) = 0.607 (unclipped); rho = e^{0.5} = 1.649
    with A = -1 -> min(-1.649, -1.2) = -1.649 (unclipped)."""
    rewards = np.array([1.0, 0.0])
    owner = np.zeros((2, 1), np.uint8)
    old = np.zeros((2, 1))
    new = np.array([[-0.5], [0.5]])
    r = grpo_objective(rewards, 2, np.array([1, 1]), owner, new, old)
    assert r["clip_frac"] == 0.0
    assert np.allclose(r["token_obj"][:, 0], [np.exp(-0.5) * r["advantages"][0], np.exp(0.5) * r["advantages"][1]], atol=1e-12)
    # mirrored ratios: both clipped branches are taken
    r2 = grpo_objective(rewards, 2, np.array([1, 1]), owner, -new, old)
    assert r2["clip_frac"] == 1.0
    assert np.allclose(r2["token_obj"][:, 0], [1.2 * r2["advantages"][0], 0.8 * r2["advantages"][1]], atol=1e-12)

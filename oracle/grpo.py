"""Senior-masked GRPO objective, forward only (TEST INFRASTRUCTURE) - SURVEY.md section 8(f) NEXT-3.

PAPER.md L69-71 (section 3.4, Eq. 1): "The senior is updated with the standard GRPO objective (Shao et al., 2024), with the
response mask set to select only senior-emitted positions; the per-token policy-gradient contribution is
L = -E[ sum_{t: a_t = sen} A_t log pi_sen(y_t | x.y_<t) ], where A_t is the standard GRPO group-relative advantage; the clipped
surrogate ratio and KL term are also identical to GRPO". Table 3 (L277-292): clip ratio 0.2, G = 8, "Advantage estimator: GRPO
(group-relative, std-normalised)", junior-token loss weight 0. Alg. 1 lines 19-21 (L370-376): rewards -> group-relative
advantages -> update "with response mask narrowed by m".

Reading R19 where the paper leaves the standard objective to its citation:
  advantage     A_i = (r_i - mean_g) / (std_g + adv_eps) over the G rollouts of the prompt, std_g = sqrt(mean (r - mean_g)^2)
                (population form), adv_eps = 1e-6; every token of rollout i carries A_i;
  ratio         rho_t = exp(logp_new_t - logp_old_t)  (logp_old: recorded by the rollout; logp_new: the policy being updated);
  surrogate     s_t = min(rho_t A_i, clip(rho_t, 1 - eps, 1 + eps) A_i), eps = 0.2;
  KL (optional) k_t = exp(logp_ref_t - logp_new_t) - (logp_ref_t - logp_new_t) - 1 (the estimator of Shao et al.), weight beta;
  aggregation   J_i = (1 / n_i) sum_{t < len_i, a_t = sen} (s_t - beta k_t), n_i = number of senior positions of rollout i
                (J_i = 0 when n_i = 0); loss = -(1 / B) sum_i J_i  (Shao et al.'s 1/G sum_i 1/|o_i| sum_t with |o_i| narrowed
                to the senior positions);
  clip_frac     a diagnostic the paper does not define: the share of senior positions where the clipped branch is the one the
                min selects (clip(rho) A < rho A), i.e. where the policy gradient is cut - not every position whose ratio left
                [1 - eps, 1 + eps] (for A > 0 and rho < 1 - eps the unclipped branch is taken).
Not covered by the paper's text: trainer stacks differ in the std convention (this reading: population std; some use the unbiased
G - 1 form, which makes every advantage sqrt((G-1)/G) times smaller) - the caller can rescale `advantages`.
"""
import numpy as np


def group_advantages(rewards, group, adv_eps=1e-6):
    """rewards [n_groups * group] (rollouts of a prompt are contiguous) -> advantages of the same shape."""
    r = np.asarray(rewards, dtype=np.float64).reshape(-1, group)
    mean = r.mean(axis=1, keepdims=True)
    std = np.sqrt(((r - mean) ** 2).mean(axis=1, keepdims=True))
    return ((r - mean) / (std + adv_eps)).reshape(-1)


def grpo_objective(rewards, group, lengths, owner, logp_new, logp_old, logp_ref=None, clip_eps=0.2, kl_beta=0.0, adv_eps=1e-6):
    """owner [B, L] (0 = senior-emitted), logp_* [B, L], lengths [B]. Returns dict(advantages [B], token_obj [B, L] (s_t - beta k_t at
    senior positions, 0 elsewhere), seq_obj [B], loss, clip_frac (share of senior positions where the clipped branch of the min is the one taken), n_senior)."""
    owner = np.asarray(owner)
    B, L = owner.shape
    A = group_advantages(rewards, group, adv_eps)
    ln = np.asarray(logp_new, dtype=np.float64)
    lo = np.asarray(logp_old, dtype=np.float64)
    tok = np.zeros((B, L), dtype=np.float64)
    seq = np.zeros(B, dtype=np.float64)
    clipped = 0
    n_sen = 0
    for i in range(B):
        acc, n = 0.0, 0
        for t in range(int(lengths[i])):
            if owner[i, t] != 0:
                continue
            rho = np.exp(ln[i, t] - lo[i, t])
            rc = min(max(rho, 1.0 - clip_eps), 1.0 + clip_eps)
            s = min(rho * A[i], rc * A[i])
            if rc * A[i] < rho * A[i]:          # the clipped branch is the one min() takes (R19): the gradient of this position is cut
                clipped += 1
            if kl_beta != 0.0 and logp_ref is not None:
                d = float(logp_ref[i][t]) - ln[i, t]
                s -= kl_beta * (np.exp(d) - d - 1.0)
            tok[i, t] = s
            acc += s
            n += 1
        seq[i] = acc / n if n else 0.0
        n_sen += n
    return dict(advantages=A, token_obj=tok, seq_obj=seq, loss=float(-seq.mean()) if B else 0.0,
                clip_frac=clipped / n_sen if n_sen else 0.0, n_senior=n_sen)

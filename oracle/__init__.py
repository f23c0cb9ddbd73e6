"""CPU oracle for the tandem rollout hot path (TEST INFRASTRUCTURE, not the product).

This package is a plain, slow, float64 NumPy restatement of what the hot path of
Tandem RLVR (arxiv/paper_2606_28166) computes: two decoder-only transformers of
the same architecture co-generating a response, alternating at word-start tokens
(§3.3; L345-367 Alg. 1), with the per-token authorship mask (L263
§B.1.1) and the senior's log-probabilities at senior-emitted positions (Eq. 1).

Rules of the house:
  * only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
    `--impl reference` legs may import this package; the product
    (`paper_2606_28166_b200/`) never does, and this package never imports the product;
  * no code, table, constant generator or helper is shared with the CUDA path;
    the only thing both sides use is the seeded input generator `workloads/`,
    which holds none of the method's arithmetic;
  * arithmetic is float64 throughout (the paper fixes no precision; BASELINE.json's
    "fp32 oracle" is satisfied a fortiori). Weights are used at the values given
    (bf16 values are widened exactly);
  * every function cites the passage it follows; the readings taken where the paper
    is silent are listed in DESIGN.md section 3 and referenced as R1..R16.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): Philox known-answer vectors, closed
forms for RoPE/RMSNorm/softmax/SwiGLU, library-routine cross-check of the forward
(torch float64 sdpa/rms_norm/silu), incremental-KV == full recompute, p=0 == solo,
p=1 closed form, brute-force coin enumeration against a table-driven transcription
of section 3.3, role-swap symmetry, same-weights schedule independence, Gumbel-max
frequencies vs softmax (chi-square), top-p hand example, senior share / run-length laws; top-k hand
examples, top-k 1 = greedy, frequencies under the renormalised distribution (sampler.kept_set, R18); overlap alpha on
hand-worked distributions and as 1 - total variation, junior cross-entropy against torch's cross_entropy, role swap,
agreement with the rollout's recorded senior log-probs (score.dual_score, R17); binary-reward advantages in closed
form, a hand-worked clipped surrogate, a torch re-composition, on-policy special cases (grpo.grpo_objective, R19).
Parity that stays unpinned: any comparison with the paper's own rollouts, rewards or
accuracy numbers (its weights, tokenizer and datasets are not available).
"""
from .rng import philox4x32_10, uniform_from_bits, uniforms_sample, uniforms_switch, gumbel_from_uniform
from .model import OracleModel, KVState
from .sampler import sample_token, log_prob, kept_set_top_p, kept_set
from .rule import (SENIOR, JUNIOR, DRAW, TOGGLE, REDRAW, TandemParams,
                   owners_from_tokens, tandem_generate, solo_generate)
from .score import teacher_forced_logits, replay_owner_logits, overlap_from_logits, dual_score
from .grpo import group_advantages, grpo_objective

__all__ = [
    "philox4x32_10", "uniform_from_bits", "uniforms_sample", "uniforms_switch", "gumbel_from_uniform",
    "OracleModel", "KVState", "sample_token", "log_prob", "kept_set_top_p", "kept_set",
    "SENIOR", "JUNIOR", "DRAW", "TOGGLE", "REDRAW", "TandemParams",
    "owners_from_tokens", "tandem_generate", "solo_generate",
    "teacher_forced_logits", "replay_owner_logits", "overlap_from_logits", "dual_score", "group_advantages", "grpo_objective",
]

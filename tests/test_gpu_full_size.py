"""-m gpu: BASELINE.json configs[2] at its FULL batch, in the launch configuration bench.py times (cfg3_4b_bf16: 128
sequences = 16 prompts x 8 rollouts, prompts of 64..512 ids, both 36-layer 4B-shape models, CUDA-graph replay of the paired
launches, the whole-rollout call on host buffers). The oracle cannot run 128 such sequences, so:

  * on ALL sequences, what is an integer function of the token stream is re-derived by the oracle's rule and compared
    bit for bit: owner flags, switch positions, the senior mask, lengths (BASELINE.json north_star; R16);
  * on SAMPLED sequences (the ones with the shortest prompts, one per GRPO group), the float64 oracle replays the GPU's
    token stream teacher-forced and the senior log-probs / the Gumbel-sampled tokens are compared one by one, with the bars
    of tests/test_gpu_bf16_slice.py at this shape (R-V);
  * properties that hold at any size: the rollouts of a group share a prompt but not their continuation; a sampled
    sequence run alone (batch of 1, same seq_id, forced onto the same stream) has the same owners and log-probs as inside the
    batch of 128 (R9: position-addressed uniforms)."""
import numpy as np
import pytest
import torch

import paper_2606_28166_b200 as T
from oracle import OracleModel, TandemParams as OParams, owners_from_tokens, replay_owner_logits, sample_token
from oracle import rng as orng
from oracle.rule import Uniforms
from oracle.sampler import log_softmax
from workloads import get_workload, make_prompts, make_weights, make_word_start

pytestmark = pytest.mark.gpu

N_NEW = 12
SEED = 2025


def test_cfg3_full_batch_sampled_sequences_and_integer_outputs():
    wl = get_workload("cfg3_4b_bf16")
    shape = wl.shape
    free, _ = torch.cuda.mem_get_info()
    if free < 60 << 30:
        pytest.skip("needs ~45 GB of device memory for the two 4B-shape models and their page pools")
    ws_ = make_weights(shape, wl.seeds["senior"], device="cuda")
    wj_ = make_weights(shape, wl.seeds["junior"], device="cuda")
    table = make_word_start(shape.vocab, wl.word_start_frac, wl.seeds["table"])
    prompts = make_prompts(wl)
    B = len(prompts)
    assert B == 128 and wl.group == 8
    max_len = max(len(p) for p in prompts) + N_NEW + 1
    prm = T.TandemParams(table, p=wl.p, temperature=1.0, seed=SEED)

    # what bench.py runs: step graph, paired launches, the rollouts of a prompt sharing its KV pages and reading them once per run (share_prompt_pages = 2)
    eng = T.Tandem(T.TandemConfig(shape, max_seqs=B, max_seq_len=max_len, use_graph=1, share_prompt_pages=2))
    eng.load_weights(0, ws_)
    eng.load_weights(1, wj_)
    out = eng.generate(prm, prompts, [N_NEW] * B)
    eng.free()
    toks, own, lp, n = out["tokens"], out["owner"], out["sen_logp"], out["len"]
    assert out["stats"]["shared_prompt_rows"] > 0 and out["stats"]["kv_bytes_shared_reads"] > 0

    # ---- all 128 sequences: integer outputs bit-exact against the oracle's rule on the GPU's own token stream
    assert (n == N_NEW).all()
    assert ((toks >= 0) & (toks < shape.vocab)).all()
    for b in range(B):
        ref_own = owners_from_tokens(toks[b], table, OParams(p=wl.p, seed=SEED), Uniforms(seed=SEED), b=b)
        assert np.array_equal(ref_own, own[b]), f"owner flags of sequence {b} differ from the rule"
        assert np.array_equal(out["mask"][b], (ref_own == 0).astype(np.uint8))
        assert (lp[b][own[b] == 1] == 0.0).all() and (lp[b][own[b] == 0] < 0.0).all()
        flips = own[b, 1:] != own[b, :-1]
        assert not flips[table[toks[b, :-1]] == 0].any(), "an owner change follows a token that starts no word"
    assert 0.2 < own.mean() < 0.8
    # rollouts of a group share the prompt, not the continuation (uniforms are addressed by sequence id)
    for g in range(0, B, wl.group):
        assert len({tuple(toks[b]) for b in range(g, g + wl.group)}) == wl.group

    # ---- sampled sequences: the shortest prompts of two different groups, replayed by the float64 oracle
    lens = np.array([len(p) for p in prompts])
    order = np.argsort(lens[::wl.group], kind="stable")[:2] * wl.group
    sampled = [int(order[0]) + 3, int(order[1]) + 6]   # not the first rollout of the group
    cpu = lambda w: dict(embed=w["embed"].cpu(), lm_head=w["lm_head"].cpu(), final_norm=w["final_norm"].cpu(),
                         layers=[{k: v.cpu() for k, v in l.items()} for l in w["layers"]])
    models = (OracleModel(shape, cpu(ws_), cache=False), OracleModel(shape, cpu(wj_), cache=False))
    dl, samp = [], []
    for b in sampled:
        z = replay_owner_logits(models, prompts[b], toks[b], own[b])
        for t in range(N_NEW):
            if own[b, t] == 0:
                dl.append(abs(lp[b, t] - log_softmax(z[t])[toks[b, t]]))
            samp.append(sample_token(z[t], 1.0, 1.0, orng.uniforms_sample(SEED, b, t + 1, shape.vocab)) == toks[b, t])
    assert len(dl) >= 4
    print("full batch: sampled", sampled, "prompt lens", lens[sampled], "max dlogp %.4f mean %.4f sampled agreement %.3f" % (max(dl), np.mean(dl), np.mean(samp)))
    assert max(dl) <= 0.08 and np.mean(dl) <= 0.02     # the 4B-shape bars of test_bf16_slice_4b_shape (DESIGN.md R-V)
    assert np.mean(samp) >= 0.9

    # ---- batch independence at full size: a sampled sequence alone (batch of 1, no chunked prefill), forced onto the same token
    # stream, has the same owners and - up to the bf16 rounding flips a different prefill chunking can cause - the same log-probs
    del models
    solo = T.Tandem(T.TandemConfig(shape, max_seqs=1, max_seq_len=max_len))
    solo.load_weights(0, ws_)
    solo.load_weights(1, wj_)
    for b in sampled:
        forced = torch.as_tensor(toks[b:b + 1].astype(np.int32)).cuda()
        o1 = solo.generate(prm, [prompts[b]], [N_NEW], seq_ids=[b], forced_tokens=forced)
        assert np.array_equal(o1["tokens"][0], toks[b]) and np.array_equal(o1["owner"][0], own[b])
        assert np.max(np.abs(o1["sen_logp"][0] - lp[b])) < 0.03
    solo.free()

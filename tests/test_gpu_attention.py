"""-m gpu: the tensor-core paged attention kernel (attention_mma.cuh) against the plain-ALU kernel (attention.cuh) and the
oracle, through the C ABI, over the (head_dim, group) instantiations and the ragged shapes of the path: decode with KV
splits, catch-ups that cross pages and q-tiles, multi-q-tile prompt prefill, chunked prefill (row budget), contexts of
several hundred positions on scattered pages. The ALU engine generates; the MMA engine replays the same token stream
(forced tokens) and must give the same senior log-probs (bf16 rounding of Q and P apart) and the same owner flags."""
import numpy as np
import pytest
import torch

import paper_2606_28166_b200 as T
from oracle import OracleModel, replay_owner_logits
from oracle.sampler import log_softmax
from workloads import ModelShape, make_weights, make_word_start
from gpu_util import dev

pytestmark = pytest.mark.gpu


def _engines(shape, B, L, **kw):
    ws = make_weights(shape, 1, device="cuda"); wj = make_weights(shape, 2, device="cuda")
    engs = []
    for impl in (T.ATTN_ALU, T.ATTN_MMA):
        e = T.Tandem(T.TandemConfig(shape, max_seqs=B, max_seq_len=L, attn_impl=impl, **kw))
        e.load_weights(0, ws); e.load_weights(1, wj)
        engs.append(e)
    return engs, (ws, wj)


@pytest.mark.parametrize("nq,nkv,d", [(4, 4, 64), (4, 2, 64), (8, 2, 64), (14, 2, 64), (8, 1, 64), (2, 2, 128), (4, 2, 128), (8, 2, 128), (8, 1, 128)])
def test_mma_matches_alu_teacher_forced(nq, nkv, d):
    shape = ModelShape(2, 256, nq, nkv, d, 512, 1024, 1e-6, 1e6, "bf16")
    rng = np.random.default_rng(nq * 100 + nkv * 10 + d)
    lens = [1, 15, 16, 17, 63, 64, 65, 130, 300, 41]
    B, n_new = len(lens), 48
    prompts = [rng.integers(0, shape.vocab, size=n).astype(np.int32) for n in lens]
    table = make_word_start(shape.vocab, 0.3, 3)
    (alu, mma), _ = _engines(shape, B, 384, max_rows_per_step=96)       # 96-row budget: the 130- and 300-token prefills are chunked
    prm = T.TandemParams(table, p=0.5, temperature=1.0, seed=7)
    a = alu.generate(prm, prompts, [n_new] * B)
    forced = np.where(np.arange(n_new)[None, :] < a["len"][:, None], a["tokens"], -1).astype(np.int32)
    m = mma.generate(prm, prompts, [n_new] * B, forced_tokens=dev(forced))
    assert np.array_equal(m["tokens"], a["tokens"]) and np.array_equal(m["owner"], a["owner"]) and np.array_equal(m["len"], a["len"])
    assert a["stats"]["catchup_rows"] > 0 and 0.1 < a["owner"].mean() < 0.9
    err = np.abs(m["sen_logp"] - a["sen_logp"])
    assert err.max() <= 0.02 and err.mean() <= 0.002, (err.max(), err.mean())
    alu.free(); mma.free()


def test_mma_long_context_against_oracle():
    """One long sequence (prompt 700, splits and q-tiles active) + short ones: MMA engine vs the float64 oracle on the senior
    log-probs of the generated positions."""
    shape = ModelShape(2, 256, 8, 2, 128, 512, 2048, 1e-6, 1e6, "bf16")
    rng = np.random.default_rng(5)
    lens = [700, 20, 333]
    prompts = [rng.integers(0, shape.vocab, size=n).astype(np.int32) for n in lens]
    table = make_word_start(shape.vocab, 0.3, 3)
    ws = make_weights(shape, 1); wj = make_weights(shape, 2)
    eng = T.Tandem(T.TandemConfig(shape, max_seqs=3, max_seq_len=768, attn_impl=T.ATTN_MMA))
    eng.load_weights(0, ws); eng.load_weights(1, wj)
    n_new = 40
    g = eng.generate(T.TandemParams(table, p=0.5, temperature=1.0, seed=11), prompts, [n_new] * 3)
    models = (OracleModel(shape, ws), OracleModel(shape, wj))
    worst = 0.0
    for b in range(3):
        z = replay_owner_logits(models, prompts[b], g["tokens"][b], g["owner"][b])
        for t in range(n_new):
            if g["owner"][b, t] == 0:
                worst = max(worst, abs(g["sen_logp"][b, t] - log_softmax(z[t])[g["tokens"][b, t]]))
    assert worst <= 0.02, worst
    eng.free()

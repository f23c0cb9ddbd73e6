"""-m gpu: S8 fused into the LM head's epilogue (gemm_tcgen05.cuh, kTcEpiSample + sample_merge_emit_kernel)
against the materialised-logits sampler (sample_switch_emit_kernel) on the same engine state, and against the oracle.

Both paths draw the same position-addressed uniforms and take the argmax of z / T + g in fp32, so tokens, owner flags and lengths must
be identical; the log-probs differ only by the order in which the log-sum-exp is accumulated (<= 2e-5). Covered: Gumbel sampling and
greedy, a vocabulary that is not a multiple of the 128-id tile (4,100) and the full 151,936, more slots than emitting rows, EOS, ragged
lengths, more than 16 and more than 32 rows per model (both 16-column groups of both epilogue warps)."""
import numpy as np
import pytest

import paper_2606_28166_b200 as T
from oracle import OracleModel, TandemParams as OParams, replay_owner_logits, sample_token
from oracle import rng as orng
from oracle.sampler import log_softmax
from workloads import ModelShape, make_weights, make_word_start

pytestmark = pytest.mark.gpu


def _run(shape, B, n_new, temperature, eos, fused, ws, wj, prompts, max_new, table, seed=9, p=0.5):
    eng = T.Tandem(T.TandemConfig(shape, max_seqs=B + 3, max_seq_len=160, use_graph=1))
    eng.load_weights(0, ws); eng.load_weights(1, wj)
    eng.set_option("fused_sampler", fused)
    out = eng.generate(T.TandemParams(table, p=p, temperature=temperature, eos_id=eos, seed=seed), prompts, max_new)
    eng.free()
    return out


@pytest.mark.parametrize("V,B,temperature,eos", [(4100, 5, 1.0, -1), (4100, 40, 0.7, 17), (4100, 70, 0.0, -1), (151936, 6, 1.0, -1), (64, 9, 1.3, 5)])
def test_fused_sampler_equals_materialised_logits(V, B, temperature, eos):
    shape = ModelShape(2, 256, 4, 2, 64, 512, V, 1e-6, 1e6, "bf16")
    ws = make_weights(shape, 1, device="cuda", gain_jitter=0.1); wj = make_weights(shape, 2, device="cuda", gain_jitter=0.1)
    table = make_word_start(V, 0.3, 3)
    rng = np.random.default_rng(B + V)
    prompts = [rng.integers(0, V, size=int(rng.integers(3, 50))).astype(np.int32) for _ in range(B)]
    max_new = rng.integers(20, 41, size=B).astype(np.int32)
    a = _run(shape, B, 40, temperature, eos, 1, ws, wj, prompts, max_new, table)
    b = _run(shape, B, 40, temperature, eos, 0, ws, wj, prompts, max_new, table)
    assert np.array_equal(a["len"], b["len"]) and np.array_equal(a["tokens"], b["tokens"]) and np.array_equal(a["owner"], b["owner"])
    assert 0.1 < a["owner"][:, :20].mean() < 0.9
    assert np.max(np.abs(a["sen_logp"] - b["sen_logp"])) <= 2e-5


def test_fused_sampler_more_than_256_emitting_rows_of_one_model():
    """The persistent LM head (lmhead_sample.cuh) with one model active and 300 emitting rows: two row chunks per weight tile, the two
    TMEM accumulators alternate within a tile, the (t, seq_id) table is reloaded per chunk; and, with p = 0.5, both models at ~150 rows
    (one CTA per model parity, 144-column accumulators)."""
    V, B = 4100, 300
    shape = ModelShape(1, 128, 2, 1, 64, 256, V, 1e-6, 1e6, "bf16")
    ws = make_weights(shape, 1, device="cuda", gain_jitter=0.1); wj = make_weights(shape, 2, device="cuda", gain_jitter=0.1)
    table = make_word_start(V, 0.3, 3)
    rng = np.random.default_rng(31)
    prompts = [rng.integers(0, V, size=int(rng.integers(2, 9))).astype(np.int32) for _ in range(B)]
    max_new = np.full(B, 6, np.int32)
    for p in (0.0, 0.5):
        a = _run(shape, B, 6, 1.0, -1, 1, ws, wj, prompts, max_new, table, p=p)
        b = _run(shape, B, 6, 1.0, -1, 0, ws, wj, prompts, max_new, table, p=p)
        assert np.array_equal(a["len"], b["len"]) and np.array_equal(a["tokens"], b["tokens"]) and np.array_equal(a["owner"], b["owner"])
        assert (a["owner"].sum() == 0) == (p == 0.0)
        assert np.max(np.abs(a["sen_logp"] - b["sen_logp"])) <= 2e-5


def test_fused_sampler_against_the_oracle():
    """The fused path's tokens are the oracle's Gumbel-max on the oracle's own logits wherever the two logit vectors agree on the
    winner (bf16 noise can flip a near-tie), and its senior log-probs are within the bf16 tolerance."""
    V = 4100
    shape = ModelShape(2, 256, 4, 2, 64, 512, V, 1e-6, 1e6, "bf16")
    ws = make_weights(shape, 1, gain_jitter=0.1); wj = make_weights(shape, 2, gain_jitter=0.1)
    table = make_word_start(V, 0.3, 3)
    rng = np.random.default_rng(2)
    prompts = [rng.integers(0, V, size=n).astype(np.int32) for n in (11, 30, 5)]
    g = _run(shape, 3, 32, 1.0, -1, 1, ws, wj, prompts, [32] * 3, table, seed=21)
    models = (OracleModel(shape, ws), OracleModel(shape, wj))
    agree, d = [], []
    for b in range(3):
        z = replay_owner_logits(models, prompts[b], g["tokens"][b], g["owner"][b])
        for t in range(32):
            agree.append(sample_token(z[t], 1.0, 1.0, orng.uniforms_sample(21, b, t + 1, V)) == g["tokens"][b, t])
            if g["owner"][b, t] == 0:
                d.append(abs(g["sen_logp"][b, t] - log_softmax(z[t])[g["tokens"][b, t]]))
    assert np.mean(agree) >= 0.97 and max(d) <= 0.02, (np.mean(agree), max(d))

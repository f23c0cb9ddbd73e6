"""-m gpu: tandem_score (teacher-forced dual scoring) against oracle.score.dual_score.
PAPER.md L126 (junior per-token cross-entropy), L134 (overlap alpha), reading R17."""
import numpy as np
import pytest

import paper_2606_28166_b200 as T
from oracle import OracleModel, dual_score
from workloads import ModelShape, make_weights, make_word_start, get_workload
from gpu_util import make_pair

pytestmark = pytest.mark.gpu

MIDI = ModelShape(4, 256, 4, 2, 64, 512, 4096, 1e-6, 1e6, "bf16")


def _streams(vocab, lengths, seed):
    rng = np.random.default_rng(seed)
    return [rng.integers(0, vocab, size=int(n)).astype(np.int32) for n in lengths]


def _check(out, refs, tol_lp, tol_alpha):
    worst = [0.0, 0.0, 0.0]
    for b, ref in enumerate(refs):
        for k, (name, tol) in enumerate((("sen_logp", tol_lp), ("jun_logp", tol_lp), ("overlap", tol_alpha))):
            assert out[name][b].shape == ref[name].shape
            assert out[name][b][0] == 0.0
            d = float(np.max(np.abs(out[name][b] - ref[name]))) if len(ref[name]) else 0.0
            worst[k] = max(worst[k], d)
            assert d <= tol, (b, name, d)
    return worst


@pytest.mark.parametrize("temperature", [1.0, 0.7])
def test_score_fp32_matches_oracle(temperature):
    """cfg-1 shape in fp32: ragged stream lengths around the page and tile sizes, more streams than slots (queued), a row cap
    that cuts every stream into several steps. Log-probs within 1e-4, alpha within 1e-4 of the float64 oracle."""
    shape = get_workload("cfg1_tiny_f32").shape
    streams = _streams(shape.vocab, (1, 2, 15, 16, 17, 33, 64, 40, 5), 21)
    eng, orc, _ = make_pair(shape, (1, 2), max_seqs=4, max_seq_len=64, gain_jitter=0.2, std=0.08, max_rows_per_step=24)
    out = eng.score(streams, temperature=temperature)
    refs = [dual_score(orc, s, temperature=temperature) for s in streams]
    _check(out, refs, 1e-4, 1e-4)
    alpha = np.concatenate([r["overlap"][1:] for r in refs])
    assert alpha.min() < 0.9 and alpha.max() <= 1.0          # the two models really differ on these inputs
    assert out["stats"]["rows_senior"] == out["stats"]["rows_junior"] == sum(len(s) - 1 for s in streams)
    eng.free()


def test_score_same_weights_gives_alpha_one():
    shape = get_workload("cfg1_tiny_f32").shape
    streams = _streams(shape.vocab, (20, 31), 22)
    eng, orc, _ = make_pair(shape, (1, 1), max_seqs=2, max_seq_len=32, same=True, std=0.08)
    out = eng.score(streams)
    for b in range(2):
        assert np.array_equal(out["sen_logp"][b], out["jun_logp"][b])
        assert np.max(np.abs(out["overlap"][b][1:] - 1.0)) < 1e-5
    eng.free()


def test_score_agrees_with_the_rollouts_recorded_log_probs():
    """The senior log-probs a rollout records at senior-written positions (decode path, one row per step) equal tandem_score's
    on the finished stream (prefill path, many rows per step), scored at the sampling temperature."""
    shape = get_workload("cfg1_tiny_f32").shape
    ws = make_word_start(shape.vocab, 0.3, 11)
    prompts = _streams(shape.vocab, (9, 20, 3), 23)
    eng, orc, _ = make_pair(shape, (1, 2), max_seqs=3, max_seq_len=64, gain_jitter=0.1, std=0.08)
    gen = eng.generate(T.TandemParams(ws, p=0.5, temperature=0.8, seed=9), prompts, [30, 24, 40])
    streams = [np.concatenate([prompts[b], gen["tokens"][b, :gen["len"][b]]]) for b in range(3)]
    out = eng.score(streams, temperature=0.8)
    n_sen = 0
    for b in range(3):
        n, P = gen["len"][b], len(prompts[b])
        m = gen["mask"][b, :n].astype(bool)
        n_sen += int(m.sum())
        assert np.max(np.abs(out["sen_logp"][b][P:][m] - gen["sen_logp"][b, :n][m])) < 2e-5
    assert n_sen > 10
    eng.free()


@pytest.mark.parametrize("gemm_impl", [T.GEMM_SIMT, T.GEMM_TCGEN05])
def test_score_bf16_midi(gemm_impl):
    """bf16 (tensor-core attention; SIMT or tcgen05 projections): against the float64 oracle on the same bf16-valued weights.
    Bars: log-probs 0.05 nats (BASELINE.json's bf16 tolerance), alpha 0.01; the weights are 2.5x wider than the rollout slices'
    (std 0.05) so that the two models disagree visibly (alpha ~ 0.57)."""
    ws_ = make_weights(MIDI, 1, std=0.05)
    wj_ = make_weights(MIDI, 2, std=0.05)
    streams = _streams(MIDI.vocab, (70, 33, 128, 1, 90), 24)
    eng = T.Tandem(T.TandemConfig(MIDI, max_seqs=3, max_seq_len=128, gemm_impl=gemm_impl, max_rows_per_step=96))
    eng.load_weights(0, ws_); eng.load_weights(1, wj_)
    out = eng.score(streams)
    orc = (OracleModel(MIDI, ws_), OracleModel(MIDI, wj_))
    refs = [dual_score(orc, s) for s in streams]
    worst = _check(out, refs, 0.05, 0.01)
    alpha = np.concatenate([r["overlap"][1:] for r in refs])
    assert alpha.min() < 0.95
    # the aggregate the paper reports (Table 1): mean junior cross-entropy and mean alpha over all scored positions
    ce_gpu = -np.concatenate([o[1:] for o in out["jun_logp"]]).mean(); ce_ref = -np.concatenate([r["jun_logp"][1:] for r in refs]).mean()
    a_gpu = np.concatenate([o[1:] for o in out["overlap"]]).mean()
    assert abs(ce_gpu - ce_ref) < 2e-3 and abs(a_gpu - alpha.mean()) < 2e-3, (worst, ce_gpu, ce_ref, a_gpu, alpha.mean())
    eng.free()


def test_score_api_errors_and_reuse():
    shape = get_workload("cfg1_tiny_f32").shape
    ws = make_word_start(shape.vocab, 0.3, 11)
    eng, orc, _ = make_pair(shape, (1, 2), max_seqs=2, max_seq_len=32)
    s = _streams(shape.vocab, (10,), 25)
    for bad in (dict(temperature=0.0), dict(temperature=-1.0)):
        with pytest.raises(T.TandemError) as e:
            eng.score(s, **bad)
        assert e.value.code == -1
    with pytest.raises(T.TandemError) as e:
        eng.score(_streams(shape.vocab, (33,), 26))                 # longer than max_seq_len
    assert e.value.code == -1
    with pytest.raises(T.TandemError) as e:
        eng.score([np.array([1, shape.vocab], np.int32)])            # id out of range
    assert e.value.code == -1
    assert eng.score([])["sen_logp"] == []
    a = eng.score(s)
    gen = eng.generate(T.TandemParams(ws, p=0.5, temperature=1.0, seed=1), [s[0][:4]], [8])   # the handle still generates
    assert gen["len"][0] == 8
    b = eng.score(s)                                                 # and scoring is repeatable, bit for bit
    for k in ("sen_logp", "jun_logp", "overlap"):
        assert np.array_equal(a[k][0], b[k][0])
    full = eng.score(_streams(shape.vocab, (32,), 27))               # exactly max_seq_len tokens
    assert len(full["overlap"][0]) == 32 and full["overlap"][0][1:].min() > 0
    eng.free()

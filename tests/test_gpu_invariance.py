"""-m gpu: properties that need no oracle (VII.4) and API error behaviour."""
import numpy as np
import pytest
import torch

import paper_2606_28166_b200 as T
from workloads import get_workload, make_weights, make_word_start, ModelShape
from gpu_util import make_pair

pytestmark = pytest.mark.gpu
SHAPE = get_workload("cfg1_tiny_f32").shape


def _prompts(n, seed=3):
    rng = np.random.default_rng(seed)
    return [rng.integers(0, SHAPE.vocab, size=int(rng.integers(4, 40))).astype(np.int32) for _ in range(n)]


@pytest.mark.parametrize("p", [0.1, 0.5, 1.0])
def test_identical_weights_tokens_equal_solo(p):
    """same-init pair => the token stream cannot depend on the ownership schedule (catch-up test)."""
    eng, _, _ = make_pair(SHAPE, same=True, max_seqs=6, max_seq_len=128)
    ws = make_word_start(SHAPE.vocab, 0.5, 4)
    prompts = _prompts(6)
    solo = eng.generate(T.TandemParams(ws, p=0.0, temperature=1.0, seed=9), prompts, [60] * 6)
    tan = eng.generate(T.TandemParams(ws, p=p, temperature=1.0, seed=9), prompts, [60] * 6)
    assert np.array_equal(solo["tokens"], tan["tokens"])
    assert not solo["owner"].any() and tan["owner"].any()
    assert tan["stats"]["catchup_rows"] > 0
    eng.free()


def test_batch_composition_and_determinism():
    """Batch of 1 vs batch of 5 vs a 2-slot engine with queueing vs a tiny row budget: identical per-sequence results;
    the same call twice gives identical bytes."""
    ws = make_word_start(SHAPE.vocab, 0.3, 4)
    prompts = _prompts(5, seed=8)
    prm = T.TandemParams(ws, p=0.5, temperature=1.0, seed=77)
    ids = np.arange(5, dtype=np.int32) + 100
    eng, _, _ = make_pair(SHAPE, max_seqs=5, max_seq_len=128)
    a = eng.generate(prm, prompts, [50] * 5, seq_ids=ids)
    b = eng.generate(prm, prompts, [50] * 5, seq_ids=ids)
    for k in ("tokens", "owner", "sen_logp", "len"):
        assert np.array_equal(a[k], b[k])
    for i in range(5):
        one = eng.generate(prm, [prompts[i]], [50], seq_ids=ids[i:i + 1])
        assert np.array_equal(one["tokens"][0], a["tokens"][i]) and np.array_equal(one["owner"][0], a["owner"][i])
        assert np.array_equal(one["sen_logp"][0], a["sen_logp"][i])
    eng.free()
    eng2, _, _ = make_pair(SHAPE, max_seqs=2, max_seq_len=128, max_rows_per_step=7, use_graph=1)
    c = eng2.generate(prm, prompts, [50] * 5, seq_ids=ids)
    for k in ("tokens", "owner", "len"):
        assert np.array_equal(a[k], c[k])
    assert np.max(np.abs(a["sen_logp"] - c["sen_logp"])) < 1e-5
    eng2.free()


def test_api_errors():
    ws = make_word_start(SHAPE.vocab, 0.3, 4)
    eng = T.Tandem(T.TandemConfig(SHAPE, max_seqs=2, max_seq_len=32))
    prm = T.TandemParams(ws)
    with pytest.raises(T.TandemError) as e:
        eng.generate(prm, _prompts(1), [4])
    assert e.value.code == -4                                   # ESTATE: no weights yet
    eng.free()
    eng, _, _ = make_pair(SHAPE, max_seqs=2, max_seq_len=32)
    for bad in (dict(p=1.5), dict(top_p=0.0), dict(top_p=1.5), dict(temperature=-1.0), dict(cap_k=-1), dict(eos_id=SHAPE.vocab)):
        with pytest.raises(T.TandemError) as e:
            eng.generate(T.TandemParams(ws, **bad), [np.arange(4, dtype=np.int32)], [4])
        assert e.value.code == -1
    with pytest.raises(T.TandemError) as e:                     # prompt + max_new > max_seq_len
        eng.generate(prm, [np.zeros(30, np.int32)], [4])
    assert e.value.code == -1
    with pytest.raises(T.TandemError) as e:                     # id out of range
        eng.generate(prm, [np.array([1, SHAPE.vocab], np.int32)], [4])
    assert e.value.code == -1
    with pytest.raises(T.TandemError) as e:                     # more admissions than slots through tandem_step
        eng.step(prm, admit=([p[:4] for p in _prompts(3)], None, [2, 2, 2]))
    assert e.value.code == -5
    out = eng.generate(prm, [p[:8] for p in _prompts(2)], [4, 4])   # the handle is still usable
    assert out["len"].tolist() == [4, 4]
    assert eng.generate(prm, [], np.zeros(0, np.int32))["len"].shape == (0,)     # empty batch
    eng.free()
    with pytest.raises(T.TandemError):
        T.Tandem(T.TandemConfig(ModelShape(1, 64, 3, 2, 32, 64, 64, dtype="f32"), max_seqs=2, max_seq_len=32))


def test_kv_pool_exhaustion_is_reported():
    ws = make_word_start(SHAPE.vocab, 0.3, 4)
    page_bytes = 2 * SHAPE.n_layers * SHAPE.n_kv_heads * 16 * SHAPE.head_dim * 4
    eng, _, _ = make_pair(SHAPE, max_seqs=4, max_seq_len=128, kv_bytes_per_model=page_bytes * 4)   # 3 usable pages
    with pytest.raises(T.TandemError) as e:
        eng.generate(T.TandemParams(ws), _prompts(4), [60] * 4)
    assert e.value.code == -2
    eng.free()


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_non_finite_logits_cannot_index_out_of_bounds(dtype):
    """Weights with a NaN (here: the final norm's gains) make every logit NaN, no id ever wins an argmax comparison and the merged id keeps its
    'none yet' value: the samplers (materialised-logits kernel for fp32, the LM head's fused epilogue + merge kernel for bf16) then emit an id
    inside the vocabulary (0 where nothing won) instead of using that value as an index into the logits, the word-start table and the embedding.
    The call returns and the device is healthy (before the guard: an illegal memory access, which is expensive to clear on a shared pool)."""
    shape = ModelShape(2, 256, 4, 2, 64, 512, 4100, 1e-6, 1e6, dtype)
    w = [make_weights(shape, s, device="cuda") for s in (1, 2)]
    for x in w:
        x["final_norm"] = torch.full_like(x["final_norm"], float("nan"))
    eng = T.Tandem(T.TandemConfig(shape, max_seqs=3, max_seq_len=48))
    eng.load_weights(0, w[0]); eng.load_weights(1, w[1])
    table = make_word_start(shape.vocab, 0.3, 4)
    for temperature in (1.0, 0.0):
        out = eng.generate(T.TandemParams(table, p=0.5, temperature=temperature, seed=3), [np.arange(5, 14, dtype=np.int32)] * 3, [6] * 3)
        assert out["len"].tolist() == [6, 6, 6] and (out["tokens"] >= 0).all() and (out["tokens"] < shape.vocab).all()
    torch.cuda.synchronize()
    eng.free()

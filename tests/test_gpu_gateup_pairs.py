"""-m gpu: the persistent gate/up + SwiGLU kernel of decode-sized steps (csrc/gemm_streamk.cuh) against the
one-tile-per-CTA tcgen05 kernel it replaces, at the only width where it is live (the 4B shape: 76 tile pairs per model on 74 CTAs).

tests/test_gpu_full_width.py compares the engine that contains it with the float64 oracle (1 and 2 layers of the 4B shape). Here:
  * every launch mode against the old kernel on the same teacher-forced stream - one model active (the senior's prompt prefill: each CTA one
    tile of every pair), both models active (tile pairs), more than 256 token rows in a launch (three 256-row chunks through the one-chunk
    scratch: prompts of 300 and 270 ids, first in the senior's prefill, then in the junior's first catch-ups while the senior decodes):
    owner flags identical, senior log-probs within 1e-3 (whole pairs give the same bits as the old kernel; the two K-sliced leftover
    pairs of each model - 512 of 19,456 gate/up rows - are summed in 37 slices instead of one run, so a bf16 SwiGLU output can move by an ulp);
  * batch invariance, bit for bit: a sequence generated alone (one row per step, the models take turns: single-tile mode) and inside a batch of
    six (tile pairs, other row counts, other chunking) gives the same tokens and the same log-prob bits - the cuts depend on the shape only;
  * the counters return to zero after every launch: the same call twice gives identical bytes.
"""
import numpy as np
import pytest
import torch

import paper_2606_28166_b200 as T
from workloads import ModelShape, make_weights, make_word_start, get_workload

pytestmark = pytest.mark.gpu
FOURB = get_workload("cfg3_4b_bf16").shape
SHAPE = ModelShape(1, FOURB.hidden, FOURB.n_q_heads, FOURB.n_kv_heads, FOURB.head_dim, FOURB.intermediate, 4096, FOURB.rms_eps, FOURB.rope_theta, "bf16")
LENS = (300, 20, 45, 270, 33, 64)
N_NEW = 24


@pytest.fixture(scope="module")
def setup():
    ws = make_weights(SHAPE, 1, device="cuda", gain_jitter=0.1); wj = make_weights(SHAPE, 2, device="cuda", gain_jitter=0.1)
    table = make_word_start(SHAPE.vocab, 0.30, 3)
    rng = np.random.default_rng(5)
    prompts = [rng.integers(0, SHAPE.vocab, size=n).astype(np.int32) for n in LENS]
    return ws, wj, table, prompts


def _engine(ws, wj, max_seqs, streamk):
    eng = T.Tandem(T.TandemConfig(SHAPE, max_seqs=max_seqs, max_seq_len=400, use_graph=1))
    eng.load_weights(0, ws); eng.load_weights(1, wj)
    eng.set_option("gateup_streamk", streamk)
    return eng


def test_every_launch_mode_against_the_one_tile_kernel(setup):
    ws, wj, table, prompts = setup
    B = len(prompts)
    prm = T.TandemParams(table, p=0.5, temperature=1.0, seed=77)
    new = _engine(ws, wj, B, 1)
    a = new.generate(prm, prompts, [N_NEW] * B)
    a2 = new.generate(prm, prompts, [N_NEW] * B)          # counters back at zero, scratch reused: identical bytes
    new.free()
    for k in ("tokens", "owner", "sen_logp", "len"):
        assert np.array_equal(a[k], a2[k]), k
    assert (a["len"] == N_NEW).all() and 0.2 < a["owner"].mean() < 0.8
    # the junior ingests a whole long prompt while the senior decodes: a launch with both models active and > 256 rows for one of them
    assert a["owner"][0].any() and a["owner"][3].any()
    old = _engine(ws, wj, B, 0)
    forced = torch.as_tensor(a["tokens"].astype(np.int32)).cuda()
    b = old.generate(prm, prompts, [N_NEW] * B, forced_tokens=forced)
    old.free()
    assert np.array_equal(a["owner"], b["owner"]) and np.array_equal(a["tokens"], b["tokens"])
    sen = a["owner"] == 0
    d = np.abs(a["sen_logp"] - b["sen_logp"])[sen]
    print("gate/up pairs vs one-tile kernel: max |dlogp| %.2e, mean %.2e over %d senior positions" % (d.max(), d.mean(), d.size))
    assert d.max() <= 1e-3 and d.mean() <= 4e-5          # measured on B200: max 4.7e-4, mean 1.9e-5 over 52 senior positions


def test_alone_equals_inside_the_batch_bit_for_bit(setup):
    ws, wj, table, prompts = setup
    B = len(prompts)
    prm = T.TandemParams(table, p=0.5, temperature=1.0, seed=77)
    eng = _engine(ws, wj, B, 1)
    full = eng.generate(prm, prompts, [N_NEW] * B)
    for b in (1, 3):                                       # a short prompt and one of more than 256 rows
        eng.reset()
        solo = eng.generate(prm, [prompts[b]], [N_NEW], seq_ids=[b])
        assert np.array_equal(solo["tokens"][0], full["tokens"][b]) and np.array_equal(solo["owner"][0], full["owner"][b])
        assert np.array_equal(solo["sen_logp"][0].view(np.uint32), full["sen_logp"][b].view(np.uint32))
    eng.free()

"""-m gpu: configs[0] (tiny tandem, fp32) free-running against the oracle - DESIGN.md section 5, VII.2.
Tokens, owners, lengths identical; owner's logits max|dz|/max|z| <= 1e-4 at every step (BASELINE.json);
senior log-probs within 1e-5."""
import numpy as np
import pytest
import torch

import paper_2606_28166_b200 as T
from oracle import TandemParams as OParams, tandem_generate, owners_from_tokens
from oracle.rule import Uniforms
from workloads import get_workload, make_word_start, make_prompts, make_explicit_uniforms, ModelShape
from gpu_util import make_pair, dev

pytestmark = pytest.mark.gpu


def _cfg1():
    wl = get_workload("cfg1_tiny_f32")
    ws = make_word_start(wl.shape.vocab, wl.word_start_frac, wl.seeds["table"])
    prompts = make_prompts(wl)
    usw, usa = make_explicit_uniforms(wl.batch, wl.max_new, wl.shape.vocab, wl.seeds["uniforms"])
    return wl, ws, prompts, usw, usa


def _compare(out, ref, B, logp_tol=1e-5):
    for b in range(B):
        n = len(ref["tokens"][b])
        assert out["len"][b] == n
        assert np.array_equal(out["tokens"][b, :n], ref["tokens"][b]), (b, out["tokens"][b, :n], ref["tokens"][b])
        assert np.array_equal(out["owner"][b, :n], ref["owner"][b])
        assert np.array_equal(out["mask"][b, :n], ref["mask"][b])
        assert np.max(np.abs(out["sen_logp"][b, :n] - ref["sen_logp"][b])) <= logp_tol


@pytest.mark.parametrize("use_graph", [0, 1])
def test_cfg1_generate_matches_oracle(use_graph):
    wl, ws, prompts, usw, usa = _cfg1()
    eng, orc, _ = make_pair(wl.shape, (wl.seeds["senior"], wl.seeds["junior"]), max_seqs=wl.batch, max_seq_len=64, use_graph=use_graph)
    ref = tandem_generate(orc, OParams(p=wl.p, temperature=0.0), prompts, [wl.max_new] * wl.batch, ws,
                          uni=Uniforms(u_switch=usw, u_sample=usa))
    out = eng.generate(T.TandemParams(ws, p=wl.p, temperature=0.0), prompts, [wl.max_new] * wl.batch, u_switch=dev(usw))
    _compare(out, ref, wl.batch)
    assert out["stats"]["tokens_emitted"] == wl.batch * wl.max_new
    assert out["stats"]["rows_junior"] > 0 and out["stats"]["catchup_rows"] > 0
    # the integer rule replayed on the GPU's own tokens reproduces its owner flags byte for byte (VII.1)
    for b in range(wl.batch):
        o = owners_from_tokens(out["tokens"][b, :out["len"][b]], ws, OParams(p=wl.p), Uniforms(u_switch=usw), b=b)
        assert np.array_equal(o, out["owner"][b, :out["len"][b]])
    eng.free()


def test_cfg1_step_logits_within_1e4():
    wl, ws, prompts, usw, usa = _cfg1()
    B, V = wl.batch, wl.shape.vocab
    eng, orc, _ = make_pair(wl.shape, (wl.seeds["senior"], wl.seeds["junior"]), max_seqs=B, max_seq_len=64)
    ref = tandem_generate(orc, OParams(p=wl.p, temperature=0.0), prompts, [wl.max_new] * B, ws,
                          uni=Uniforms(u_switch=usw, u_sample=usa), want_logits=True)
    prm = T.TandemParams(ws, p=wl.p, temperature=0.0)
    o = dict(token=torch.zeros(B, dtype=torch.int32, device="cuda"), owner=torch.zeros(B, dtype=torch.uint8, device="cuda"),
             sen_logp=torch.zeros(B, device="cuda"), done=torch.zeros(B, dtype=torch.uint8, device="cuda"),
             argmax=torch.zeros(B, dtype=torch.int32, device="cuda"), n_active=torch.zeros(1, dtype=torch.int32, device="cuda"))
    dbg = torch.zeros(B, V, device="cuda")
    usw_d = dev(usw)
    worst = 0.0
    for t in range(wl.max_new):
        slots = eng.step(prm, admit=(prompts, None, [wl.max_new] * B) if t == 0 else None, out=o, u_switch=usw_d, dbg_logits=dbg)
        if t == 0:
            assert slots.tolist() == list(range(B))
        torch.cuda.synchronize()
        tok = o["token"].cpu().numpy(); own = o["owner"].cpu().numpy(); z = dbg.cpu().numpy().astype(np.float64)
        for b in range(B):
            assert tok[b] == ref["tokens"][b][t] and own[b] == ref["owner"][b][t]
            zr = ref["logits"][b][t]
            worst = max(worst, np.max(np.abs(z[b] - zr)) / np.max(np.abs(zr)))
            assert o["argmax"][b].item() == int(np.argmax(zr))
        assert int(o["n_active"].item()) == (B if t < wl.max_new - 1 else 0)
    assert worst <= 1e-4, worst
    assert o["done"].cpu().numpy().all()
    eng.free()


@pytest.mark.parametrize("mode,start,p,cap", [(T.TOGGLE, T.SENIOR, 0.5, 0), (T.REDRAW, T.DRAW, 0.5, 0), (T.TOGGLE, T.JUNIOR, 1.0, 0),
                                              (T.TOGGLE, T.SENIOR, 0.0, 0), (T.REDRAW, T.SENIOR, 0.3, 3), (T.TOGGLE, T.DRAW, 0.7, 2)])
def test_sampled_rollouts_match_oracle_counter_rng(mode, start, p, cap):
    """T = 1 sampling from the counter generator (no explicit arrays), both rule modes, DRAW start, cap, EOS,
    ragged prompt lengths and ragged max_new, B > max_seqs (queued admission), multi-page contexts."""
    shape = get_workload("cfg1_tiny_f32").shape
    ws = make_word_start(shape.vocab, 0.3, 11)
    rng = np.random.default_rng(5)
    B = 7
    prompts = [rng.integers(0, shape.vocab, size=int(n)).astype(np.int32) for n in (1, 15, 16, 17, 33, 40, 5)]
    max_new = np.array([40, 7, 33, 1, 20, 37, 48], dtype=np.int32)
    seq_ids = np.array([10, 11, 12, 13, 14, 15, 99], dtype=np.int32)
    eng, orc, _ = make_pair(shape, (1, 2), max_seqs=4, max_seq_len=96, gain_jitter=0.1, max_rows_per_step=24)
    op = OParams(p=p, switch_mode=mode, start_owner=start, cap_k=cap, temperature=1.0, eos_id=3, seed=1234)
    ref = tandem_generate(orc, op, prompts, max_new, ws, uni=Uniforms(seed=1234, seq_ids=seq_ids))
    out = eng.generate(T.TandemParams(ws, p=p, switch_mode=mode, start_owner=start, cap_k=cap, temperature=1.0, eos_id=3, seed=1234),
                       prompts, max_new, seq_ids=seq_ids)
    _compare(out, ref, B, logp_tol=2e-5)
    eng.free()


@pytest.mark.parametrize("temperature,top_p,top_k", [(0.7, 0.8, 0), (1.0, 0.3, 0), (0.6, 0.95, 0), (0.7, 0.8, 20), (1.0, 1.0, 5), (0.9, 1.0, 1)])
def test_nucleus_rollouts_match_oracle(temperature, top_p, top_k):
    """top-p < 1 and top-k (the evaluation setting T = 0.7, top-p 0.8, top-k 20 of Table 3 among them; top-k 1 = greedy): tokens,
    owners, mask as the oracle's; the log-prob is that of the untruncated softmax(z/T) (R11)."""
    shape = get_workload("cfg1_tiny_f32").shape
    ws = make_word_start(shape.vocab, 0.3, 11)
    rng = np.random.default_rng(8)
    B = 5
    prompts = [rng.integers(0, shape.vocab, size=int(n)).astype(np.int32) for n in (3, 16, 21, 9, 30)]
    max_new = np.array([30, 24, 17, 32, 8], dtype=np.int32)
    eng, orc, _ = make_pair(shape, (1, 2), max_seqs=3, max_seq_len=64, gain_jitter=0.1)
    op = OParams(p=0.5, temperature=temperature, top_p=top_p, top_k=top_k, eos_id=3, seed=77)
    ref = tandem_generate(orc, op, prompts, max_new, ws, uni=Uniforms(seed=77, seq_ids=np.arange(B, dtype=np.int32)))
    out = eng.generate(T.TandemParams(ws, p=0.5, temperature=temperature, top_p=top_p, top_k=top_k, eos_id=3, seed=77), prompts, max_new)
    _compare(out, ref, B, logp_tol=2e-5)
    solo = eng.generate(T.TandemParams(ws, p=0.5, temperature=temperature, top_p=1.0, eos_id=3, seed=77), prompts, max_new)
    assert any(not np.array_equal(solo["tokens"][b, :out["len"][b]], out["tokens"][b, :out["len"][b]]) for b in range(B))  # the filter bites
    eng.free()


@pytest.mark.parametrize("mode,p", [(T.TOGGLE, 1.0), (T.REDRAW, 0.5)])
def test_reasoning_step_handoff_protocol(mode, p):
    """The paper's evaluation protocol (L99 section 4.3: strict alternation at every boundary token; L480 App. C.5: Bernoulli(0.5)
    draw of the next contributor) with the evaluation sampler (T 0.7, top-p 0.8, top-k 20): a sparse boundary table, TOGGLE p = 1
    or REDRAW p = 0.5. Tokens / owners / mask as the oracle's; under strict alternation the owner changes exactly after each
    boundary token and never elsewhere."""
    shape = get_workload("cfg1_tiny_f32").shape
    ws = make_word_start(shape.vocab, 0.08, 13)
    rng = np.random.default_rng(9)
    B = 4
    prompts = [rng.integers(0, shape.vocab, size=int(n)).astype(np.int32) for n in (5, 18, 31, 12)]
    max_new = np.array([48, 40, 33, 48], dtype=np.int32)
    eng, orc, _ = make_pair(shape, (1, 2), max_seqs=4, max_seq_len=96, gain_jitter=0.1)
    kw = dict(p=p, switch_mode=mode, temperature=0.7, top_p=0.8, top_k=20, seed=31)
    ref = tandem_generate(orc, OParams(**kw), prompts, max_new, ws, uni=Uniforms(seed=31, seq_ids=np.arange(B, dtype=np.int32)))
    out = eng.generate(T.TandemParams(ws, **kw), prompts, max_new)
    _compare(out, ref, B, logp_tol=2e-5)
    switches = 0
    for b in range(B):
        n = out["len"][b]
        tok, own = out["tokens"][b, :n], out["owner"][b, :n]
        flips = own[1:] != own[:-1]
        boundary = ws[tok[:-1]].astype(bool)
        if mode == T.TOGGLE:
            assert np.array_equal(flips, boundary)
        else:
            assert not flips[~boundary].any()
        switches += int(flips.sum())
    assert switches >= 3
    eng.free()


def test_explicit_sample_uniforms_and_forced_tokens():
    shape = get_workload("cfg1_tiny_f32").shape
    ws = make_word_start(shape.vocab, 0.3, 11)
    rng = np.random.default_rng(6)
    B, L = 3, 12
    prompts = [rng.integers(0, shape.vocab, size=9).astype(np.int32) for _ in range(B)]
    usw, usa = make_explicit_uniforms(B, L, shape.vocab, 9)
    forced = np.full((B, L), -1, dtype=np.int32)
    forced[1, 3:6] = [7, 8, 9]
    forced[2, 8] = 5                                       # EOS forced at t = 9
    eng, orc, _ = make_pair(shape, (1, 2), max_seqs=B, max_seq_len=32)
    op = OParams(p=0.5, temperature=0.8, eos_id=5)
    ref = tandem_generate(orc, op, prompts, [L] * B, ws, uni=Uniforms(u_switch=usw, u_sample=usa), forced=list(forced))
    out = eng.generate(T.TandemParams(ws, p=0.5, temperature=0.8, eos_id=5), prompts, [L] * B, u_switch=dev(usw), u_sample=dev(usa),
                       forced_tokens=dev(forced))
    _compare(out, ref, B, logp_tol=2e-5)
    assert out["len"][2] <= 9
    eng.free()


def test_generate_queues_when_the_kv_pool_is_short():
    """A page pool that holds about two rollouts at a time: tandem_generate admits by reservation (whole context of a sequence
    must fit in each model's pool), the rest waits; results still equal the oracle's and no page runs out mid-rollout. A
    sequence that can never fit is refused with TANDEM_ENOMEM up front."""
    shape = get_workload("cfg1_tiny_f32").shape
    ws = make_word_start(shape.vocab, 0.3, 11)
    rng = np.random.default_rng(8)
    B = 6
    prompts = [rng.integers(0, shape.vocab, size=int(n)).astype(np.int32) for n in (20, 33, 7, 48, 16, 30)]
    max_new = np.array([30, 12, 40, 16, 25, 31], dtype=np.int32)
    page_bytes = 2 * shape.n_layers * shape.n_kv_heads * 16 * shape.head_dim * 4
    eng, orc, _ = make_pair(shape, (1, 2), max_seqs=6, max_seq_len=96, kv_bytes_per_model=9 * page_bytes)   # 8 usable pages = 128 positions
    op = OParams(p=0.5, temperature=1.0, seed=77)
    ref = tandem_generate(orc, op, prompts, max_new, ws, uni=Uniforms(seed=77))
    out = eng.generate(T.TandemParams(ws, p=0.5, temperature=1.0, seed=77), prompts, max_new)
    _compare(out, ref, B, logp_tol=2e-5)
    assert out["stats"]["peak_resident"] < B and max(out["stats"]["peak_pages_senior"], out["stats"]["peak_pages_junior"]) <= 8
    with pytest.raises(T.TandemError) as e:
        eng.generate(T.TandemParams(ws, p=0.5, temperature=1.0, seed=77), [np.zeros(90, np.int32)], [60])
    assert e.value.code == -1 or e.value.code == -2      # prompt + max_new > max_seq_len (EINVAL) or > pool (ENOMEM)
    eng.free()
    eng2, _, _ = make_pair(shape, (1, 2), max_seqs=2, max_seq_len=96, kv_bytes_per_model=4 * page_bytes)   # 3 usable pages = 48 positions
    with pytest.raises(T.TandemError) as e:
        eng2.generate(T.TandemParams(ws, p=0.5, temperature=1.0, seed=77), [np.zeros(40, np.int32)], [16])   # 56 positions = 4 pages
    assert e.value.code == -2
    eng2.free()


def test_generate_preempts_when_a_pool_runs_dry_and_redoes_bit_identically():
    """Continuous batching: admission on current need + a watermark lets all four sequences in, their
    growth then exhausts a 16-page pool (each needs 7 pages per model at the end), the scheduler stalls what it cannot serve and
    tandem_generate preempts the youngest sequence and redoes it later from its prompt. Position-addressed random draws make the
    redo bit-identical: tokens, owners, lengths equal the oracle's, which knows nothing of pages."""
    shape = get_workload("cfg1_tiny_f32").shape
    ws = make_word_start(shape.vocab, 0.3, 11)
    rng = np.random.default_rng(18)
    B = 4
    prompts = [rng.integers(0, shape.vocab, size=10).astype(np.int32) for _ in range(B)]
    max_new = np.array([100, 100, 100, 100], dtype=np.int32)
    page_bytes = 2 * shape.n_layers * shape.n_kv_heads * 16 * shape.head_dim * 4
    eng, orc, _ = make_pair(shape, (1, 2), max_seqs=4, max_seq_len=128, kv_bytes_per_model=17 * page_bytes)   # 16 usable pages
    op = OParams(p=0.5, temperature=1.0, seed=5)
    ref = tandem_generate(orc, op, prompts, max_new, ws, uni=Uniforms(seed=5))
    out = eng.generate(T.TandemParams(ws, p=0.5, temperature=1.0, seed=5), prompts, max_new)
    _compare(out, ref, B, logp_tol=2e-5)
    st = out["stats"]
    assert st["preemptions"] >= 1 and st["starved"] >= 1, st
    assert st["peak_resident"] == 4 and max(st["peak_pages_senior"], st["peak_pages_junior"]) <= 16
    again = eng.generate(T.TandemParams(ws, p=0.5, temperature=1.0, seed=5), prompts, max_new)      # and the call is repeatable
    for k in ("tokens", "owner", "sen_logp", "len"):
        assert np.array_equal(out[k], again[k])
    eng.free()


def test_step_stalls_on_an_empty_pool_and_reports_the_dead_lock():
    """tandem_step on a pool too small for the admitted sequences: the scheduler stalls sequences instead of handing out the dummy
    page (tokens emitted so far equal the oracle's), `starved` counts the stalls, and once nothing can move the next call returns
    TANDEM_ENOMEM. tandem_reset makes the handle usable again."""
    shape = get_workload("cfg1_tiny_f32").shape
    ws = make_word_start(shape.vocab, 0.3, 11)
    rng = np.random.default_rng(19)
    B = 3
    prompts = [rng.integers(0, shape.vocab, size=12).astype(np.int32) for _ in range(B)]
    page_bytes = 2 * shape.n_layers * shape.n_kv_heads * 16 * shape.head_dim * 4
    eng, orc, _ = make_pair(shape, (1, 2), max_seqs=B, max_seq_len=128, kv_bytes_per_model=7 * page_bytes)    # 6 usable pages = 96 positions
    prm = T.TandemParams(ws, p=0.5, temperature=1.0, seed=6)
    ref = tandem_generate(orc, OParams(p=0.5, temperature=1.0, seed=6), prompts, [100] * B, ws, uni=Uniforms(seed=6))
    o = dict(token=torch.zeros(B, dtype=torch.int32, device="cuda"), owner=torch.zeros(B, dtype=torch.uint8, device="cuda"))
    got = [[] for _ in range(B)]
    err = None
    for t in range(200):
        try:
            eng.step(prm, admit=(prompts, None, [100] * B) if t == 0 else None, out=o)
        except T.TandemError as e:
            err = e
            break
        torch.cuda.synchronize()
        tok = o["token"].cpu().numpy()
        for b in range(B):
            if tok[b] >= 0:
                got[b].append(int(tok[b]))
    assert err is not None and err.code == -2, "the dead lock must surface as TANDEM_ENOMEM"
    for b in range(B):                                       # everything emitted before the stall is right
        assert len(got[b]) > 0 and got[b] == [int(x) for x in ref["tokens"][b][:len(got[b])]]
    assert sum(len(g) for g in got) < 3 * 100
    # tandem_evict gives the pages of one sequence back: the others move again and stay on the oracle's token streams
    eng.evict(2)
    before = [len(g) for g in got]
    for t in range(40):
        try:
            eng.step(prm, out=o)
        except T.TandemError:
            break
        torch.cuda.synchronize()
        tok = o["token"].cpu().numpy()
        assert tok[2] < 0
        for b in range(2):
            if tok[b] >= 0:
                got[b].append(int(tok[b]))
    assert len(got[0]) + len(got[1]) > before[0] + before[1]
    for b in range(2):
        assert got[b] == [int(x) for x in ref["tokens"][b][:len(got[b])]]
    with pytest.raises(T.TandemError):
        eng.evict(2)                                          # the slot is empty now
    eng.reset()
    out = eng.generate(prm, [prompts[0]], [20])
    assert np.array_equal(out["tokens"][0, :20], ref["tokens"][0][:20])
    eng.free()


@pytest.mark.parametrize("mode,start,p,share", [(T.TOGGLE, T.SENIOR, 0.5, 0), (T.REDRAW, T.DRAW, 0.5, 1), (T.TOGGLE, T.JUNIOR, 1.0, 0)])
def test_dual_forward_measurement_mode_follows_the_same_rule(mode, start, p, share):
    """The paper's own engine as a measurement mode (tandem_test_set_option "dual_forward"):
    both models ingest every emitted token in lock-step and only the owner samples, so the rollout is the oracle's, token for token,
    while each model computes one row per resident sequence and step (no catch-up bursts) - both models end up with the same row count."""
    shape = get_workload("cfg1_tiny_f32").shape
    ws = make_word_start(shape.vocab, 0.3, 11)
    rng = np.random.default_rng(6)
    B = 6
    base = [rng.integers(0, shape.vocab, size=int(n)).astype(np.int32) for n in (3, 17, 33)]
    prompts = [base[i // 2] for i in range(B)]                      # groups of two rollouts per prompt
    max_new = np.array([30, 12, 33, 5, 20, 37], dtype=np.int32)
    eng, orc, _ = make_pair(shape, (1, 2), max_seqs=6, max_seq_len=96, gain_jitter=0.1, max_rows_per_step=24, share_prompt_pages=share)
    eng.set_option("dual_forward", 1)
    op = OParams(p=p, switch_mode=mode, start_owner=start, temperature=1.0, eos_id=3, seed=77)
    ref = tandem_generate(orc, op, prompts, max_new, ws, uni=Uniforms(seed=77, seq_ids=np.arange(B, dtype=np.int32)))
    out = eng.generate(T.TandemParams(ws, p=p, switch_mode=mode, start_owner=start, temperature=1.0, eos_id=3, seed=77), prompts, max_new)
    _compare(out, ref, B, logp_tol=2e-5)
    st = out["stats"]
    # every model ingested every prompt (less what it took from shared pages) and every emitted token but each sequence's last one
    ingested = sum(len(p_) for p_ in prompts) + int(out["len"].sum()) - B
    assert st["rows_senior"] == st["rows_junior"] == ingested - st["shared_prompt_rows"] // 2
    # the default engine on the same problem computes fewer rows (a model that never takes a sequence over again skips its tail)
    eng.set_option("dual_forward", 0)
    out2 = eng.generate(T.TandemParams(ws, p=p, switch_mode=mode, start_owner=start, temperature=1.0, eos_id=3, seed=77), prompts, max_new)
    _compare(out2, ref, B, logp_tol=2e-5)
    assert out2["stats"]["rows_senior"] + out2["stats"]["rows_junior"] <= st["rows_senior"] + st["rows_junior"]
    eng.free()

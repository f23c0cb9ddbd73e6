"""-m gpu: prompt-page sharing across the G rollouts of a prompt (tandem_config.share_prompt_pages; SURVEY.md section 8(a)
"pages"). The K/V of equal prefixes are equal, so the outputs must be those of the oracle (which knows
nothing about pages) and of the engine without sharing; what changes is the bookkeeping: prompt rows computed once per model and
group, fewer pages in use, every page back in the pool at the end."""
import numpy as np
import pytest
import torch

import paper_2606_28166_b200 as T
from oracle import TandemParams as OParams, tandem_generate
from oracle.rule import Uniforms
from workloads import get_workload, make_word_start, ModelShape
from gpu_util import make_pair

pytestmark = pytest.mark.gpu
TINY = get_workload("cfg1_tiny_f32").shape


def _grouped_prompts(shape, lens, group, seed):
    rng = np.random.default_rng(seed)
    out = []
    for n in lens:
        ids = rng.integers(0, shape.vocab, size=n).astype(np.int32)
        out.extend([ids.copy() for _ in range(group)])
    return out


def _same(out, ref, B, logp_tol):
    for b in range(B):
        n = out["len"][b]
        assert n == len(ref["tokens"][b])
        assert np.array_equal(out["tokens"][b, :n], ref["tokens"][b]), b
        assert np.array_equal(out["owner"][b, :n], ref["owner"][b]), b
        assert np.max(np.abs(out["sen_logp"][b, :n] - ref["sen_logp"][b])) < logp_tol


@pytest.mark.parametrize("share", [1, 2])
@pytest.mark.parametrize("start,rows,graph", [(T.SENIOR, 0, 1), (T.DRAW, 0, 0), (T.SENIOR, 24, 1), (T.JUNIOR, 9, 0)])
def test_shared_prompt_pages_match_oracle(start, rows, graph, share):
    """fp32, 3 prompts x 4 rollouts (lengths 40, 17, 70: 2, 1 and 4 shared pages) plus an ungrouped short prompt; also with
    a row budget that chunks the donor's prefill over several steps (followers wait) and with drawn start owners.
    share = 2: the members of a group that a model serves in a step also READ the shared pages once (shared-prefix runs: q-tiles over
    the members' rows against positions [0, Ls), merged with each member's own splits by the combine kernel)."""
    table = make_word_start(TINY.vocab, 0.3, 5)
    prompts = _grouped_prompts(TINY, (40, 17, 70), 4, seed=21) + [np.arange(9, dtype=np.int32)]
    B = len(prompts)
    max_new = [28] * B
    eng, orc, _ = make_pair(TINY, (1, 2), max_seqs=B, max_seq_len=112, share_prompt_pages=share, max_rows_per_step=rows, use_graph=graph)
    ref = tandem_generate(orc, OParams(p=0.5, temperature=1.0, seed=91, start_owner=start), prompts, max_new, table, uni=Uniforms(seed=91))
    out = eng.generate(T.TandemParams(table, p=0.5, temperature=1.0, seed=91, start_owner=start), prompts, max_new)
    _same(out, ref, B, 2e-5)
    st = out["stats"]
    # the start model computes each group's shared prefix once: the other three members take it over (32 + 16 + 64 positions)
    assert st["shared_prompt_rows"] >= 3 * (32 + 16 + 64)
    assert (st["kv_bytes_shared_reads"] > 0) == (share == 2)      # runs of members were formed and read the shared pages together
    assert 0 < out["owner"].mean() < 1
    eng.free()
    # without sharing: same outputs, more rows, more pages
    eng0, _, _ = make_pair(TINY, (1, 2), max_seqs=B, max_seq_len=112, share_prompt_pages=0, max_rows_per_step=rows, use_graph=graph)
    out0 = eng0.generate(T.TandemParams(table, p=0.5, temperature=1.0, seed=91, start_owner=start), prompts, max_new)
    eng0.free()
    for k in ("tokens", "owner", "len"):
        assert np.array_equal(out[k], out0[k])
    assert np.max(np.abs(out["sen_logp"] - out0["sen_logp"])) < 2e-5
    st0 = out0["stats"]
    assert st0["shared_prompt_rows"] == 0
    assert st["rows_senior"] + st["rows_junior"] + st["shared_prompt_rows"] == st0["rows_senior"] + st0["rows_junior"]
    assert st["peak_pages_senior"] < st0["peak_pages_senior"] or st["peak_pages_junior"] < st0["peak_pages_junior"]


def test_shared_pages_are_returned_and_groups_recycled():
    """Queued admission with a pool of a few rollouts: groups come and go (their table entries and pages are reused); a leaked
    page or a stale group entry would end in the pool-exhausted error or in wrong tokens. Some members finish early (EOS)."""
    table = make_word_start(TINY.vocab, 0.3, 5)
    prompts = _grouped_prompts(TINY, (36, 20, 50, 33, 41), 3, seed=4)
    B = len(prompts)
    max_new = np.array([10 + 3 * (b % 5) for b in range(B)], dtype=np.int32)
    page_bytes = 2 * TINY.n_layers * TINY.n_kv_heads * 16 * TINY.head_dim * 4
    eng, orc, _ = make_pair(TINY, (1, 2), max_seqs=4, max_seq_len=96, share_prompt_pages=1, kv_bytes_per_model=21 * page_bytes)
    op = OParams(p=0.5, temperature=1.0, seed=13, eos_id=7)
    ref = tandem_generate(orc, op, prompts, max_new, table, uni=Uniforms(seed=13))
    prm = T.TandemParams(table, p=0.5, temperature=1.0, seed=13, eos_id=7)
    for _ in range(2):
        out = eng.generate(prm, prompts, max_new)
        _same(out, ref, B, 2e-5)
        assert out["stats"]["peak_resident"] <= 4
    eng.free()


def test_shared_prompt_pages_through_tandem_step():
    """The step call with two admissions: a group admitted at step 1, a second group (same prompt as an unrelated single) a few
    steps later while the first is running; a waiting member emits nothing (token -1) until its donor has stored the prefix.
    Per-sequence streams equal the oracle's."""
    table = make_word_start(TINY.vocab, 0.3, 5)
    first = _grouped_prompts(TINY, (40,), 3, seed=6)
    second = [np.arange(30, dtype=np.int32)] + _grouped_prompts(TINY, (52,), 2, seed=7)
    n_new = 20
    eng, orc, _ = make_pair(TINY, (1, 2), max_seqs=6, max_seq_len=96, share_prompt_pages=2, use_graph=1)   # 2: with shared-prefix runs
    prm = T.TandemParams(table, p=0.5, temperature=1.0, seed=3)
    o = dict(token=torch.zeros(6, dtype=torch.int32, device="cuda"), owner=torch.zeros(6, dtype=torch.uint8, device="cuda"),
             done=torch.zeros(6, dtype=torch.uint8, device="cuda"))
    streams = {i: [] for i in range(6)}
    owners = {i: [] for i in range(6)}
    slot_of = {}
    waited = 0
    for t in range(80):
        admit = None
        if t == 0:
            admit = (first, [10, 11, 12], [n_new] * 3)
        elif t == 5:
            admit = (second, [20, 21, 22], [n_new] * 3)
        slots = eng.step(prm, admit=admit, out=o)
        torch.cuda.synchronize()
        if admit is not None:
            for sid, sl in zip(admit[1], slots):
                slot_of[int(sl)] = sid
        tok = o["token"].cpu().numpy(); own = o["owner"].cpu().numpy()
        for sl, sid in slot_of.items():
            if tok[sl] >= 0:
                streams[sl].append(int(tok[sl])); owners[sl].append(int(own[sl]))
            elif len(streams[sl]) < n_new:
                waited += 1
        if all(len(streams[sl]) == n_new for sl in slot_of) and len(slot_of) == 6:
            break
    assert waited >= 2          # the followers of both groups sat out the donor's prefill step
    ref = tandem_generate(orc, OParams(p=0.5, temperature=1.0, seed=3), first + second, [n_new] * 6, table,
                          uni=Uniforms(seed=3, seq_ids=[10, 11, 12, 20, 21, 22]))
    sid_to_b = {10: 0, 11: 1, 12: 2, 20: 3, 21: 4, 22: 5}
    for sl, sid in slot_of.items():
        b = sid_to_b[sid]
        assert streams[sl] == list(ref["tokens"][b]) and owners[sl] == list(ref["owner"][b]), sid
    assert eng.get_stats()["shared_prompt_rows"] >= 2 * 32 + 48
    eng.free()


def test_shared_prompt_pages_bf16():
    """bf16 (tcgen05 GEMM, tensor-core attention): compared with the engine without sharing on the same forced token stream
    (owners exact, log-probs up to bf16 rounding of a different q-tiling)."""
    shape = ModelShape(3, 256, 4, 2, 64, 512, 2048, 1e-6, 1e6, "bf16")
    table = make_word_start(shape.vocab, 0.3, 5)
    prompts = _grouped_prompts(shape, (45, 70), 4, seed=2)
    B, n_new = len(prompts), 24
    prm = T.TandemParams(table, p=0.5, temperature=1.0, seed=5)
    res = []
    forced = None
    for share in (0, 1, 2):
        eng, _, _ = make_pair(shape, (1, 2), max_seqs=B, max_seq_len=128, share_prompt_pages=share, use_graph=1)
        out = eng.generate(prm, prompts, [n_new] * B, forced_tokens=forced)
        res.append(out)
        if forced is None:
            forced = torch.as_tensor(out["tokens"].astype(np.int32)).cuda()
        eng.free()
    a, b, c = res
    for x in (b, c):                                       # 1: shared pages; 2: shared pages read once per run of members as well
        assert np.array_equal(a["tokens"], x["tokens"]) and np.array_equal(a["owner"], x["owner"])
        assert np.max(np.abs(a["sen_logp"] - x["sen_logp"])) < 0.02
        assert x["stats"]["shared_prompt_rows"] >= 3 * (32 + 64)
    assert a["stats"]["shared_prompt_rows"] == 0 and b["stats"]["kv_bytes_shared_reads"] == 0 and c["stats"]["kv_bytes_shared_reads"] > 0


def test_shared_prefix_runs_at_the_4b_width():
    """share_prompt_pages = 2 at the head geometry the benchmark runs (32 q / 8 kv heads of 128: G = 4, 16-token q-tiles, KV splits of 1024
    positions): 2 prompts x 8 rollouts (lengths 150 and 333: 9 and 20 shared pages), one layer of the 4B shape. The engine without sharing and
    the engine with shared-prefix runs follow the same forced token stream; owners are exact, and BOTH are compared with the float64 oracle:
    the runs change where the softmax is cut (at the shared length) and with it the bf16 rounding of P, not the sums - their error against
    the oracle must be the error of the plain path (one layer of this width: max 0.02 / mean 0.006, tests/test_gpu_full_width.py)."""
    from workloads import get_workload
    from oracle import replay_owner_logits
    from oracle.sampler import log_softmax
    f = get_workload("cfg3_4b_bf16").shape
    shape = ModelShape(1, f.hidden, f.n_q_heads, f.n_kv_heads, f.head_dim, f.intermediate, 4096, f.rms_eps, f.rope_theta, "bf16")
    table = make_word_start(shape.vocab, 0.3, 5)
    prompts = _grouped_prompts(shape, (150, 333), 8, seed=4)
    B, n_new = len(prompts), 24
    prm = T.TandemParams(table, p=0.5, temperature=1.0, seed=15)
    res, forced = [], None
    for share in (0, 2):
        eng, models, _ = make_pair(shape, (1, 2), max_seqs=B, max_seq_len=400, share_prompt_pages=share, use_graph=1)
        out = eng.generate(prm, prompts, [n_new] * B, forced_tokens=forced)
        res.append(out)
        if forced is None:
            forced = torch.as_tensor(out["tokens"].astype(np.int32)).cuda()
        eng.free()
    a, c = res
    assert np.array_equal(a["tokens"], c["tokens"]) and np.array_equal(a["owner"], c["owner"]) and 0.2 < a["owner"].mean() < 0.8
    assert c["stats"]["kv_bytes_shared_reads"] > 0.3 * c["stats"]["kv_bytes_read"]
    err = {0: [], 2: []}
    for b in (0, 3, 8, 13):                                 # two members of each group
        z = replay_owner_logits(models, prompts[b], a["tokens"][b], a["owner"][b])
        for t in range(n_new):
            if a["owner"][b, t] == 0:
                ref = log_softmax(z[t])[int(a["tokens"][b, t])]
                err[0].append(abs(float(a["sen_logp"][b, t]) - ref)); err[2].append(abs(float(c["sen_logp"][b, t]) - ref))
    e0, e2 = np.array(err[0]), np.array(err[2])
    print("4B width, 1 layer, vs float64 oracle over %d senior positions: no sharing max %.4f mean %.4f; shared-prefix runs max %.4f mean %.4f; shared reads %.0f%% of the KV bytes"
          % (e0.size, e0.max(), e0.mean(), e2.max(), e2.mean(), 100.0 * c["stats"]["kv_bytes_shared_reads"] / c["stats"]["kv_bytes_read"]))
    # measured on B200: no sharing max 0.0201 / mean 0.0059, shared-prefix runs max 0.0191 / mean 0.0056, 69% of the KV bytes read shared
    assert e0.max() <= 0.04 and e0.mean() <= 0.012          # the bars of tests/test_gpu_full_width.py for one layer
    assert e2.max() <= 0.04 and e2.mean() <= 0.012 and e2.mean() <= 1.3 * e0.mean() + 1e-3

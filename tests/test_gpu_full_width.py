"""-m gpu: parity where the metric is quoted (BASELINE.json north_star, "the tests that guard the kernels").

The 36-layer slice of tests/test_gpu_bf16_slice.py reports what BASELINE.json asks for, but 36 layers of bf16 rounding on flat
random-init logits amplify one flipped rounding into ~0.05 nats, so its bars cannot see a kernel error of 0.03 nats. These tests
are sharp instead:
  * shallow at full width - 1 and 2 layers of the 4B shape (hidden 2560, 32 q / 8 kv heads of 128, intermediate 9728, vocabulary
    151,936: every kernel instantiation and tile shape of cfg 3, no deep amplification), 2 sequences x 64 tokens, senior log-probs
    against the float64 oracle inside BASELINE.json's 0.05 nats and against the rounding-point-faithful oracle (DESIGN.md R-V,
    `round_bf16` + `round_qp`), plus the relative L2 error of the whole logit vector at every position; 1 layer vs 2 layers
    localises an error to a layer's kernels;
  * long contexts - prompts of 2,450 / 4,383 / 8,703 ids (the bench's context, cfg 4's mid range and its last position) on
    scattered, high-numbered KV pages of a pool of tens of GB, so that RoPE table rows, tensor-map row indices and 640-position KV
    chunks are checked numerically where the benchmark runs; catch-ups of tens of tokens; senior log-probs within 0.007;
  * tandem_score in its benchmarked launch configuration (row budget >= 1024: row chunks dealt to CTAs, no K-splits, CTA pairs)
    against oracle.dual_score.
Every bar is at most twice what the test measured on B200 when it was written (the measured values stand beside the bars).
"""
import numpy as np
import pytest
import torch

import paper_2606_28166_b200 as T
from oracle import OracleModel, TandemParams as OParams, owners_from_tokens, replay_owner_logits, dual_score
from oracle.rule import Uniforms
from oracle.sampler import log_softmax
from workloads import ModelShape, make_weights, make_word_start, get_workload

pytestmark = pytest.mark.gpu
FOURB = get_workload("cfg3_4b_bf16").shape


def _cpu(w):
    return dict(embed=w["embed"].cpu(), lm_head=w["lm_head"].cpu(), final_norm=w["final_norm"].cpu(),
                layers=[{k: v.cpu() for k, v in l.items()} for l in w["layers"]])


def _senior_dlogp(models, prompts, g, n_new):
    """max / mean |senior log-prob - oracle| over the senior-emitted positions, and the raw top-1 agreement where `argmax` is given."""
    d = []
    for b in range(len(prompts)):
        z = replay_owner_logits(models, prompts[b], g["tokens"][b][:n_new], g["owner"][b][:n_new])
        for t in range(n_new):
            if g["owner"][b][t] == 0:
                d.append(abs(float(g["sen_logp"][b][t]) - log_softmax(z[t])[int(g["tokens"][b][t])]))
    return float(np.max(d)), float(np.mean(d)), len(d)


@pytest.mark.parametrize("n_layers", [1, 2])
def test_shallow_full_width_slice(n_layers):
    """Matching the rounding points removes only the noise of the points
    before the first P.V product (the tiled online softmax rounds P relative to its running maximum, which no plain definition
    reproduces bit for bit), so the faithful oracle is ~30% closer, not 10x; what makes this test sharp is (i) the mean over all
    senior positions and (ii) the relative L2 error of the WHOLE logit vector (151,936 entries) at every position: bf16 noise
    gives 0.6-1.0% on these flat random-init logits, a kernel that drops, permutes or mis-scales anything gives far more."""
    shape = ModelShape(n_layers, FOURB.hidden, FOURB.n_q_heads, FOURB.n_kv_heads, FOURB.head_dim, FOURB.intermediate, FOURB.vocab,
                       FOURB.rms_eps, FOURB.rope_theta, "bf16")
    ws = make_weights(shape, 1, device="cuda", gain_jitter=0.1); wj = make_weights(shape, 2, device="cuda", gain_jitter=0.1)
    table = make_word_start(shape.vocab, 0.30, 3)
    rng = np.random.default_rng(12)
    prompts = [rng.integers(0, shape.vocab, size=n).astype(np.int32) for n in (37, 52)]
    B, n_new, seed = 2, 64, 4242
    eng = T.Tandem(T.TandemConfig(shape, max_seqs=B, max_seq_len=128))
    eng.load_weights(0, ws); eng.load_weights(1, wj)
    prm = T.TandemParams(table, p=0.5, temperature=1.0, seed=seed)
    o = dict(token=torch.zeros(B, dtype=torch.int32, device="cuda"), owner=torch.zeros(B, dtype=torch.uint8, device="cuda"),
             sen_logp=torch.zeros(B, device="cuda"))
    dbg = torch.zeros(B, shape.vocab, device="cuda")
    toks = np.zeros((B, n_new), np.int64); own = np.zeros((B, n_new), np.uint8); lp = np.zeros((B, n_new)); zg = np.zeros((B, n_new, shape.vocab), np.float32)
    for t in range(n_new):
        eng.step(prm, admit=(prompts, None, [n_new] * B) if t == 0 else None, out=o, dbg_logits=dbg)
        torch.cuda.synchronize()
        toks[:, t] = o["token"].cpu().numpy(); own[:, t] = o["owner"].cpu().numpy(); lp[:, t] = o["sen_logp"].cpu().numpy()
        zg[:, t] = dbg.cpu().numpy()
    eng.free()
    ws_c, wj_c = _cpu(ws), _cpu(wj)
    del ws, wj
    torch.cuda.empty_cache()
    assert (toks >= 0).all() and 0.1 < own.mean() < 0.9
    for b in range(B):   # ownership is an integer function of (tokens, uniforms, table, rule): bit-exact
        assert np.array_equal(owners_from_tokens(toks[b], table, OParams(p=0.5, seed=seed), Uniforms(seed=seed), b=b), own[b])
    res = {}
    for mode, kw in (("fp64", {}), ("faithful", dict(round_bf16=True, round_qp=True))):
        models = (OracleModel(shape, ws_c, cache=False, **kw), OracleModel(shape, wj_c, cache=False, **kw))
        d, rel, top1 = [], [], []
        for b in range(B):
            z = replay_owner_logits(models, prompts[b], toks[b], own[b])
            for t in range(n_new):
                if own[b, t] == 0:
                    d.append(abs(lp[b, t] - log_softmax(z[t])[toks[b, t]]))
                rel.append(np.linalg.norm(zg[b, t] - z[t]) / np.linalg.norm(z[t]))
                top1.append(int(np.argmax(z[t])) == int(np.argmax(zg[b, t])))
        res[mode] = dict(max_dlogp=float(np.max(d)), mean_dlogp=float(np.mean(d)), n_senior=len(d), max_rel_l2=float(np.max(rel)),
                         mean_rel_l2=float(np.mean(rel)), top1=float(np.mean(top1)))
    print("shallow full width, %d layer(s): %s" % (n_layers, res))
    f, s = res["fp64"], res["faithful"]
    # measured (1 / 2 layers): fp64 max 0.0199 / 0.0219, mean 0.0060 / 0.0070, rel L2 0.0079 / 0.0100; faithful max 0.0135 / 0.0171,
    # mean 0.0042 / 0.0051, rel L2 0.0061 / 0.0078; raw top-1 98% (margins of ~1e-3 on flat logits)
    assert f["max_dlogp"] <= 0.04 and f["mean_dlogp"] <= 0.012, f     # inside BASELINE.json's 0.05
    assert s["max_dlogp"] <= 0.03 and s["mean_dlogp"] <= 0.009, s
    assert f["max_rel_l2"] <= 0.016 and s["max_rel_l2"] <= 0.013, (f, s)
    assert f["top1"] >= 0.95


def test_long_context_scattered_pages():
    shape = ModelShape(2, 256, 4, 1, 128, 512, 4096, 1e-6, 1e6, "bf16")       # d = 128, G = 4: cfg 3's attention instantiation
    lens = [2450, 4383, 8703]
    rng = np.random.default_rng(31)
    prompts = [rng.integers(0, shape.vocab, size=n).astype(np.int32) for n in lens]
    table = make_word_start(shape.vocab, 0.05, 3)                              # runs of ~40 tokens per owner: catch-ups of tens of tokens
    ws = make_weights(shape, 1, gain_jitter=0.1); wj = make_weights(shape, 2, gain_jitter=0.1)
    n_new, seed = 48, 77
    free, _ = torch.cuda.mem_get_info()
    kv = int(min(48e9, (free - 8e9) / 2))                                      # tens of GB per model: page ids up to ~1.5 million
    eng = T.Tandem(T.TandemConfig(shape, max_seqs=3, max_seq_len=8768, kv_bytes_per_model=kv, max_rows_per_step=4096, use_graph=1))
    eng.load_weights(0, ws); eng.load_weights(1, wj)
    eng.set_page_order(2026)                                                   # scattered, high-numbered pages from the first one on
    g = eng.generate(T.TandemParams(table, p=0.5, temperature=1.0, seed=seed), prompts, [n_new] * 3)
    st = g["stats"]
    eng.free()
    assert (g["len"] == n_new).all() and 0.05 < g["owner"].mean() < 0.95
    runs = [np.diff(np.flatnonzero(np.diff(np.concatenate([[-1], g["owner"][b], [-1]])) != 0)).max() for b in range(3)]
    assert max(runs) > 16, runs                                                # at least one catch-up longer than a page
    assert st["catchup_rows"] > sum(lens)                                      # the junior ingested the prompts when it first took over
    for b in range(3):
        assert np.array_equal(owners_from_tokens(g["tokens"][b], table, OParams(p=0.5, seed=seed), Uniforms(seed=seed), b=b), g["owner"][b])
    models = (OracleModel(shape, ws), OracleModel(shape, wj))
    mx, mean, n = _senior_dlogp(models, prompts, g, n_new)
    print("long context (2450 / 4383 / 8703, scattered pages of a %.0f GB pool): max %.5f mean %.5f (n=%d)" % (kv / 1e9, mx, mean, n))
    assert mx <= 0.007 and mean <= 0.002, (mx, mean)                           # measured 0.0036 / 0.00096


def _score_check(out, refs, tol_lp, tol_alpha):
    worst = [0.0, 0.0, 0.0]
    for b, ref in enumerate(refs):
        for k, name in enumerate(("sen_logp", "jun_logp", "overlap")):
            assert out[name][b].shape == ref[name].shape and out[name][b][0] == 0.0
            worst[k] = max(worst[k], float(np.max(np.abs(out[name][b] - ref[name]))))
    assert worst[0] <= tol_lp and worst[1] <= tol_lp and worst[2] <= tol_alpha, worst
    return worst


def test_score_benchmarked_configuration_small_model():
    """Row budget 1024 with > 768 live rows per step: four row chunks per weight tile on different CTAs, no K-splits, CTA pairs."""
    shape = ModelShape(2, 256, 4, 1, 128, 512, 4096, 1e-6, 1e6, "bf16")
    rng = np.random.default_rng(41)
    streams = [rng.integers(0, shape.vocab, size=n).astype(np.int32) for n in (700, 333, 650, 17, 1200)]
    ws = make_weights(shape, 1, gain_jitter=0.1); wj = make_weights(shape, 2, gain_jitter=0.1)
    eng = T.Tandem(T.TandemConfig(shape, max_seqs=4, max_seq_len=1216, max_rows_per_step=1024))
    eng.load_weights(0, ws); eng.load_weights(1, wj)
    out = eng.score(streams)
    eng.free()
    assert out["stats"]["rows_senior"] == out["stats"]["rows_junior"] == sum(len(s) - 1 for s in streams)
    assert out["stats"]["steps"] <= 4                                           # ~2,900 rows in steps of up to 1,024
    models = (OracleModel(shape, ws), OracleModel(shape, wj))
    worst = _score_check(out, [dual_score(models, s) for s in streams], 0.01, 2e-4)   # measured 0.0054 / 1.0e-4 over 2,900 positions
    print("tandem_score, row budget 1024, small model: worst |dlogp| sen %.5f jun %.5f, |dalpha| %.5f" % tuple(worst))


def test_score_benchmarked_configuration_full_width():
    """The same launch configuration on two layers of the 4B shape (the projection shapes of cfg 3, vocabulary 151,936)."""
    shape = ModelShape(2, FOURB.hidden, FOURB.n_q_heads, FOURB.n_kv_heads, FOURB.head_dim, FOURB.intermediate, FOURB.vocab,
                       FOURB.rms_eps, FOURB.rope_theta, "bf16")
    rng = np.random.default_rng(43)
    streams = [rng.integers(0, shape.vocab, size=n).astype(np.int32) for n in (301, 290, 310)]      # 898 rows in one step
    ws = make_weights(shape, 1, device="cuda", gain_jitter=0.1); wj = make_weights(shape, 2, device="cuda", gain_jitter=0.1)
    eng = T.Tandem(T.TandemConfig(shape, max_seqs=3, max_seq_len=320, max_rows_per_step=1024))
    eng.load_weights(0, ws); eng.load_weights(1, wj)
    out = eng.score(streams)
    eng.free()
    ws_c, wj_c = _cpu(ws), _cpu(wj)
    del ws, wj
    torch.cuda.empty_cache()
    assert out["stats"]["steps"] == 1
    models = (OracleModel(shape, ws_c, cache=False), OracleModel(shape, wj_c, cache=False))
    worst = _score_check(out, [dual_score(models, s) for s in streams], 0.05, 2e-4)   # measured 0.036 (max over 1,796 log-probs) / 1.0e-4
    print("tandem_score, row budget 1024, 2 layers at full width: worst |dlogp| sen %.5f jun %.5f, |dalpha| %.5f" % tuple(worst))

#!/usr/bin/env python
"""bench.py - tandem rollout throughput on B200 (BASELINE.json metric: "tandem rollout tokens/s (4B-shape bf16, 1 B200)").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME] [--fast-forward G]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P bench.py --gpus N ...

One "step" = one pass of the whole hot path (S0-S8) over the resident batch: every unfinished
sequence of the workload emits exactly one token (`tandem_step`). The workload is BASELINE.json configs[2]
(cfg3_4b_bf16: two 36-layer 4B-shape models, batch 128 = 16 prompts x 8 rollouts, prompts U[64,512], p = 0.5,
T = 1, 16-token KV pages), synthetic and seeded (workloads/). Phases of the default arm:
  setup   (untimed) weights -> engine, admission, prompt prefill, `--ramp` steps so that both models hold KV
  warmup  W steps (>= 3 enforced)
  timed   exactly K steps between CUDA events on the launching stream; barrier + synchronize on both sides; max over ranks
  profile `--profile-steps` more steps in the library's per-kernel timing mode -> "roofline" of the dominant kernel
  e2e     `tandem_generate` on HOST buffers (prompts H2D, tokens/owner/log-probs D2H inside the timed region)
  cpu     the oracle (oracle/, float64 NumPy) on a bounded sample of the same workload, rank 0, N = 1 only
`--impl reference` times the oracle alone (rank 0; other ranks exit 0) and prints the same JSON line shape.
Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "tandem rollout tokens/s (4B-shape bf16, 1 B200)"
NOMINAL_HBM_GBS = 8000.0            # BASELINE.json: "decode HBM GB/s vs 8 TB/s"
FALLBACK_HBM_GBS = 6650.0           # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
FALLBACK_BF16_TFLOPS = 1590.0


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=128)
    ap.add_argument("--warmup", type=int, default=8)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3_4b_bf16")
    ap.add_argument("--p", type=float, default=None, help="override the workload's switch probability (cfg5 sweep)")
    ap.add_argument("--switch-mode", default=None, choices=["TOGGLE", "REDRAW"], help="override the workload's meaning of p (cfg5: REDRAW p = 1 is solo senior decoding too)")
    ap.add_argument("--grpo", action="store_true", help="time tandem_grpo_objective (senior-masked GRPO forward, NEXT-3) on the workload's batch x max_new")
    ap.add_argument("--score", type=int, default=0, help="N > 0: time tandem_score (teacher-forced dual scoring, NEXT-1) on N synthetic streams instead of the rollout")
    ap.add_argument("--score-len", type=int, default=2048, help="tokens per stream for --score")
    ap.add_argument("--dual-forward", action="store_true",
                    help="measurement: the paper's lock-step engine (both models forward every token, no catch-up prefill) instead of the owner split")
    ap.add_argument("--max-rows", type=int, default=0,
                    help="tandem_config.max_rows_per_step: row budget of a step per model (prefills and catch-ups beyond it are chunked). 0 = 4096, except 256 for a "
                         "whole rollout with >= 256 resident sequences (cfg 4): the projections pass over the weights once per 256 token rows, and with ~256 rows "
                         "per model and step a budget of 256 keeps every step at one pass (160.1 -> 151.1 s measured)")
    ap.add_argument("--set-option", action="append", default=[], metavar="NAME=VALUE",
                    help="measurement: a tandem_test_set_option knob (include/tandem_test.h) for an A/B on one box, e.g. gateup_cluster=0; repeatable")
    ap.add_argument("--skip-class", default=None,
                    help="measurement: leave the launches of one kernel class (a name of the kernels table, e.g. gemm_gateup) out of the timed steps; the "
                         "difference to the full step is the class's marginal cost inside the step graph (results of those steps are garbage)")
    ap.add_argument("--attn-prefill-tc", type=int, default=1, help="--score: 0 = attention on the mma.sync kernel of the rollout instead of the tcgen05 kernel (A/B)")
    ap.add_argument("--score-rows", type=int, default=2048, help="rows per step and model for --score (max_rows_per_step)")
    ap.add_argument("--top-k", type=int, default=0, help="top-k filter of the sampler (0 = off; the paper evaluates with 20)")
    ap.add_argument("--temperature", type=float, default=None, help="override the workload's sampling temperature")
    ap.add_argument("--top-p", type=float, default=None, help="override the workload's top-p (the paper trains at 1.0, evaluates at 0.8)")
    ap.add_argument("--word-start-frac", type=float, default=None, help="override the word-start table density (cfg5 sweep)")
    ap.add_argument("--fast-forward", type=int, default=-1,
                    help="tokens already generated per sequence before the timed window (ingested as context by prefill); "
                         "-1 = half of the workload's max_new: step time is affine in the context length, so a step at the "
                         "rollout's midpoint costs what the whole rollout costs on average")
    ap.add_argument("--ramp", type=int, default=48, help="untimed steps after prefill so that both models own KV")
    ap.add_argument("--max-drain", type=int, default=256, help="upper bound on the extra untimed steps that drain the first catch-ups")
    ap.add_argument("--profile-steps", type=int, default=4)
    ap.add_argument("--e2e-new", type=int, default=64, help="new tokens per sequence in the SHORT end-to-end tandem_generate leg (e2e_short)")
    ap.add_argument("--no-e2e-full", action="store_true",
                    help="skip the whole-workload tandem_generate call (e2e: every sequence to its max_new, ~50 s for cfg 3); e2e then falls back to the short leg")
    ap.add_argument("--profiler-range", action="store_true",
                    help="cudaProfilerStart/Stop around the timed region (for `ncu --profile-from-start off`)")
    ap.add_argument("--full-rollout", type=float, default=0.0, metavar="SCALE",
                    help="instead of timed steps: run the WHOLE workload through tandem_generate (host buffers, admission queue) with "
                         "every max_new multiplied by SCALE (1.0 = the workload as specified) and report tokens/s of the call")
    ap.add_argument("--catchup-share", action="store_true",
                    help="BASELINE.json configs[4]: also report the catch-up-prefill share of STEP TIME - attention over the catch-up items "
                         "(q_len > 1) timed by a second, filtered launch in the per-kernel pass, the row-proportional kernels apportioned by rows")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-share-prompt-pages", action="store_true",
                    help="every rollout computes and stores its own copy of the prompt's KV (default: the G rollouts of a prompt share its full pages)")
    ap.add_argument("--share-mode", type=int, default=2, choices=[1, 2],
                    help="tandem_config.share_prompt_pages when sharing is on: 1 = the rollouts of a prompt share its full KV pages; 2 = and the members a model "
                         "serves in a step read them once (shared-prefix runs)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-new", type=int, default=8, help="new tokens of the oracle's bounded sample")
    return ap.parse_args()


def code_state():
    """sha256 over the sources of the dominant kernel (the paged attention kernel and what it includes): `roofline.traffic` is an
    ncu measurement stored beside this hash (profiles/traffic_r2.json) and is reported only while the hash still matches."""
    import hashlib
    h = hashlib.sha256()
    for f in ("attention_mma.cuh", "common.cuh"):
        h.update(open(os.path.join(ROOT, "paper_2606_28166_b200", "csrc", f), "rb").read())
    return h.hexdigest()[:16]


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm_gbs=float(p["hbm_gbs"]), bf16_tflops=float(p["bf16_tflops"]),
                    bf16_tflops_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])), source="measured")
    return dict(hbm_gbs=FALLBACK_HBM_GBS, bf16_tflops=FALLBACK_BF16_TFLOPS, bf16_tflops_sustained=1400.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md's clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------ workload
def build_inputs(wl, fast_forward, rank):
    """Seeded synthetic inputs of the workload for this rank: prompts (+ `fast_forward` already-generated ids appended
    as context), the word-start table and the per-sequence ids that address the counter RNG."""
    from workloads import make_prompts, make_word_start
    prompts = make_prompts(wl, seed=wl.seeds["prompts"] + 1000 * rank)
    if fast_forward > 0:
        rng = np.random.default_rng(wl.seeds["prompts"] + 1000 * rank + 77)
        prompts = [np.concatenate([p, rng.integers(0, wl.shape.vocab, size=fast_forward).astype(np.int32)]) for p in prompts]
    table = make_word_start(wl.shape.vocab, wl.word_start_frac, wl.seeds["table"])
    seq_ids = np.arange(wl.batch, dtype=np.int32) + wl.batch * rank
    return prompts, table, seq_ids


def reduce_over_ranks(dist, seconds_or_ms, tokens, device):
    """Whole-job aggregation of one timed region: (max over ranks of the time, sum over ranks of the units). Works on any
    backend (nccl on the GPUs, gloo in the CPU test); without a process group it is the identity."""
    if dist is None:
        return float(seconds_or_ms), float(tokens)
    import torch
    t = torch.tensor([float(seconds_or_ms), float(tokens)], dtype=torch.float64, device=device)
    tmax = t.clone(); dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    tsum = t.clone(); dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
    return float(tmax[0]), float(tsum[1])


def weight_bytes_per_model(shape):
    return shape.params_read_per_step * (4 if shape.dtype == "f32" else 2)


def class_bytes(shape, cls, rows, kv_bytes_per_layer_launch, emit_rows, n_models=2):
    """ALGORITHMIC HBM bytes of one launch of kernel class `cls`. Every launch serves `n_models` models:
    `rows`, `emit_rows` and the KV bytes are the totals over those models; weights are streamed once per model. Counted: the
    operand that must be streamed (weights / KV) + activations in + one copy of the result. bf16 = 2 bytes, fp32 = 4."""
    H, I, V = shape.hidden, shape.intermediate, shape.vocab
    qd, kd = shape.n_q_heads * shape.head_dim, shape.n_kv_heads * shape.head_dim
    es = 4 if shape.dtype == "f32" else 2
    g = lambda N, K, r: n_models * N * K * es + r * K * es + r * N * 4
    if cls == "gemm_qkv":
        return g(qd + 2 * kd, H, rows)
    if cls == "gemm_o":
        return g(H, qd, rows)
    if cls == "gemm_gateup":
        return g(2 * I, H, rows)
    if cls == "gemm_down":
        return g(H, I, rows)
    if cls == "gemm_lmhead":   # fused S8: the output is one 32-byte partial per (128-id tile, row), not fp32 logits
        return n_models * V * H * es + emit_rows * H * es + emit_rows * ((V + 127) // 128) * 32
    if cls == "attention":
        return kv_bytes_per_layer_launch + rows * qd * (4 + es)
    if cls == "rope_append":
        return rows * (qd + 2 * kd) * 4 + rows * qd * 4 + rows * 2 * kd * es
    if cls == "residual_norm":
        return rows * H * (4 + 4 + 4 + es)
    if cls == "swiglu":
        return rows * 2 * I * 4 + rows * I * es
    if cls == "embed_norm":
        return rows * H * (es + 4 + es)
    if cls == "sample_switch_emit":   # fused S8: the merge reads the partials
        return emit_rows * ((V + 127) // 128) * 32
    return 0


def run_full_rollout(args):
    """The whole workload through one tandem_generate call: prompts in, tokens / owner flags / senior log-probs out, sequences
    admitted as KV pages allow (cfg 4 does not fit at once). Sanity checks here use no oracle code (the parity tests do that): every
    sequence reaches its length and an owner change only ever follows a word-start token."""
    import torch
    import paper_2606_28166_b200 as T
    from workloads import get_workload, make_weights, make_word_start, make_prompts, make_max_new
    torch.cuda.set_device(0)
    T.build()
    wl = get_workload(args.workload)
    shape = wl.shape
    prompts = make_prompts(wl)
    max_new = np.maximum(1, (make_max_new(wl) * args.full_rollout).astype(np.int32))
    B = len(prompts)
    table = make_word_start(shape.vocab, wl.word_start_frac, wl.seeds["table"])
    # weights are drawn on the GPU, parked on the host and loaded from there, so that no staging copy competes with the KV pools
    to_cpu = lambda w: dict(embed=w["embed"].cpu(), lm_head=w["lm_head"].cpu(), final_norm=w["final_norm"].cpu(),
                            layers=[{k: v.cpu() for k, v in l.items()} for l in w["layers"]])
    w_host = []
    for seed in (wl.seeds["senior"], wl.seeds["junior"]):
        w = make_weights(shape, seed, device="cuda"); w_host.append(to_cpu(w)); del w; torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    wbytes = 2 * (shape.params_read_per_step + shape.vocab * shape.hidden) * 2      # both models, embedding included
    need = sum((len(p) + int(n) + 15) // 16 + 1 for p, n in zip(prompts, max_new)) * shape.kv_elems_per_token * 2 * 16
    kv_per_model = int(min((free - wbytes - 4.5e9) / 2, need + (64 << 20)))            # workspaces and the CUDA context stay free
    max_seqs = min(B, 256)
    max_rows = args.max_rows or (256 if max_seqs >= 256 else 4096)
    eng = T.Tandem(T.TandemConfig(shape, max_seqs=max_seqs, max_seq_len=(max(len(p) for p in prompts) + int(max_new.max()) + 31) // 16 * 16,
                                  kv_bytes_per_model=kv_per_model, max_rows_per_step=max_rows, use_graph=1,
                                  share_prompt_pages=0 if args.no_share_prompt_pages else args.share_mode))
    for m in range(2):
        eng.load_weights(m, w_host[m])
    del w_host
    seed = 20260628
    prm = T.TandemParams(table, p=wl.p, switch_mode=wl.switch_mode, temperature=wl.temperature, top_p=wl.top_p, top_k=args.top_k or wl.top_k, seed=seed)
    t0 = time.perf_counter()
    g = eng.generate(prm, prompts, max_new)
    dt = time.perf_counter() - t0
    assert (g["len"] == max_new).all()
    for b in range(B):                                   # TOGGLE / REDRAW without cap: the author changes only after a word-start token
        n = int(g["len"][b])
        flips = g["owner"][b, 1:n] != g["owner"][b, :n - 1]
        assert not flips[table[g["tokens"][b, :n - 1]] == 0].any(), "an owner change follows a token that starts no word"
    st = g["stats"]
    tok = int(g["len"].sum())
    pk = peaks()
    gbs = (st["kv_bytes_read"] + st["weight_bytes_read"]) / dt / 1e9
    print(json.dumps({"metric": METRIC, "value": tok / dt, "unit": "tokens/s", "n_gpus": 1, "steps": int(st["steps"]), "warmup": 0,
                      "ms_per_step": dt / max(1, st["steps"]) * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
                      "data": "synthetic",
                      "config": {"workload": wl.name, "mode": "full rollout through tandem_generate (prefill, admission queue, host buffers)",
                                 "sequences": B, "max_new_scale": args.full_rollout, "mean_new": float(max_new.mean()), "tokens": tok, "seconds": dt,
                                 "max_seqs": max_seqs, "max_rows_per_step": max_rows, "peak_resident": int(st["peak_resident"]), "kv_gb_per_model": kv_per_model / 1e9,
                                 "peak_pages": [int(st["peak_pages_senior"]), int(st["peak_pages_junior"])],
                                 "share_prompt_pages": 0 if args.no_share_prompt_pages else args.share_mode, "shared_prompt_rows": int(st["shared_prompt_rows"]),
                                 "kv_bytes_shared_reads": int(st["kv_bytes_shared_reads"]), "kv_bytes_read": int(st["kv_bytes_read"]),
                                 "senior_share": float(g["mask"].sum() / max(1, tok))},
                      "gpu_launches": int(st["kernel_launches"]),
                      "step_roofline": {"bound": "hbm", "achieved": gbs, "unit": "GB/s", "frac_of_measured": gbs / pk["hbm_gbs"], "frac_of_8TBs": gbs / NOMINAL_HBM_GBS},
                      "e2e": {"value": tok / dt, "unit": "tokens/s", "h2d_bytes_per_step": sum(len(p) for p in prompts) * 4 / max(1, st["steps"]),
                              "d2h_bytes_per_step": tok * 9 / max(1, st["steps"])}}))
    eng.free()


def run_grpo(args):
    """tandem_grpo_objective on device buffers of the workload's rollout shape (B = prompts x G rollouts, L = max_new): advantages,
    clipped senior-masked surrogate, loss. HBM-bound element-wise work: bytes = B L (owner 1 + two log-probs 8 [+ 4 token output])."""
    import torch
    import paper_2606_28166_b200 as T
    from workloads import get_workload
    torch.cuda.set_device(0)
    T.build()
    wl = get_workload(args.workload)
    B, L, G = wl.batch, wl.max_new, wl.group
    g = torch.Generator(device="cuda"); g.manual_seed(1)
    rewards = (torch.rand(B, device="cuda", generator=g) < 0.4).float()
    lengths = torch.randint(L // 2, L + 1, (B,), device="cuda", generator=g, dtype=torch.int32)
    owner = (torch.rand(B, L, device="cuda", generator=g) < 0.5).to(torch.uint8)
    old = -3 * torch.rand(B, L, device="cuda", generator=g)
    new = old + 0.1 * torch.randn(B, L, device="cuda", generator=g)
    out = {}
    for want_tokens in (False, True):
        for _ in range(5):
            r = T.grpo_objective(rewards, G, lengths, owner, new, old, want_tokens=want_tokens)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n = max(20, args.steps)
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
        res = torch.empty(8, device="cuda")
        tot = 0.0
        for _ in range(n):
            flush.zero_()                                # inputs (4.7 MB) would otherwise sit in L2
            e0.record()
            lib_rc = T.binding.lib().tandem_grpo_objective(B // G, G, L, rewards.data_ptr(), lengths.data_ptr(), owner.data_ptr(), new.data_ptr(),
                                                           old.data_ptr(), None, 0.2, 0.0, 1e-6, r["advantages"].data_ptr(),
                                                           r["token_obj"].data_ptr() if want_tokens else None, r["seq_obj"].data_ptr(),
                                                           res.data_ptr(), None)
            e1.record(); torch.cuda.synchronize()
            assert lib_rc == 0
            tot += e0.elapsed_time(e1)
        us = tot / n * 1e3
        byt = B * L * (9 + (4 if want_tokens else 0))
        out["with_token_obj" if want_tokens else "scalars_only"] = {"us_per_call": us, "alg_bytes": byt, "gbs": byt / us / 1e3}
    pk = peaks()
    best = out["scalars_only"]
    print(json.dumps({"metric": "senior-masked GRPO objective, forward (rollout tokens/s consumed)", "value": B * L / (best["us_per_call"] * 1e-6),
                      "unit": "tokens/s", "n_gpus": 1, "steps": max(20, args.steps), "warmup": 5, "ms_per_step": best["us_per_call"] * 1e-3,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": wl.name, "mode": "tandem_grpo_objective", "rollouts": B, "group": G, "stride": L, "l2": "flushed between calls"},
                      "gpu_launches": 1, "variants": out,
                      "roofline": {"bound": "hbm", "achieved": best["gbs"], "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": best["gbs"] / pk["hbm_gbs"],
                                   "traffic": None, "note": "one memset and one kernel of a few microseconds: launch latency and the tail of 128 CTAs, not bandwidth, set the time at this size"},
                      "loss": r["loss"], "clip_frac": r["clip_frac"]}))


def run_score(args):
    """tandem_score on N streams of the workload's shape (host buffers in and out): both models read every stream through the
    ragged prefill path, every position reaches the LM head, and the score kernel reduces the two logit rows to (log p_sen(y),
    log p_jun(y), alpha). Parity with oracle.dual_score is the job of tests/test_gpu_score.py; here only ranges are checked."""
    import torch
    import paper_2606_28166_b200 as T
    from workloads import get_workload, make_weights
    torch.cuda.set_device(0)
    T.build()
    wl = get_workload(args.workload)
    shape = wl.shape
    N, L = args.score, args.score_len
    rng = np.random.default_rng(wl.seeds["prompts"] if "prompts" in wl.seeds else 1)
    streams = [rng.integers(0, shape.vocab, size=L).astype(np.int32) for _ in range(N)]
    max_seqs = min(N, 64)
    kv = (max_seqs + 1) * ((L + 15) // 16 + 1) * shape.kv_elems_per_token * 2 * 16
    eng = T.Tandem(T.TandemConfig(shape, max_seqs=max_seqs, max_seq_len=(L + 15) // 16 * 16, kv_bytes_per_model=kv, max_rows_per_step=args.score_rows))
    for m, seed in enumerate((wl.seeds["senior"], wl.seeds["junior"])):
        w = make_weights(shape, seed, device="cuda"); eng.load_weights(m, w); del w; torch.cuda.empty_cache()
    if not args.attn_prefill_tc:
        eng.set_option("attn_prefill_tc", 0)
    eng.score(streams[:min(N, 2)])                       # warm-up: buffers, tensor maps
    t0 = time.perf_counter()
    out = eng.score(streams)
    dt = time.perf_counter() - t0
    eng.set_profile(True)                                # a second pass with one event pair per kernel launch: where the time goes
    eng.score(streams[:min(N, 8)])
    prof = eng.get_profile()
    eng.set_profile(False)
    tot = sum(ms for ms, n in prof.values()) or 1.0
    kernels = {k: {"ms_per_launch": ms / n, "launches": n, "share": ms / tot} for k, (ms, n) in prof.items() if n}
    st = out["stats"]
    tok = N * (L - 1)
    alpha = float(np.mean(np.concatenate([o[1:] for o in out["overlap"]])))
    ce = float(-np.mean(np.concatenate([o[1:] for o in out["jun_logp"]])))
    assert 0.0 < alpha <= 1.0 + 1e-5 and np.isfinite(ce)
    pk = peaks()
    flops = 2.0 * 2 * (shape.params_read_per_step + shape.vocab * shape.hidden) * tok     # both models, projections and LM head (attention extra)
    wbytes = float(st["weight_bytes_read"])
    print(json.dumps({"metric": "dual-scored tokens/s (teacher-forced, both models, 1 B200)", "value": tok / dt, "unit": "tokens/s", "n_gpus": 1,
                      "steps": int(st["steps"]), "warmup": 1, "ms_per_step": dt / max(1, st["steps"]) * 1e3, "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                      "config": {"workload": wl.name, "mode": "tandem_score (host buffers)", "streams": N, "tokens_per_stream": L,
                                 "rows_per_step_and_model": args.score_rows, "attention": "tcgen05" if args.attn_prefill_tc else "mma.sync", "seconds": dt, "mean_alpha": alpha, "junior_cross_entropy": ce},
                      "gpu_launches": int(st["kernel_launches"]), "kernels": kernels,
                      "step_roofline": {"tensor_tflops": flops / dt / 1e12, "tensor_peak": pk.get("bf16_tflops_sustained", pk.get("bf16_tflops")),
                                        "weights_gbs": wbytes / dt / 1e9, "hbm_peak": pk["hbm_gbs"]},
                      "e2e": {"value": tok / dt, "unit": "tokens/s", "h2d_bytes_per_step": N * L * 4 / max(1, st["steps"]),
                              "d2h_bytes_per_step": tok * 12 / max(1, st["steps"])}}))
    eng.free()


def run_ours(args):
    import torch
    import paper_2606_28166_b200 as T
    from workloads import get_workload, make_weights

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if local == 0:
        T.build()                     # one rank per node compiles (a stale pushed .so would otherwise be rebuilt by N ranks at once)
    if dist:
        dist.barrier()
    T.lib()
    wl = get_workload(args.workload)
    if args.p is not None:
        wl = wl.with_(p=args.p)
    if args.switch_mode is not None:
        wl = wl.with_(switch_mode=1 if args.switch_mode == "REDRAW" else 0)
    if args.word_start_frac is not None:
        wl = wl.with_(word_start_frac=args.word_start_frac)
    if args.top_p is not None:
        wl = wl.with_(top_p=args.top_p)
    if args.temperature is not None:
        wl = wl.with_(temperature=args.temperature)
    shape, B = wl.shape, wl.batch
    W, K = max(3, args.warmup), args.steps
    if args.fast_forward < 0:
        args.fast_forward = wl.max_new // 2
    prompts, table, seq_ids = build_inputs(wl, args.fast_forward, rank)
    max_prompt = max(len(p) for p in prompts)
    prefill_rows = sum(len(p) for p in prompts)
    row_cap = args.max_rows or 4096
    prefill_steps = (prefill_rows + row_cap - 1) // row_cap + 2
    gen_budget = prefill_steps + max(args.ramp, int(8.0 / max(wl.p * wl.word_start_frac, 1e-3))) + args.max_drain + W + K + args.profile_steps + 64
    e2e_len = args.e2e_new if (args.no_e2e or args.no_e2e_full) else max(args.e2e_new, wl.max_new)
    max_seq_len = ((max_prompt + max(gen_budget, e2e_len) + 15) // 16) * 16
    # weights are drawn on the GPU, parked on the host and loaded from there, so that no staging copy competes with the KV pools
    to_cpu = lambda w: dict(embed=w["embed"].cpu(), lm_head=w["lm_head"].cpu(), final_norm=w["final_norm"].cpu(),
                            layers=[{k: v.cpu() for k, v in l.items()} for l in w["layers"]])
    w_host = []
    for seed in (wl.seeds["senior"], wl.seeds["junior"]):
        w = make_weights(shape, seed, device="cuda"); w_host.append(to_cpu(w)); del w; torch.cuda.empty_cache()
    # KV pools: what the timed steps need and, for the e2e leg, the whole workload (every sequence at prompt + max_new), as far as
    # the device allows beside 2 x (layers + LM head + embedding) of weights and the workspaces; what does not fit queues in tandem_generate
    from workloads import make_max_new
    page_bytes = shape.kv_elems_per_token * 2 * 16
    need_pages = B * ((max_prompt + gen_budget + 15) // 16 + 1)
    if not (args.no_e2e or args.no_e2e_full):
        need_pages = max(need_pages, sum((len(p) + int(n) + 15) // 16 + 1 for p, n in zip(build_inputs(wl, 0, rank)[0], make_max_new(wl))))
    free, _ = torch.cuda.mem_get_info()
    wbytes = 2 * (shape.params_read_per_step + shape.vocab * shape.hidden) * 2
    kv_per_model = int(min((free - wbytes - 5.5e9) / 2, (need_pages + 64) * page_bytes))
    eng = T.Tandem(T.TandemConfig(shape, max_seqs=B, max_seq_len=max_seq_len, device=local, max_rows_per_step=row_cap, use_graph=1,
                                  kv_bytes_per_model=kv_per_model, share_prompt_pages=0 if args.no_share_prompt_pages else args.share_mode))
    for m in range(2):
        eng.load_weights(m, w_host[m])
    if args.dual_forward:
        eng.set_option("dual_forward", 1)
    for kv in args.set_option:
        eng.set_option(kv.split("=")[0], int(kv.split("=")[1]))
    w_cpu = w_host if (rank == 0 and world == 1 and not args.no_cpu) else []
    del w_host
    prm = T.TandemParams(table, p=wl.p, switch_mode=wl.switch_mode, temperature=wl.temperature, top_p=wl.top_p, top_k=args.top_k or wl.top_k, seed=20260628)
    out = dict(token=torch.zeros(B, dtype=torch.int32, device="cuda"), owner=torch.zeros(B, dtype=torch.uint8, device="cuda"),
               sen_logp=torch.zeros(B, device="cuda"), done=torch.zeros(B, dtype=torch.uint8, device="cuda"))
    stream = torch.cuda.current_stream().cuda_stream

    # ---- setup: admission, prompt prefill (row-capped chunks), ramp
    t0 = time.perf_counter()
    eng.step(prm, admit=(prompts, seq_ids, [gen_budget] * B), out=out, stream=stream)
    n_setup = 1
    while True:
        st = eng.get_stats()
        if st["tokens_emitted"] >= B or n_setup > 4 * prefill_steps + 16:
            break
        eng.step(prm, out=out, stream=stream); n_setup += 1
    # every sequence should have changed hands a few times before timing: ~8 expected switches per sequence (e^-8 of them none) (rate p * f per token)
    ramp = max(args.ramp, int(8.0 / (wl.p * wl.word_start_frac)) if wl.p * wl.word_start_frac > 0 else 0)
    for _ in range(ramp):
        eng.step(prm, out=out, stream=stream)
    # keep stepping until the partner's first catch-up over the (fast-forwarded) context has drained: steady state is
    # ~2 rows per sequence per step; the budget above reserves room for these steps
    n_drain, prev = 0, eng.get_stats()
    while n_drain < args.max_drain:
        for _ in range(8):
            eng.step(prm, out=out, stream=stream)
        n_drain += 8
        cur = eng.get_stats()
        rows8 = cur["rows_senior"] + cur["rows_junior"] - prev["rows_senior"] - prev["rows_junior"]
        prev = cur
        if rows8 <= 8 * 3 * B:
            break
    torch.cuda.synchronize()
    if args.skip_class:   # after the setup: the state the timed steps start from is the real one
        names = [T.lib().tandem_kernel_class_name(i).decode() for i in range(T.binding.KC_NUM)]
        eng.set_option("skip_class", names.index(args.skip_class))
    setup_s = time.perf_counter() - t0

    # ---- warmup + timed region
    for _ in range(W):
        eng.step(prm, out=out, stream=stream)
    torch.cuda.synchronize()
    s0 = eng.get_stats()
    if dist: dist.barrier()
    torch.cuda.synchronize()
    clocks = ClockSampler(local); clocks.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if args.profiler_range:
        torch.cuda.profiler.start()
    e0.record()
    for _ in range(K):
        eng.step(prm, out=out, stream=stream)
    e1.record()
    torch.cuda.synchronize()
    if args.profiler_range:
        torch.cuda.profiler.stop()
    if dist: dist.barrier()
    ms = e0.elapsed_time(e1)
    clk = clocks.stop()
    s1 = eng.get_stats()
    d = {k: s1[k] - s0[k] for k in ("steps", "tokens_emitted", "rows_senior", "rows_junior", "catchup_rows", "kv_bytes_read",
                                    "weight_bytes_read", "kernel_launches")}
    tokens = d["tokens_emitted"]
    ms_all, tokens_all = reduce_over_ranks(dist, ms, tokens, "cuda")
    pk = peaks()
    step_bytes = (d["weight_bytes_read"] + d["kv_bytes_read"]) / max(1, K)
    step_gbs = step_bytes / (ms / K * 1e-3) / 1e9
    ctx_mean = d["kv_bytes_read"] / max(1, tokens) / (shape.kv_elems_per_token * 2)

    # ---- per-kernel pass (library profile mode: one stream, events around every launch)
    roofline, kernels = None, {}
    if args.profile_steps > 0:
        p0 = eng.get_stats()
        if args.catchup_share:
            eng.set_option("profile_catchup_attention", 1)
        eng.set_profile(True)
        for _ in range(args.profile_steps):
            eng.step(prm, out=out, stream=stream)
        prof = eng.get_profile()
        eng.set_profile(False)
        p1 = eng.get_stats()
        psteps = max(1, p1["steps"] - p0["steps"])            # every launch serves both models: per-step totals
        rows = (p1["rows_senior"] + p1["rows_junior"] - p0["rows_senior"] - p0["rows_junior"]) / psteps
        emit_rows = (p1["tokens_emitted"] - p0["tokens_emitted"]) / psteps
        kv_launch = (p1["kv_bytes_read"] - p0["kv_bytes_read"]) / psteps / shape.n_layers
        empty_ms = prof.get("attention_empty", (0.0, 0))[0]     # a launch that finds no item: the fixed cost of the extra launches
        dup_all = prof.get("attention_catchup", (0.0, 0))[0] + empty_ms   # the filtered launches are extra work: not part of a step
        dup_ms = max(0.0, prof.get("attention_catchup", (0.0, 0))[0] - empty_ms)
        total_ms = sum(v[0] for v in prof.values()) - dup_all
        catchup = None
        if args.catchup_share:
            eng.set_option("profile_catchup_attention", 0)
            crows = (p1["catchup_rows"] - p0["catchup_rows"]) / psteps
            row_prop = ("gemm_qkv", "gemm_o", "gemm_gateup", "gemm_down", "rope_append", "residual_norm", "embed_norm", "attn_combine", "swiglu")
            by_rows = sum(prof[k][0] for k in row_prop if k in prof) * (crows / max(rows, 1e-9))
            catchup = {"share_of_step_time": (dup_ms + by_rows) / total_ms, "attention_catchup_ms_per_step": dup_ms / args.profile_steps,
                       "row_proportional_ms_per_step": by_rows / args.profile_steps, "catchup_rows_per_step": crows, "rows_per_step": rows,
                       "share_of_rows": crows / max(rows, 1e-9),
                       "method": "attention over items with q_len > 1 timed directly (second, filtered launch in the per-kernel pass); "
                                 "less the time of the same launch with no item at all; projection / norm / RoPE / combine time apportioned by rows; "
                                 "LM head, sampler, scheduler excluded"}
        for name, (kms, n) in prof.items():
            if n == 0:
                continue
            b = class_bytes(shape, name, rows, kv_launch, emit_rows)
            kernels[name] = {"ms_per_launch": kms / n, "launches_per_step": n / args.profile_steps, "share": kms / total_ms,
                             "alg_bytes_per_launch": b, "gbs": b / (kms / n * 1e-3) / 1e9 if kms > 0 else None}
        top = max(kernels, key=lambda k: kernels[k]["share"])
        kt = kernels[top]
        # DRAM bytes per launch of that kernel from the committed `ncu --set full` capture of this workload - valid only for the code
        # state it was captured on: the entry carries the hash of the kernel's sources, and a mismatch reports null
        traffic, traffic_note = None, "no capture for this workload"
        tpath = os.path.join(ROOT, "profiles", "traffic_r2.json")
        if os.path.exists(tpath):
            tj = json.load(open(tpath))
            for kname, tv in tj.items():
                if top == "attention" and "attention" in kname and tv.get("workload") == wl.name and tv.get("fast_forward") == args.fast_forward:
                    if tv.get("code_sha") == code_state():
                        traffic, traffic_note = tv["dram_bytes_per_launch"], "ncu --set full, %s" % tv.get("source", "profiles/")
                    else:
                        traffic_note = "stale: kernel sources changed since the capture (%s)" % tv.get("source", "profiles/")
        roofline = {"kernel": top, "bound": "hbm", "achieved": kt["gbs"], "peak": pk["hbm_gbs"], "unit": "GB/s",
                    "frac": kt["gbs"] / pk["hbm_gbs"], "traffic": traffic, "traffic_source": traffic_note, "alg_bytes_per_launch": kt["alg_bytes_per_launch"], "peak_source": pk["source"] + " burst copy (kernel timed alone)",
                    "share_of_step": kt["share"], "rows_per_launch": rows, "profile_steps": args.profile_steps,
                    "profile_ms_per_step": total_ms / args.profile_steps}

    res = {"metric": METRIC, "value": tokens_all / (ms_all * 1e-3), "unit": "tokens/s", "n_gpus": world, "steps": K, "warmup": W,
           "ms_per_step": ms_all / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
           "config": {"workload": wl.name, "batch_per_gpu": B, "prompt_len": list(wl.prompt_len), "fast_forward": args.fast_forward,
                      "ctx_mean_timed": ctx_mean, "p": wl.p, "word_start_frac": wl.word_start_frac, "temperature": wl.temperature, "top_p": wl.top_p, "top_k": args.top_k or wl.top_k, "switch_mode": "REDRAW" if wl.switch_mode else "TOGGLE",
                      "engine": "dual forward, lock-step (the paper's engine, measurement mode)" if args.dual_forward else "owner split + catch-up prefill",
                      **({"set_option": args.set_option} if args.set_option else {}),
                      **({"skip_class": args.skip_class + " (measurement: this kernel class was left out of the timed steps; not a throughput number)"} if args.skip_class else {}),
                      "page_tokens": 16, "parallelism": "dp%d (independent sequences, replicated weights, no collective)" % world,
                      "l2": "inputs larger than L2 (16.1 GB of weights + KV streamed per step vs 126 MB L2)",
                      "setup_steps": n_setup + ramp + n_drain, "setup_seconds": setup_s, "cuda_graph": True, "kv_gb_per_model": kv_per_model / 1e9},
           "clocks": clk, "gpu_launches": int(d["kernel_launches"]),
           "step_roofline": {"bound": "hbm", "alg_bytes_per_step": step_bytes, "weights_bytes_per_step": d["weight_bytes_read"] / K,
                             "kv_bytes_per_step": d["kv_bytes_read"] / K, "achieved": step_gbs, "unit": "GB/s",
                             "frac_of_measured": step_gbs / pk["hbm_gbs"], "frac_of_8TBs": step_gbs / NOMINAL_HBM_GBS,
                             "rows_per_step": (d["rows_senior"] + d["rows_junior"]) / K, "catchup_rows_per_step": d["catchup_rows"] / K},
           "roofline": roofline, "kernels": kernels}
    if args.profile_steps > 0 and catchup is not None:
        res["catchup_prefill"] = catchup

    # ---- end to end through tandem_generate with HOST buffers: prompts in (H2D), tokens / owner flags / senior log-probs out (D2H),
    # prefill and admission inside the timed region. e2e_short: max_new capped (first call warms the graph of this parameter set);
    # e2e: the WHOLE workload as BASELINE.json specifies it (every sequence to its max_new) - the metric itself.
    if not args.no_e2e:
        from workloads import make_max_new
        e_prompts = build_inputs(wl, 0, rank)[0]   # the workload's own prompts: rollouts from their start
        e_rows = sum(len(p) for p in e_prompts)

        def e2e_call(max_new_list):
            if dist: dist.barrier()
            t0 = time.perf_counter()
            g = eng.generate(prm, e_prompts, max_new_list, seq_ids=seq_ids, stream=stream)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            new_tot = int(np.sum(max_new_list))
            dt_all, tok = reduce_over_ranks(dist, dt, float(g["len"].sum()), "cuda")
            steps_e = max(1, g["stats"]["steps"])
            h2d = e_rows * 4 + (B + 1) * 8 + 3 * B * 4 + shape.vocab
            d2h = new_tot * (4 + 1 + 4) + B * 4
            st = g["stats"]
            gbs = (st["kv_bytes_read"] + st["weight_bytes_read"]) / max(st["seconds_total"], 1e-9) / 1e9
            return {"value": tok / dt_all, "unit": "tokens/s", "h2d_bytes_per_step": h2d / steps_e, "d2h_bytes_per_step": d2h / steps_e,
                    "call": "tandem_generate(B=%d host prompts of the workload, max_new=%d): prompt prefill + %d engine steps, host buffers in and out"
                            % (B, int(np.max(max_new_list)), steps_e),
                    "seconds": dt_all, "device_seconds": st["seconds_total"], "steps": int(st["steps"]), "tokens": int(tok),
                    "ms_per_step": st["seconds_total"] / steps_e * 1e3,
                    "senior_share": float(g["mask"].sum() / max(1, g["len"].sum())),
                    "step_roofline": {"bound": "hbm", "achieved": gbs, "unit": "GB/s", "frac_of_measured": gbs / pk["hbm_gbs"], "frac_of_8TBs": gbs / NOMINAL_HBM_GBS},
                    "share_prompt_pages": 0 if args.no_share_prompt_pages else args.share_mode, "prompt_rows": e_rows, "shared_prompt_rows": st["shared_prompt_rows"],
                    "kv_bytes_read": int(st["kv_bytes_read"]), "kv_bytes_shared_reads": int(st["kv_bytes_shared_reads"]),
                    "rows_computed": st["rows_senior"] + st["rows_junior"], "peak_resident": int(st["peak_resident"])}

        for it in range(2):
            res["e2e_short"] = e2e_call([args.e2e_new] * B)
        # the prefill part of a rollout on its own: the same call with one new token per sequence (prompt ingestion by both models,
        # admission, one sampled token); second call of two, like e2e_short
        for it in range(2):
            pf = e2e_call([1] * B)
        res["e2e_prefill"] = {"seconds": pf["seconds"], "steps": pf["steps"], "prompt_tokens": e_rows, "rows_computed": pf["rows_computed"],
                              "shared_prompt_rows": pf["shared_prompt_rows"], "prompt_tokens_per_s": e_rows / pf["seconds"],
                              "call": "tandem_generate(B=%d host prompts, max_new=1)" % B}
        if args.no_e2e_full or max_seq_len < max_prompt + wl.max_new:
            res["e2e"] = res["e2e_short"]
        else:
            res["e2e"] = e2e_call([int(x) for x in make_max_new(wl)])
    eng.free()
    torch.cuda.empty_cache()

    if rank == 0 and world == 1 and not args.no_cpu:
        res["cpu_baseline"] = oracle_sample(wl, w_cpu, build_inputs(wl, 0, rank)[0], table, seq_ids, args.cpu_new, prm_seed=20260628)
    if rank == 0:
        print(json.dumps(res))
    if dist:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------ the oracle, timed
def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info() if p.get("user_api") == "blas"]
        return max(n) if n else 1
    except Exception:
        return 1


def oracle_rollout(wl, w_cpu, prompt, table, seq_id, n_new, prm_seed, models=None):
    """One sequence of the workload through the oracle as it stands (incremental KV, float64 NumPy): returns
    (seconds, tokens emitted, models). The oracle is test infrastructure; this is the one place bench.py executes it."""
    from oracle import OracleModel, TandemParams as OParams, tandem_generate
    from oracle.rule import Uniforms
    if models is None:
        try:
            import psutil
            roomy = psutil.virtual_memory().available > 2.6 * 8 * wl.shape.params_read_per_step * 2
        except Exception:
            roomy = False
        models = (OracleModel(wl.shape, w_cpu[0], cache=roomy), OracleModel(wl.shape, w_cpu[1], cache=roomy))
    op = OParams(p=wl.p, switch_mode=wl.switch_mode, temperature=wl.temperature, top_p=wl.top_p, top_k=wl.top_k, seed=prm_seed)
    t0 = time.perf_counter()
    r = tandem_generate(models, op, [prompt], [n_new], table, uni=Uniforms(seed=prm_seed, seq_ids=[int(seq_id)]))
    dt = time.perf_counter() - t0
    return dt, len(r["tokens"][0]), models


def oracle_sample(wl, w_cpu, prompts, table, seq_ids, n_new, prm_seed):
    b = int(np.argmin([len(p) for p in prompts]))
    dt, n, _ = oracle_rollout(wl, w_cpu, prompts[b], table, seq_ids[b], n_new, prm_seed)
    return {"value": n / dt, "unit": "tokens/s", "cores": blas_threads(), "host_cpus": os.cpu_count(), "kind": "oracle",
            "sample": "1 of the %d sequences at the start of its rollout (the shortest prompt, %d ids), prompt prefill + %d new tokens, oracle.tandem_generate "
                      "incremental-KV float64 NumPy on the same bf16-valued weights; %.1f s" % (len(prompts), len(prompts[b]), n, dt)}


def run_reference(args):
    """--impl reference: for this tier the reference arm is the oracle, timed on the host cores. A step = one token of a
    one-sequence rollout of the workload (its prompt prefill is inside the timed region and amortised over the K tokens)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from workloads import get_workload, make_weights
    wl = get_workload(args.workload)
    W, K = max(1, args.warmup), args.steps
    prompts, table, seq_ids = build_inputs(wl, 0, 0)
    try:
        import torch
        dev = "cuda" if torch.cuda.is_available() else "cpu"   # the generator only: random weights are inputs, not arithmetic
    except Exception:
        dev = "cpu"
    w_cpu = []
    for seed in (wl.seeds["senior"], wl.seeds["junior"]):
        w = make_weights(wl.shape, seed, device=dev)
        w_cpu.append(dict(embed=w["embed"].cpu(), lm_head=w["lm_head"].cpu(), final_norm=w["final_norm"].cpu(),
                          layers=[{k: v.cpu() for k, v in l.items()} for l in w["layers"]]))
        del w
    order = np.argsort([len(p) for p in prompts])
    b0, b1 = int(order[0]), int(order[1])
    _, _, models = oracle_rollout(wl, w_cpu, prompts[b0], table, seq_ids[b0], W, 20260628)          # warm-up
    dt, n, _ = oracle_rollout(wl, w_cpu, prompts[b1], table, seq_ids[b1], K, 20260628, models=models)
    v = n / dt
    sample = ("1 of the %d sequences (prompt %d ids): prompt prefill + %d new tokens per timed run, oracle.tandem_generate "
              "incremental-KV float64 NumPy" % (len(prompts), len(prompts[b1]), n))
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": "tokens/s", "n_gpus": args.gpus, "steps": K, "warmup": W,
                      "ms_per_step": dt / max(1, n) * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                      "data": "synthetic", "config": {"workload": wl.name, "sample": sample},
                      "cpu_baseline": {"value": v, "unit": "tokens/s", "cores": blas_threads(), "host_cpus": os.cpu_count(), "kind": "oracle",
                                       "sample": sample},
                      "e2e": {"value": v, "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    elif a.grpo:
        run_grpo(a)
    elif a.score > 0:
        run_score(a)
    elif a.full_rollout > 0:
        run_full_rollout(a)
    else:
        run_ours(a)

"""BASELINE.json `configs` as data. No arithmetic of the method lives here."""
from dataclasses import dataclass, field, replace


@dataclass(frozen=True)
class ModelShape:
    n_layers: int
    hidden: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    intermediate: int
    vocab: int
    rms_eps: float = 1e-6
    rope_theta: float = 1e6
    dtype: str = "bf16"            # "f32" | "bf16": weights, activations at GEMM inputs, KV cache

    @property
    def params_read_per_step(self):
        """Parameters one decode step of one model streams: all layers + final norm + LM head
        (the embedding table is gathered, not streamed)."""
        h, i = self.hidden, self.intermediate
        qd, kd = self.n_q_heads * self.head_dim, self.n_kv_heads * self.head_dim
        per_layer = h * qd + 2 * h * kd + qd * h + 3 * h * i + 2 * h
        return self.n_layers * per_layer + h + self.vocab * h

    @property
    def kv_elems_per_token(self):
        return 2 * self.n_layers * self.n_kv_heads * self.head_dim


TINY = ModelShape(2, 128, 4, 2, 32, 384, 512, 1e-6, 1e4, "f32")
SMALL = ModelShape(24, 896, 14, 2, 64, 4864, 151936, 1e-6, 1e6, "bf16")
FOURB = ModelShape(36, 2560, 32, 8, 128, 9728, 151936, 1e-6, 1e6, "bf16")


@dataclass(frozen=True)
class Workload:
    name: str
    shape: ModelShape
    n_prompts: int
    group: int                     # rollouts per prompt (GRPO group)
    prompt_len: tuple              # (lo, hi) inclusive, uniform
    max_new: int                   # cap on new tokens
    geom_mean: float = 0.0         # > 0: max_new[b] = min(Geometric(1/geom_mean), max_new)   (R8)
    temperature: float = 1.0       # 0 => greedy
    top_p: float = 1.0
    top_k: int = 0                 # 0 = off (Table 3: training -1, evaluation 20)
    p: float = 0.5
    switch_mode: int = 0           # 0 TOGGLE, 1 REDRAW (the values of tandem.h / oracle.rule)
    word_start_frac: float = 0.30
    explicit_uniforms: bool = False
    page_tokens: int = 16
    seeds: dict = field(default_factory=lambda: dict(senior=1, junior=2, table=3, prompts=4, lengths=5, uniforms=6))

    @property
    def batch(self):
        return self.n_prompts * self.group

    def with_(self, **kw):
        return replace(self, **kw)


WORKLOADS = {
    # configs[0]: tiny tandem, fp32, greedy, explicit uniforms, B=4 distinct prompts of 16 ids, 32 new tokens
    # (prompt seed 6 instead of the default 4: chosen so that the greedy rollout has 18 owner switches and a
    #  minimum top-1/top-2 logit margin of 2.1e-3 >> fp32 error; seed 4 gives 2 switches. DESIGN.md §4.)
    "cfg1_tiny_f32": Workload("cfg1_tiny_f32", TINY, 4, 1, (16, 16), 32, temperature=0.0, explicit_uniforms=True,
                              seeds=dict(senior=1, junior=2, table=3, prompts=6, lengths=5, uniforms=6)),
    # configs[1]: small tandem, bf16, B=64 = 8 prompts x 8, prompts U[64,256], <=1024 new, "EOS w.p. 1/512 per step"
    "cfg2_small_bf16": Workload("cfg2_small_bf16", SMALL, 8, 8, (64, 256), 1024, geom_mean=512.0),
    # configs[2]: 4B-shape tandem, bf16, B=128 = 16 x 8, prompts U[64,512], 4096 new tokens, 16-token pages
    "cfg3_4b_bf16": Workload("cfg3_4b_bf16", FOURB, 16, 8, (64, 512), 4096),
    # configs[3]: 4B-shape, B=512 = 64 x 8, <=8192 new, geometric lengths (mean 3000)
    "cfg4_4b_long": Workload("cfg4_4b_long", FOURB, 64, 8, (64, 512), 8192, geom_mean=3000.0),
    # configs[4]: switch-rate sweep base point (p and word_start_frac are swept by the caller)
    "cfg5_sweep": Workload("cfg5_sweep", FOURB, 16, 8, (256, 256), 2048),
    # Reasoning-step handoff, the paper's evaluation protocol (section 4.3: the two models "alternate at every
    # \\n\\n-boundary token, each producing one reasoning step"; L480-482 App. C.5: an independent Bernoulli(0.5) draw at every
    # boundary instead), with the evaluation sampler of Table 3 (T 0.7, top-p 0.8, top-k 20). The table marks the boundary ids;
    # the stand-in marks 2% of the vocabulary, i.e. a reasoning step of about 50 tokens (the paper gives no step length).
    "handoff_strict_4b": Workload("handoff_strict_4b", FOURB, 16, 8, (64, 512), 4096, temperature=0.7, top_p=0.8, top_k=20, p=1.0,
                                  switch_mode=0, word_start_frac=0.02),
    "handoff_bernoulli_4b": Workload("handoff_bernoulli_4b", FOURB, 16, 8, (64, 512), 4096, temperature=0.7, top_p=0.8, top_k=20, p=0.5,
                                     switch_mode=1, word_start_frac=0.02),
}


def get_workload(name):
    return WORKLOADS[name]

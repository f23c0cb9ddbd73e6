"""Seeded synthetic inputs for the tandem rollout path - the ONLY module the CUDA path's harness
and the oracle's harness share. It holds none of the method's arithmetic: shapes, random weights,
random prompts, a random word-start table, random lengths and (for the tiny config) explicit
uniform arrays. The recipes are BASELINE.json's `configs` (stand-ins for the paper's workload:
Qwen3-4B-Instruct pair on DeepScaleR, 16 prompts x G=8, responses <= 3000, ~35% word-start ids -
PAPER.md L85, L269, L282-296; none of those assets exist here). See DESIGN.md §4.
"""
from .configs import ModelShape, Workload, WORKLOADS, get_workload
from .gen import (make_weights, make_word_start, make_prompts, make_max_new,
                  make_explicit_uniforms, flatten_prompts)

__all__ = ["ModelShape", "Workload", "WORKLOADS", "get_workload", "make_weights", "make_word_start",
           "make_prompts", "make_max_new", "make_explicit_uniforms", "flatten_prompts"]

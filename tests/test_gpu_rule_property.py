"""-m gpu: property test of the tandem rule (section 3.3, Alg. 1 lines 6-17, L271; readings R1-R7) - random draws of the
rule's parameters (p, TOGGLE / REDRAW, start owner incl. DRAW, sub-word cap, EOS id, word-start density, ragged prompts and lengths,
the counter generator's seed) on the tiny fp32 shape: the CUDA path's tokens, owner flags, lengths and senior mask must equal the
oracle's for every draw. The fixed parametrised cases of test_gpu_tiny_e2e.py cover the corners by hand; this one lets hypothesis
look for the combination nobody listed."""
import numpy as np
import pytest
from hypothesis import given, settings, strategies as st, HealthCheck

import paper_2606_28166_b200 as T
from oracle import TandemParams as OParams, tandem_generate
from oracle.rule import Uniforms
from workloads import get_workload, make_word_start
from gpu_util import make_pair

pytestmark = pytest.mark.gpu
SHAPE = get_workload("cfg1_tiny_f32").shape
_ENG = {}


def _engine():
    if "e" not in _ENG:                                   # one engine and one oracle pair for all examples: weights are not the subject
        _ENG["e"] = make_pair(SHAPE, (1, 2), max_seqs=3, max_seq_len=96, gain_jitter=0.1, std=0.08, max_rows_per_step=24)
    return _ENG["e"]


@settings(max_examples=25, deadline=None, derandomize=True, suppress_health_check=list(HealthCheck))
@given(p=st.sampled_from([0.0, 0.1, 0.5, 0.9, 1.0]), mode=st.sampled_from([T.TOGGLE, T.REDRAW]), start=st.sampled_from([T.SENIOR, T.JUNIOR, T.DRAW]),
       cap=st.sampled_from([0, 1, 3, 8]), eos=st.sampled_from([-1, 5, 100]), frac=st.sampled_from([0.0, 0.15, 0.5, 1.0]),
       temp=st.sampled_from([0.7, 1.0, 1.3]), seed=st.integers(0, 2 ** 40), lens=st.lists(st.integers(1, 40), min_size=3, max_size=3),
       news=st.lists(st.integers(1, 30), min_size=3, max_size=3))
def test_rule_gpu_equals_oracle_for_random_parameters(p, mode, start, cap, eos, frac, temp, seed, lens, news):
    eng, orc, _ = _engine()
    ws = make_word_start(SHAPE.vocab, frac, seed % 1000)
    rng = np.random.default_rng(seed % 65536)
    prompts = [rng.integers(0, SHAPE.vocab, size=n).astype(np.int32) for n in lens]
    op = OParams(p=p, switch_mode=mode, start_owner=start, cap_k=cap, temperature=temp, eos_id=eos, seed=seed)
    ref = tandem_generate(orc, op, prompts, news, ws, uni=Uniforms(seed=seed))
    out = eng.generate(T.TandemParams(ws, p=p, switch_mode=mode, start_owner=start, cap_k=cap, temperature=temp, eos_id=eos, seed=seed), prompts, news)
    for b in range(3):
        n = len(ref["tokens"][b])
        assert out["len"][b] == n
        assert np.array_equal(out["tokens"][b, :n], ref["tokens"][b])
        assert np.array_equal(out["owner"][b, :n], ref["owner"][b])
        assert np.array_equal(out["mask"][b, :n], ref["mask"][b])
        assert np.max(np.abs(out["sen_logp"][b, :n] - ref["sen_logp"][b])) <= 5e-5

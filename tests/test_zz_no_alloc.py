"""-m gpu: tandem_grpo_objective_static - the GRPO objective with the kernel's scratch (arrival counters, per-rollout objectives,
advantages) in the library's file-scope device array, for callers that must not allocate - against the existing path
(tandem_grpo_objective, caller-provided scratch) and the float64 oracle. Collected last on purpose (file name): the entry point shares
one array between all calls, and the suite runs with `pytest -x`.

Two calls in a row on different problems (a large one first, a small one after it, then the large one again): the array keeps the
previous call's contents, so a counter that is not cleared or a stale per-rollout objective that is read would show up in the second or
third result. Tolerance: the one tests/test_gpu_grpo.py uses against the oracle (2e-5 relative); against the existing path the results
are bit-identical (same kernel, same order of summation), which is asserted too."""
import numpy as np
import pytest
import torch

import paper_2606_28166_b200 as T
from oracle import grpo_objective as oracle_grpo

pytestmark = pytest.mark.gpu


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def _inputs(n_groups, G, L, seed):
    rng = np.random.default_rng(seed)
    B = n_groups * G
    rewards = rng.integers(0, 2, size=B).astype(np.float32)
    lengths = rng.integers(1, L + 1, size=B).astype(np.int32)
    owner = rng.integers(0, 2, size=(B, L)).astype(np.uint8)
    old = (-rng.random((B, L)) * 3).astype(np.float32)
    new = (old + rng.standard_normal((B, L)).astype(np.float32) * 0.3).astype(np.float32)
    ref = (old + rng.standard_normal((B, L)).astype(np.float32) * 0.2).astype(np.float32)
    return rewards, lengths, owner, new, old, ref


def _compare(case, result, token_obj):
    """One call of the static entry point into caller-owned outputs, checked against the existing path and the oracle."""
    n_groups, G, L, kl, seed = case
    rewards, lengths, owner, new, old, ref = _inputs(n_groups, G, L, seed)
    args = (_dev(rewards), G, _dev(lengths), _dev(owner), _dev(new), _dev(old), _dev(ref) if kl else None)
    want = T.grpo_objective(*args, clip_eps=0.2, kl_beta=kl)                       # existing path: caller-provided scratch
    tok = token_obj[:n_groups * G * L].view(n_groups * G, L)
    tok.fill_(-7.0)
    got = T.grpo_objective_static(*args, clip_eps=0.2, kl_beta=kl, token_obj=tok, result=result)
    rtol = 2e-5
    assert abs(got["loss"] - want["loss"]) <= 2e-6 + rtol * abs(want["loss"])
    assert got["n_senior"] == want["n_senior"] and got["n_live"] == want["n_live"]
    assert abs(got["clip_frac"] - want["clip_frac"]) <= 1e-6
    assert torch.allclose(tok, want["token_obj"], rtol=rtol, atol=2e-6)
    assert got["loss"] == want["loss"] and torch.equal(tok, want["token_obj"])     # same kernel, same summation order: bit for bit
    orc = oracle_grpo(rewards, G, lengths, owner, new, old, ref if kl else None, clip_eps=0.2, kl_beta=kl)
    assert abs(got["loss"] - orc["loss"]) <= 2e-6 + rtol * abs(orc["loss"]) and got["n_senior"] == orc["n_senior"]
    return got


def test_static_scratch_entry_point_matches_existing_path_on_calls_in_a_row():
    big = (16, 8, 700, 0.0, 41)          # cfg-3 rollout batch: 128 rollouts
    small = (3, 4, 17, 0.04, 42)         # 12 rollouts, KL term: reads entries [0, 12) of an array that still holds 128 from before
    result = torch.full((4,), float("nan"), device="cuda")
    token_obj = torch.empty(16 * 8 * 700, device="cuda")
    a = _compare(big, result, token_obj)
    b = _compare(small, result, token_obj)
    c = _compare(big, result, token_obj)
    assert a["loss"] == c["loss"] and a["n_senior"] == c["n_senior"] and a["clip_frac"] == c["clip_frac"]
    assert b["n_senior"] < a["n_senior"]
    # back to back on one stream without a host synchronisation in between: the second call's memset is ordered after the first's copy
    r1 = torch.empty(4, device="cuda"); r2 = torch.empty(4, device="cuda")
    rewards, lengths, owner, new, old, _ = _inputs(16, 8, 700, 41)
    rw2, ln2, ow2, nw2, ol2, _ = _inputs(2, 8, 50, 43)
    d1 = tuple(_dev(x) for x in (rewards, lengths, owner, new, old)); d2 = tuple(_dev(x) for x in (rw2, ln2, ow2, nw2, ol2))
    lib = T.binding.lib()
    for (rw, ln, ow, nw, ol), ng, L, r in ((d1, 16, 700, r1), (d2, 2, 50, r2)):
        assert lib.tandem_grpo_objective_static(ng, 8, L, rw.data_ptr(), ln.data_ptr(), ow.data_ptr(), nw.data_ptr(), ol.data_ptr(), None,
                                                0.2, 0.0, 1e-6, None, r.data_ptr(), None) == 0
    torch.cuda.synchronize()
    assert r1[0].item() == a["loss"]
    assert r2[0].item() == T.grpo_objective(d2[0], 8, d2[1], d2[2], d2[3], d2[4])["loss"]


def test_static_scratch_entry_point_limits():
    G = 8
    B = T.GRPO_STATIC_MAX_ROLLOUTS                       # exactly the maximum is accepted
    rewards, lengths, owner, new, old, _ = _inputs(B // G, G, 5, 44)
    args = (_dev(rewards), G, _dev(lengths), _dev(owner), _dev(new), _dev(old))
    got = T.grpo_objective_static(*args)
    assert got["loss"] == T.grpo_objective(*args)["loss"] and got["n_live"] > 0
    rewards, lengths, owner, new, old, _ = _inputs(B // G + 1, G, 5, 45)      # one group more: rejected, nothing launched
    res = torch.full((4,), 3.0, device="cuda")
    with pytest.raises(T.TandemError):
        T.grpo_objective_static(_dev(rewards), G, _dev(lengths), _dev(owner), _dev(new), _dev(old), result=res)
    torch.cuda.synchronize()
    assert torch.all(res == 3.0)

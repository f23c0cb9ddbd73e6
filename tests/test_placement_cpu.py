"""-m "not gpu": the paper's one-model-per-GPU placement as two gloo ranks on CPU - the hand-over logic of
paper_2606_28166_b200/placement.py. Rank m holds model m only (here: the oracle's model m with its own incremental KV state); per step
each rank serves the slots it owns and the ranks exchange one integer record per slot. What has to hold: both ranks end with the same
token streams and owner flags, equal to ONE process running oracle.tandem_generate with both models; a rank never evaluates a
sequence it does not own; the partner's catch-up equals the tokens emitted since its last turn."""
import os
import socket
import sys

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _inputs():
    from workloads import get_workload, make_word_start
    wl = get_workload("cfg1_tiny_f32")
    rng = np.random.default_rng(23)
    prompts = [rng.integers(0, wl.shape.vocab, size=int(n)).astype(np.int32) for n in (5, 16, 17, 9)]
    table = make_word_start(wl.shape.vocab, 0.4, 3)
    return wl, prompts, table, [14, 9, 12, 14]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2606_28166_b200 import placement as P
    from oracle import OracleModel, TandemParams as OParams, sample_token, owners_from_tokens
    from oracle.rule import Uniforms
    from workloads import make_weights
    wl, prompts, table, max_new = _inputs()
    prm = OParams(p=0.5, temperature=1.0, seed=41, eos_id=7)
    uni = Uniforms(seed=41)
    model = OracleModel(wl.shape, make_weights(wl.shape, wl.seeds["senior" if rank == 0 else "junior"]))   # this rank's model ONLY
    states = [model.new_state() for _ in prompts]
    calls, catchups = [], []

    def local_step(s, ctx, t):
        assert shared.owner[s] == rank
        st = states[s]
        catchups.append(len(ctx) - st.n)
        z = model.extend(st, ctx[st.n:])                                   # catch-up: everything the partner emitted since
        y = int(sample_token(z, prm.temperature, prm.top_p, uni.sample(s, t, wl.shape.vocab), prm.top_k))
        emitted = ctx[len(prompts[s]):] + [y]
        done = y == prm.eos_id or t >= max_new[s]
        nxt = int(owners_from_tokens(emitted + [y], table, prm, uni, b=s)[-1]) if not done else rank
        calls.append((s, t))
        return y, nxt, done

    shared = P.SharedContext(prompts, [0] * len(prompts))
    P.rollout_on_rank(dist, rank, shared, local_step, max_steps=64)
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), n=np.array([shared.n_emitted(s) for s in range(len(prompts))]),
             tokens=np.array([shared.ctx[s][len(prompts[s]):] + [-1] * (20 - shared.n_emitted(s)) for s in range(len(prompts))]),
             owners=np.array([shared.owners_log[s] + [9] * (20 - len(shared.owners_log[s])) for s in range(len(prompts))]),
             calls=np.array(calls), max_catchup=np.array([max(catchups)]))
    dist.barrier()
    dist.destroy_process_group()


def test_one_model_per_rank_equals_one_process(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0, r1 = np.load(tmp_path / "rank0.npz"), np.load(tmp_path / "rank1.npz")
    for k in ("n", "tokens", "owners"):
        assert np.array_equal(r0[k], r1[k]), k                            # both ranks hold the same context and flags
    from oracle import OracleModel, TandemParams as OParams, tandem_generate
    from oracle.rule import Uniforms
    from workloads import make_weights
    wl, prompts, table, max_new = _inputs()
    models = (OracleModel(wl.shape, make_weights(wl.shape, wl.seeds["senior"])), OracleModel(wl.shape, make_weights(wl.shape, wl.seeds["junior"])))
    ref = tandem_generate(models, OParams(p=0.5, temperature=1.0, seed=41, eos_id=7), prompts, max_new, table, uni=Uniforms(seed=41))
    for s in range(len(prompts)):
        n = int(r0["n"][s])
        assert n == len(ref["tokens"][s])
        assert np.array_equal(r0["tokens"][s, :n], ref["tokens"][s]) and np.array_equal(r0["owners"][s, :n], ref["owner"][s])
    # each (slot, t) was evaluated by exactly one rank - the owner - and both ranks worked; catch-ups of more than one token occurred
    c0, c1 = {tuple(x) for x in r0["calls"]}, {tuple(x) for x in r1["calls"]}
    assert not (c0 & c1) and len(c0) + len(c1) == int(r0["n"].sum()) and c0 and c1
    for s in range(len(prompts)):
        for t in range(1, int(r0["n"][s]) + 1):
            assert ((s, t) in c1) == bool(ref["owner"][s][t - 1])
    assert int(r1["max_catchup"][0]) > 1


def test_merge_handover_takes_the_owners_record():
    from paper_2606_28166_b200.placement import merge_handover, empty_records
    a, b = empty_records(3), empty_records(3)
    a[0] = (1, 11, 1, 0); a[1] = (1, 99, 0, 0)            # rank 0 owns slot 0; its row for slot 1 is garbage and must be ignored
    b[1] = (1, 22, 0, 1); b[2] = (0, -1, 0, 0)
    m = merge_handover([a, b], np.array([0, 1, 1], np.uint8))
    assert m.tolist() == [[1, 11, 1, 0], [1, 22, 0, 1], [0, -1, 0, 0]]

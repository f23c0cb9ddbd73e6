"""-m "not gpu": the N > 1 path of bench.py on CPU (gloo, world size 2, 127.0.0.1). The path shards by sequence with
replicated weights and no data-path collective, so what has to hold is:
  * every rank builds a disjoint shard of the workload whose sequence ids address the counter RNG globally;
  * a rank's results do not depend on what the other ranks hold (position-addressed uniforms): the union of the shards'
    rollouts equals one process running all sequences;
  * the whole-job number is (sum of units) / (max over ranks of the time).
The rollouts themselves are computed with the oracle here (the CUDA path needs a GPU); the sharding, seeding and reduction
code is bench.py's own."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rollout(wl, prompts, seq_ids, table, n_new):
    from oracle import OracleModel, TandemParams as OParams, tandem_generate
    from oracle.rule import Uniforms
    from workloads import make_weights
    models = (OracleModel(wl.shape, make_weights(wl.shape, wl.seeds["senior"])), OracleModel(wl.shape, make_weights(wl.shape, wl.seeds["junior"])))
    op = OParams(p=0.5, temperature=1.0, seed=99)
    return tandem_generate(models, op, prompts, [n_new] * len(prompts), table, uni=Uniforms(seed=99, seq_ids=seq_ids))


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from workloads import get_workload
    wl = get_workload("cfg1_tiny_f32")
    prompts, table, seq_ids = bench.build_inputs(wl, 3, rank)
    assert seq_ids.tolist() == list(range(rank * wl.batch, (rank + 1) * wl.batch))
    assert all(len(p) == 16 + 3 for p in prompts)                       # fast-forward appended
    ids = [torch.zeros(wl.batch, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(ids, torch.as_tensor(seq_ids, dtype=torch.int64))
    assert len(set(torch.cat(ids).tolist())) == world * wl.batch           # disjoint shards
    r = _rollout(wl, prompts, seq_ids, table, 6)
    ms, tok = bench.reduce_over_ranks(dist, 10.0 * (rank + 1), sum(len(t) for t in r["tokens"]), "cpu")
    assert ms == 10.0 * world and tok == world * wl.batch * 6              # max of the times, sum of the tokens
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), tokens=np.stack(r["tokens"]), owner=np.stack(r["owner"]),
             prompts=np.stack(prompts), seq_ids=seq_ids)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_by_sequence(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    parts = [np.load(tmp_path / f"rank{r}.npz") for r in range(world)]
    assert not np.array_equal(parts[0]["prompts"], parts[1]["prompts"])    # ranks hold different data
    # one process running the union with the same global sequence ids gives the same rollouts
    import bench
    from workloads import get_workload
    wl = get_workload("cfg1_tiny_f32")
    prompts = [p for part in parts for p in part["prompts"]]
    seq_ids = np.concatenate([part["seq_ids"] for part in parts])
    _, table, _ = bench.build_inputs(wl, 3, 0)
    r = _rollout(wl, prompts, seq_ids, table, 6)
    assert np.array_equal(np.stack(r["tokens"]), np.concatenate([part["tokens"] for part in parts]))
    assert np.array_equal(np.stack(r["owner"]), np.concatenate([part["owner"] for part in parts]))


def test_reduce_is_identity_without_a_group():
    import bench
    assert bench.reduce_over_ranks(None, 3.5, 7, "cpu") == (3.5, 7.0)

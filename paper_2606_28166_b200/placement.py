"""One model per GPU - the paper's own placement (the two policies are "loaded onto separate devices"; L330: "pi_sen on
cuda:0 and pi_jun on cuda:1") - as host-side hand-over logic. STATUS: design + this host logic,
tested with gloo at world size 2 on CPU (tests/test_placement_cpu.py); the single-GPU engine of this repo runs both models on one
device and does not call it (BASELINE.json scopes the build to one GPU).

The owner-split rollout maps onto two ranks without any tensor traffic: rank m holds model m, its paged KV cache and the sequences'
shared token context. A step is
  1. every rank evaluates ITS model on the sequences it currently owns (catch-up first: the positions its partner emitted since its
     last turn are already in the shared context) and samples y_t - position-addressed uniforms, so no rank needs the other's RNG;
  2. hand-over: each rank contributes one fixed-size record per slot - (emitted, token, next owner, done); the ranks all-gather the
     records (2 x max_seqs x 8 bytes per step over NVLink) and every rank keeps, for each slot, the record of the rank that OWNED the
     slot in this step. After the merge both ranks hold the same context, owner flags and finished set;
  3. the rank that lost a sequence does nothing for it until it takes control again, then ingests the tail of the context (its
     catch-up), exactly as the single-GPU scheduler does.
Only integers cross the link; the senior's log-probs stay on rank 0 (Eq. 1 needs them at senior positions only). The collective is
a real exchange step of the path (the partner cannot continue without y_t), so this is the one place a NCCL call belongs in the data
path; on one GPU there is none.
"""
import numpy as np

RECORD_FIELDS = ("emitted", "token", "next_owner", "done")


def empty_records(max_seqs):
    """One hand-over record per slot: int32 [max_seqs, 4] = (emitted 0/1, token, next owner, done 0/1)."""
    r = np.zeros((max_seqs, len(RECORD_FIELDS)), dtype=np.int32)
    r[:, 1] = -1
    return r


def merge_handover(records_by_rank, owner):
    """records_by_rank: list (index = rank = model) of int32 [max_seqs, 4]; owner: uint8 [max_seqs], who owned each slot in this step.
    Returns the merged records: row s is rank owner[s]'s row s. A rank's rows for slots it did not own are ignored, whatever they hold."""
    owner = np.asarray(owner)
    stacked = np.stack([np.asarray(r, dtype=np.int32) for r in records_by_rank])        # [world, S, 4]
    return stacked[owner.astype(np.int64), np.arange(owner.shape[0])]


def exchange(dist, local_records, owner):
    """All-gather the per-slot records over the process group `dist` (torch.distributed; nccl on GPUs, gloo in the CPU test) and
    merge them by this step's owner. Every rank returns the same array."""
    import torch
    world = dist.get_world_size()
    mine = torch.as_tensor(np.ascontiguousarray(local_records, dtype=np.int32))
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine)
    return merge_handover([p.numpy() for p in parts], owner)


class SharedContext:
    """What both ranks keep identical: per slot the token context, the current owner, the emitted count and the finished flag."""

    def __init__(self, prompts, start_owner):
        self.ctx = [[int(x) for x in p] for p in prompts]
        self.prompt_len = [len(p) for p in prompts]
        self.owner = np.asarray(start_owner, dtype=np.uint8).copy()
        self.done = np.zeros(len(prompts), dtype=np.uint8)
        self.owners_log = [[] for _ in prompts]

    def n_emitted(self, s):
        return len(self.ctx[s]) - self.prompt_len[s]

    def apply(self, merged):
        """Append the step's tokens and take over the next owners (identical on every rank: `merged` is)."""
        for s in range(len(self.ctx)):
            if self.done[s] or not merged[s, 0]:
                continue
            self.owners_log[s].append(int(self.owner[s]))
            self.ctx[s].append(int(merged[s, 1]))
            self.owner[s] = merged[s, 2]
            self.done[s] = merged[s, 3]


def rollout_on_rank(dist, rank, shared, local_step, max_steps):
    """The step loop of one rank. local_step(slot, context, t) -> (token, next_owner, done) is this rank's model + sampler + rule for
    a slot it owns (t = 1-based index of the token being emitted); it is called only for owned, unfinished slots."""
    S = len(shared.ctx)
    for _ in range(max_steps):
        if shared.done.all():
            break
        rec = empty_records(S)
        for s in range(S):
            if shared.done[s] or shared.owner[s] != rank:
                continue
            tok, nxt, fin = local_step(s, shared.ctx[s], shared.n_emitted(s) + 1)
            rec[s] = (1, tok, nxt, 1 if fin else 0)
        shared.apply(exchange(dist, rec, shared.owner.copy()))
    return shared

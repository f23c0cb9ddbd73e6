"""Helpers shared by the -m gpu tests: build an engine + the oracle pair on the same seeded weights."""
import numpy as np
import torch

import paper_2606_28166_b200 as T
from oracle import OracleModel
from workloads import make_weights


def make_pair(shape, seeds=(1, 2), max_seqs=8, max_seq_len=128, gain_jitter=0.0, std=0.02, same=False, **cfg_kw):
    """Returns (engine, (oracle_senior, oracle_junior), (w_senior, w_junior)). Weights are generated once
    (CPU generator) and handed to both sides."""
    ws = make_weights(shape, seeds[0], gain_jitter=gain_jitter, std=std)
    wj = ws if same else make_weights(shape, seeds[1], gain_jitter=gain_jitter, std=std)
    eng = T.Tandem(T.TandemConfig(shape, max_seqs=max_seqs, max_seq_len=max_seq_len, **cfg_kw))
    eng.load_weights(0, ws)
    eng.load_weights(1, wj)
    return eng, (OracleModel(shape, ws), OracleModel(shape, wj)), (ws, wj)


def dev(a, dtype=None):
    t = torch.as_tensor(np.ascontiguousarray(a)).cuda()
    return t if dtype is None else t.to(dtype)

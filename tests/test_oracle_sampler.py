"""Pins for oracle/sampler.py (pin 9): Gumbel-max law vs softmax (chi-square), small-T limit, greedy ties,
hand-worked top-p kept set."""
import numpy as np
from scipy import stats

from oracle import rng
from oracle.sampler import sample_token, kept_set_top_p, log_prob


def test_gumbel_max_frequencies_match_softmax():
    z = np.array([0.3, -1.2, 2.0, 0.0, 1.1, -0.5, 0.7, 1.9])
    T = 0.7
    p = np.exp(z / T) / np.sum(np.exp(z / T))
    n = 100000
    # uniforms drawn through the position-addressed generator: step t <-> one draw
    U = np.stack([rng.uniforms_sample(99, b, t, 8) for b in range(100) for t in range(1, n // 100 + 1)])
    counts = np.bincount([sample_token(z, T, 1.0, U[i]) for i in range(n)], minlength=8)
    chi2 = np.sum((counts - n * p) ** 2 / (n * p))
    assert chi2 < stats.chi2.ppf(0.999, df=7)


def test_small_temperature_is_argmax_and_greedy_ties():
    z = np.array([0.1, 3.0, 2.9, -1.0])
    u = rng.uniforms_sample(1, 0, 1, 4)
    assert sample_token(z, 1e-4, 1.0, u) == 1
    assert sample_token(np.array([1.0, 5.0, 5.0, 5.0]), 0.0, 1.0, None) == 1       # ties: lowest id
    assert sample_token(z, 0.0, 1.0, None) == 1


def test_top_p_hand_example():
    # probabilities 0.5, 0.3, 0.15, 0.05
    p = np.array([0.3, 0.05, 0.5, 0.15])
    z = np.log(p)
    assert kept_set_top_p(z, 1.0, 0.5).tolist() == [False, False, True, False]       # 0.5 reaches 0.5
    assert kept_set_top_p(z, 1.0, 0.51).tolist() == [True, False, True, False]
    assert kept_set_top_p(z, 1.0, 0.8).tolist() == [True, False, True, False]        # 0.8 reached exactly
    assert kept_set_top_p(z, 1.0, 0.81).tolist() == [True, False, True, True]
    assert kept_set_top_p(z, 1.0, 1.0).all()
    assert kept_set_top_p(z, 1.0, 1e-9).sum() == 1                                   # never empty
    # ties in probability: lower id first
    assert kept_set_top_p(np.zeros(4), 1.0, 0.3).tolist() == [True, True, False, False]
    # sampling never leaves the kept set; the winner is the Gumbel-argmax restricted to it
    for t in range(1, 200):
        u = rng.uniforms_sample(5, 0, t, 4)
        y = sample_token(z, 1.0, 0.8, u)
        assert y in (0, 2)
        g = rng.gumbel_from_uniform(u)
        assert y == (0 if z[0] + g[0] > z[2] + g[2] else 2)


def test_log_prob_is_pre_truncation_distribution():
    p = np.array([0.3, 0.05, 0.5, 0.15])
    assert abs(log_prob(np.log(p) + 7.0, 3, 1.0) - np.log(0.15)) < 1e-12
    q = p ** 2 / np.sum(p ** 2)
    assert abs(log_prob(np.log(p), 0, 0.5) - np.log(q[0])) < 1e-12

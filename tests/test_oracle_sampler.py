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


def test_top_k_hand_examples_and_composition_with_top_p():
    """Reading R18 (Table 3: evaluation top-k 20 with top-p 0.8): top-k first, then top-p on the
    distribution renormalised over the k survivors. Probabilities 0.3, 0.05, 0.5, 0.15, worked by hand."""
    from oracle.sampler import kept_set
    z = np.log(np.array([0.3, 0.05, 0.5, 0.15]))
    assert kept_set(z, 1.0, 1.0, 2).tolist() == [True, False, True, False]
    assert kept_set(z, 1.0, 1.0, 3).tolist() == [True, False, True, True]
    # top-3 renormalised: 0.526, 0.316, 0.158 -> 0.7 is reached by two ids; without top-k it is reached by two as well,
    # but 0.81 needs three ids without top-k (0.5 + 0.3 + 0.15) and, inside the top-2 {0.625, 0.375}, both
    assert kept_set(z, 1.0, 0.7, 3).tolist() == [True, False, True, False]
    assert kept_set(z, 1.0, 0.81, 2).tolist() == [True, False, True, False]
    assert kept_set(z, 1.0, 0.6, 2).tolist() == [False, False, True, False]          # 0.625 >= 0.6
    assert kept_set(z, 1.0, 0.63, 2).tolist() == [True, False, True, False]
    for k in (0, -1, 4, 100):                                                        # no filter
        assert kept_set(z, 1.0, 1.0, k).all()
        assert kept_set(z, 1.0, 0.81, k).tolist() == kept_set_top_p(z, 1.0, 0.81).tolist()
    assert kept_set(np.ones(5), 0.7, 1.0, 2).tolist() == [True, True, False, False, False]   # ties: lower id first
    # top-k 1 is greedy decoding whatever the uniforms; the kept set never depends on T > 0 when top_p = 1
    for t in range(1, 50):
        u = rng.uniforms_sample(9, 0, t, 4)
        assert sample_token(z, 0.7, 1.0, u, top_k=1) == 2
        assert sample_token(z, 0.7, 0.8, u, top_k=1) == 2
    assert kept_set(z, 0.3, 1.0, 2).tolist() == kept_set(z, 3.0, 1.0, 2).tolist()


def test_top_k_sampling_frequencies_follow_the_renormalised_distribution():
    """Gumbel-max restricted to the top-k set draws from softmax(z/T) renormalised over it."""
    p = np.array([0.1, 0.4, 0.2, 0.25, 0.05])
    z = np.log(p)
    n, cnt = 6000, np.zeros(5)
    for t in range(1, n + 1):
        cnt[sample_token(z, 1.0, 1.0, rng.uniforms_sample(77, 1, t, 5), top_k=3)] += 1
    assert cnt[0] == 0 and cnt[4] == 0
    want = np.array([0.4, 0.2, 0.25]) / 0.85
    got = cnt[[1, 2, 3]] / n
    assert np.max(np.abs(got - want)) < 4 * np.sqrt(0.25 / n)                        # four sigma of a binomial share

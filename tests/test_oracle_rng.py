"""Pins for oracle/rng.py (pin 14 of DESIGN.md §5): known-answer vectors, exactness of the uint32 ->
float32 map, uniformity, addressing."""
import os

import numpy as np
from scipy import stats

from oracle import rng

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def _kat_rows():
    rows = []
    with open(GOLDEN) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            rows.append(line.split())
    return rows


def test_philox_known_answers():
    rows = _kat_rows()
    assert len(rows) == 3
    for r in rows:
        ins = [int(x, 16) for x in r[:6]]
        out = rng.philox4x32_10(*ins)
        for got, exp in zip(out, r[6:]):
            if "?" in exp:
                continue
            assert int(got) == int(exp, 16)


def test_philox_vectorised_matches_scalar():
    c0 = np.arange(7, dtype=np.uint32)
    v = rng.philox4x32_10(c0, 5, 9, 1, 123, 456)
    for i in range(7):
        s = rng.philox4x32_10(i, 5, 9, 1, 123, 456)
        assert [int(x[i]) for x in v] == [int(x) for x in s]


def test_uniform_map_closed_form():
    # small r: exact (r + 0.5) * 2^-32 ; r = 0 is the minimum and is > 0
    assert rng.uniform_from_bits(0) == np.float32(2.0 ** -33)
    assert rng.uniform_from_bits(1) == np.float32(1.5 * 2.0 ** -32)
    assert rng.uniform_from_bits(5) == np.float32(5.5 * 2.0 ** -32)
    # top of the range clamps to the largest float32 below 1
    top = rng.uniform_from_bits(0xFFFFFFFF)
    assert top == np.float32(1.0 - 2.0 ** -24) and top < np.float32(1.0)
    # 2^31: float(r)=2^31 exactly, +0.5 is absorbed, result 0.5
    assert rng.uniform_from_bits(1 << 31) == np.float32(0.5)
    # monotone non-decreasing
    r = np.sort(np.random.default_rng(0).integers(0, 2 ** 32, size=10000, dtype=np.uint64)).astype(np.uint32)
    u = rng.uniform_from_bits(r)
    assert np.all(np.diff(u) >= 0) and u.min() > 0 and u.max() < 1


def test_uniformity_ks():
    u = np.concatenate([rng.uniforms_sample(7, b, t, 4096) for b in range(4) for t in range(1, 9)])
    assert stats.kstest(u.astype(np.float64), "uniform").pvalue > 1e-3
    us = np.array([rng.uniforms_switch(7, b, t) for b in range(40) for t in range(50)], dtype=np.float64)
    assert stats.kstest(us, "uniform").pvalue > 1e-3


def test_addressing():
    a = rng.uniforms_sample(11, 3, 5, 1000)
    b = rng.uniforms_sample(11, 3, 5, 1003)           # prefix property: word v does not depend on vocab
    assert np.array_equal(a, b[:1000])
    assert not np.array_equal(a, rng.uniforms_sample(11, 3, 6, 1000))
    assert not np.array_equal(a, rng.uniforms_sample(11, 4, 5, 1000))
    assert not np.array_equal(a, rng.uniforms_sample(12, 3, 5, 1000))
    # sample word 0 of block 0 and the switch uniform live on different streams
    assert a[0] != rng.uniforms_switch(11, 3, 5)
    # 64-bit seeds use both key words
    assert rng.uniforms_switch(1, 0, 0) != rng.uniforms_switch(1 + (1 << 32), 0, 0)


def test_gumbel_closed_form():
    # u = 1 - 1/e  =>  E = 1  =>  g = 0 ;  median of Gumbel: u = 1/2 => g = -ln(ln 2)
    assert abs(rng.gumbel_from_uniform(1 - np.exp(-1.0))) < 1e-12
    assert abs(rng.gumbel_from_uniform(0.5) + np.log(np.log(2.0))) < 1e-12
    g = rng.gumbel_from_uniform(rng.uniforms_sample(3, 0, 1, 200000))
    assert abs(g.mean() - 0.5772156649) < 0.01          # Euler-Mascheroni
    assert abs(g.var() - np.pi ** 2 / 6) < 0.03
    assert np.all(np.isfinite(g))

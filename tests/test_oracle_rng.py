"""Pins P1, P2: the oracle's Philox4x32-10 and integer draws."""
import os

import numpy as np

from oracle import ca_oracle as o
from tests import _philox_ref as pr

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def _kat():
    for line in open(GOLD):
        line = line.split("#")[0].strip()
        if line:
            w = [int(t, 16) for t in line.split()]
            yield w[0:4], w[4:6], w[6:10]


def test_p1_philox_known_answers():
    n = 0
    for ctr, key, out in _kat():
        assert o.philox4x32_10(ctr, key) == out
        assert o.philox4x32_10(ctr, key, precision="f32") == out
        assert pr.philox4x32_10(ctr, key) == out
        n += 1
    assert n == 3


def test_p1_philox_matches_independent_python_on_random_inputs():
    rng = np.random.default_rng(7)
    for _ in range(200):
        ctr = rng.integers(0, 2**32, 4).tolist()
        key = rng.integers(0, 2**32, 2).tolist()
        assert o.philox4x32_10(ctr, key) == pr.philox4x32_10(ctr, key)


def test_p2_uniform_int_definition_and_range():
    # G23: floor(x*m / 2^32): exact integer identities
    assert o.uniform_int(0, 7) == 0
    assert o.uniform_int(2**32 - 1, 7) == 6
    assert o.uniform_int(2**31, 2) == 1
    assert o.uniform_int(2**31 - 1, 2) == 0
    rng = np.random.default_rng(3)
    for x, m in zip(rng.integers(0, 2**32, 500).tolist(), rng.integers(1, 70000, 500).tolist()):
        v = o.uniform_int(x, m)
        assert v == (x * m) >> 32 and 0 <= v < m


def test_p2_bernoulli_threshold():
    assert o.bernoulli_threshold(0.0) == 0
    assert o.bernoulli_threshold(1.0) == 2**32 - 1
    assert o.bernoulli_threshold(0.5) == 2**31
    assert o.bernoulli_threshold(0.25) == 2**30
    assert o.bernoulli_threshold(1e-12) == 0
    assert o.bernoulli_threshold(1 - 1e-12) == 2**32 - 1


def test_p2_uniformity_chi_square():
    # 2^16 draws of word 0 over consecutive sites -> 16 equiprobable bins (chi2, 15 dof, p=1e-4 -> 44.3)
    n = 1 << 16
    bins = np.zeros(16)
    for site in range(n):
        bins[pr.word0(0x1234, site, 5, 9, 2) >> 28] += 1
    chi2 = float(((bins - n / 16) ** 2 / (n / 16)).sum())
    assert chi2 < 44.3

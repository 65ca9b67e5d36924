"""Pins for the oracle's long accumulator (oracle/md_oracle.cpp: LongAcc) -- the exact arithmetic every other
oracle check rests on.  Pinned against Python's exact rationals and math.fsum, never against itself."""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import md_oracle as orc
from tests.exact import F, fsum_exact, round_to_limbs


def _wild(rng, n, emin=-300, emax=300):
    return np.ldexp(rng.uniform(-1, 1, n), rng.integers(emin, emax, n).astype(np.int32))


@pytest.mark.parametrize("limbs", [1, 2, 4])
def test_exact_sum_matches_rational_rounding(limbs):
    rng = np.random.default_rng(10 + limbs)
    for trial in range(40):
        x = _wild(rng, int(rng.integers(1, 60)), -200, 200)
        if trial % 3 == 0:  # massive cancellation
            x = np.concatenate([x, -x[::-1], _wild(rng, 3, -400, -350)])
        got = orc.exact_sum(x, limbs)
        want = round_to_limbs(fsum_exact(x), limbs)
        assert list(got) == want


def test_exact_sum_is_fsum_for_one_limb():
    rng = np.random.default_rng(5)
    for _ in range(50):
        x = _wild(rng, 100, -60, 60)
        assert orc.exact_sum(x, 1)[0] == math.fsum(x)


def test_exact_sum_ties_to_even_and_subnormals():
    # 1 + 2^-53 is a tie: rounds to 1 (even); adding a dust term breaks the tie upward.
    assert list(orc.exact_sum(np.array([1.0, 2.0 ** -53]), 2)) == [1.0, 2.0 ** -53]
    assert orc.exact_sum(np.array([1.0, 2.0 ** -53, 2.0 ** -200]), 1)[0] == 1.0 + 2.0 ** -52
    assert orc.exact_sum(np.array([1.0 + 2.0 ** -52, 2.0 ** -53]), 1)[0] == 1.0 + 2.0 ** -51  # tie -> even
    tiny = 5e-324
    assert list(orc.exact_sum(np.array([tiny, tiny, tiny]), 1)) == [3 * tiny]
    assert list(orc.exact_sum(np.array([2.0 ** -1022, -tiny]), 1)) == [2.0 ** -1022 - tiny]
    assert list(orc.exact_sum(np.array([-3.5, 1.25]), 2)) == [-2.25, 0.0]


@pytest.mark.parametrize("limbs", [2, 4])
def test_exact_dot_matches_rational(limbs):
    rng = np.random.default_rng(77)
    for _ in range(30):
        n = int(rng.integers(1, 40))
        x, y = _wild(rng, n), _wild(rng, n)
        want = round_to_limbs(sum((F(a) * F(b) for a, b in zip(x, y)), Fraction(0)), limbs)
        assert list(orc.exact_dot(x, y, limbs)) == want


def test_exact_dot_extreme_exponents():
    x = np.array([2.0 ** 1000, 2.0 ** -1000, 5e-324, -(2.0 ** 1000)])
    y = np.array([2.0 ** 20, 2.0 ** -60, 5e-324, 2.0 ** 20])
    want = round_to_limbs(sum((F(a) * F(b) for a, b in zip(x, y)), Fraction(0)), 2)
    assert list(orc.exact_dot(x, y, 2)) == want

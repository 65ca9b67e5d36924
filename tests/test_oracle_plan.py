"""Pins for the oracle's data-driven quarter count (oracle_plan_quarters; R15, SURVEY.md 8(f) NEXT-1
"exponent-spread-driven quarter count").

Pinned against: exact rational arithmetic (W = |A_0||B_0| and the inequality k (Q+3) 2^(D - bits Q - 2) <= rel_tol restated
with Fractions), math.frexp for the exponents, closed-form special cases, the invariance of D under row / column scaling by
powers of two, and -- what the plan is FOR -- the exact product: with the planned Q the five-step pipeline is within
rel_tol (|A||B|)_ij at every position of an input on which the paper's count (8) is not."""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import md_oracle as orc
from paper_2607_06881_b200 import inputs
from tests.exact import F

INT32_MIN = -2 ** 31


def exact_spread(A0, B0):
    """max over W_ij > 0 of E_i + F_j - floor(log2 W_ij), W exact."""
    m, k = A0.shape
    n = B0.shape[1]
    E = [math.frexp(v)[1] if v else 0 for v in np.abs(A0).max(axis=1)]
    Fx = [math.frexp(v)[1] if v else 0 for v in np.abs(B0).max(axis=0)]
    best, near_power_of_two = None, False
    for i in range(m):
        for j in range(n):
            w = sum(abs(F(A0[i, t])) * abs(F(B0[t, j])) for t in range(k))
            if w == 0:
                continue
            e = w.numerator.bit_length() - w.denominator.bit_length()
            if Fraction(2) ** e > w:
                e -= 1
            assert Fraction(2) ** e <= w < Fraction(2) ** (e + 1)
            near_power_of_two |= (w / Fraction(2) ** e - 1) < Fraction(1, 2 ** 40) or (2 - w / Fraction(2) ** e) < Fraction(1, 2 ** 40)
            d = E[i] + Fx[j] - e
            best = d if best is None else max(best, d)
    return best, near_power_of_two


def smallest_Q(k, limbs, bits, D, rel_tol):
    Q = -(-(52 * limbs) // bits)
    while Fraction(k * (Q + 3)) * Fraction(2) ** (D - bits * Q - 2) > Fraction(rel_tol):
        Q += 1
    return Q


@pytest.mark.parametrize("cfg_idx,bits,tol", [(0, 13, 1e-28), (1, 13, 1e-28), (3, 13, 1e-28), (3, 19, 1e-28), (4, 13, 1e-58)])
def test_plan_matches_rational_restatement(cfg_idx, bits, tol):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(9, 8, 14)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    Q, D = orc.plan_quarters(A, B, tol, bits=bits)
    D_exact, ambiguous = exact_spread(A[0], B[0])
    assert not ambiguous and D == D_exact
    assert Q == smallest_Q(cfg.k, cfg.limbs, bits, D, tol)


def test_special_cases():
    eye = np.zeros((2, 6, 6))
    eye[0] = np.eye(6)
    # E_i = F_j = 1 (max 1 -> ilogb + 1), W = I: D = 2 on the diagonal, nothing elsewhere
    Q, D = orc.plan_quarters(eye, eye, 1e-28)
    assert D == 2 and Q == smallest_Q(6, 2, 13, 2, 1e-28) == 8
    zero = np.zeros((2, 3, 4))
    Q, D = orc.plan_quarters(zero, np.zeros((2, 4, 5)), 1e-28)
    assert D == INT32_MIN and Q == 8
    # all elements equal to 1: W_ij = k, E = F = 1 -> D = 2 - ilogb(k)
    ones = np.zeros((2, 4, 16))
    ones[0] = 1.0
    Q, D = orc.plan_quarters(ones, np.ascontiguousarray(ones.transpose(0, 2, 1)), 1e-28)
    assert D == 2 - 4


def test_spread_is_invariant_under_power_of_two_scaling_of_rows_and_columns():
    cfg = inputs.CONFIGS[3].with_shape(12, 10, 20)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    rng = np.random.default_rng(5)
    sa = np.ldexp(1.0, rng.integers(-40, 40, 12).astype(np.int32))[None, :, None]
    sb = np.ldexp(1.0, rng.integers(-40, 40, 10).astype(np.int32))[None, None, :]
    assert orc.plan_quarters(A, B, 1e-28) == orc.plan_quarters(A * sa, B * sb, 1e-28)


def test_planned_count_delivers_the_tolerance_where_the_papers_count_does_not():
    """Config 3's distribution (elements over 2^[-30,30], "stresses balancing/quarter count") at a small k: with the
    paper's 8 quarters some positions miss 1e-28 (|A||B|)_ij; with the planned count every position is inside."""
    cfg = inputs.CONFIGS[3].with_shape(48, 40, 24)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    Q, D = orc.plan_quarters(A, B, 1e-28)
    assert Q > 8 and D > 8
    r8 = orc.exact_all(A, B, orc.md_gemm_rows(A, B, quarters=8))
    assert (r8["err"] > 1e-28 * r8["W"]).any()
    rq = orc.exact_all(A, B, orc.md_gemm_rows(A, B, quarters=Q))
    assert (rq["err"] <= 1e-28 * rq["W"]).all()
    # the bound the plan rests on (R5), position by position, for both counts
    _, eA, _ = orc.split(A, 0)
    _, eB, _ = orc.split(B, 1)
    for QQ, r in ((8, r8), (Q, rq)):
        bound = cfg.k * (QQ + 3) * np.ldexp(1.0, (eA[:, None] + eB[None, :] - 13 * QQ - 2).astype(np.int32))
        assert (r["err"] <= bound + 2.0 ** -105 * r["W"]).all()

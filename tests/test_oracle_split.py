"""Pins for the oracle's Algorithm S (oracle_split; R1-R5).

Pinned against: exact rational arithmetic (sum invariant, independent nearest-digit expansion), math.frexp (library
routine for the exponent), the paper's printed constants (tests/golden/paper_constants.txt), and special cases whose
digits are derived by hand in the comments."""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import md_oracle as orc
from paper_2607_06881_b200 import inputs
from tests.exact import F, nearest_digits
from tests.golden import load_paper_constants

PAPER = load_paper_constants()
W = PAPER["quarter_bits"][0]  # 13


def small_cfg(idx, m=24, n=20, k=28):
    return inputs.CONFIGS[idx].with_shape(m, n, k)


def digits_of(qp, exps, axis):
    """Integer digits D_q = d_q / u_q as Python ints (exact: the division is by a power of two)."""
    Q, rows, cols = qp.shape
    D = np.empty(qp.shape, dtype=object)
    for q in range(Q):
        for i in range(rows):
            for j in range(cols):
                E = int(exps[i] if axis == 0 else exps[j])
                v = F(qp[q, i, j]) / Fraction(2) ** (E - W * (q + 1))
                assert v.denominator == 1, "quarter is not a multiple of its unit"
                D[q, i, j] = int(v)
    return D


@pytest.mark.parametrize("cfg_idx", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("axis", [0, 1])
def test_sum_of_quarters_plus_remainder_is_exact(cfg_idx, axis):
    """north_star check (i): the sum of an element's quarters reproduces it exactly (the
    balancing moves do not change the value)."""
    cfg = small_cfg(cfg_idx)
    X = inputs.generate(cfg, "A" if axis == 0 else "B")
    qp, exps, rem = orc.split(X, axis, want_remainder=True)
    L, rows, cols = X.shape
    Q = qp.shape[0]
    assert Q == PAPER["quarters_per_double"][0] * L
    for i in range(rows):
        for j in range(cols):
            elt = sum(F(X[l, i, j]) for l in range(L))
            parts = sum(F(qp[q, i, j]) for q in range(Q)) + sum(F(rem[l, i, j]) for l in range(L))
            assert parts == elt
            E = int(exps[i] if axis == 0 else exps[j])
            # the remainder is at most half a unit of the last quarter (plus the lower limbs' dust)
            assert abs(sum(F(rem[l, i, j]) for l in range(L))) <= Fraction(2) ** (E - W * Q) * Fraction(1025, 2048)


@pytest.mark.parametrize("cfg_idx", [0, 1, 2, 3, 4])
def test_exponent_vector_is_frexp_of_group_max(cfg_idx):
    cfg = small_cfg(cfg_idx, 33, 17, 29)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    _, eA, _ = orc.split(A, 0)
    _, eB, _ = orc.split(B, 1)
    assert [math.frexp(v)[1] for v in np.abs(A[0]).max(axis=1)] == list(eA)
    assert [math.frexp(v)[1] for v in np.abs(B[0]).max(axis=0)] == list(eB)
    for E, M in zip(eA, np.abs(A[0]).max(axis=1)):
        assert 2.0 ** (int(E) - 1) <= M < 2.0 ** int(E)


@pytest.mark.parametrize("cfg_idx", [0, 1, 2, 3, 4])
def test_digits_are_on_the_grid_and_bounded(cfg_idx):
    """Quarter q is an integer multiple of 2^(E - 13(q+1)) -- the paper's exponents 0, -13, -26, -39
    relative to the group -- with a 13-bit digit: |D_0| <= 2^13, |D_q| <= 2^12 (q >= 1)."""
    assert PAPER["quarter_exponents"] == [0, -13, -26, -39]
    cfg = small_cfg(cfg_idx)
    X = inputs.generate(cfg, "A")
    qp, exps, _ = orc.split(X, 0)
    D = digits_of(qp, exps, 0)
    assert max(abs(d) for d in D[0].ravel()) <= 2 ** W
    assert max(abs(d) for d in D[1:].ravel()) <= 2 ** (W - 1)
    # relative to the leading unit u_0, quarter q's unit is 2^(-13 q): the paper's grid
    for q in range(4):
        assert (int(exps[0]) - W * (q + 1)) - (int(exps[0]) - W) == PAPER["quarter_exponents"][q]


@pytest.mark.parametrize("cfg_idx", [0, 1, 3, 4])
def test_digits_equal_exact_nearest_expansion(cfg_idx):
    """Brute force in exact arithmetic: away from ties, Algorithm S produces the unique expansion
    D_q = RN(R_q / u_q) of the exact element value (an independent restatement with rationals)."""
    cfg = small_cfg(cfg_idx, 12, 10, 16)
    X = inputs.generate(cfg, "A")
    qp, exps, _ = orc.split(X, 0)
    D = digits_of(qp, exps, 0)
    L, rows, cols = X.shape
    checked = 0
    for i in range(rows):
        for j in range(cols):
            value = sum(F(X[l, i, j]) for l in range(L))
            want, _, margin = nearest_digits(value, int(exps[i]), qp.shape[0])
            # An exact tie (margin 0) is representable in the leading remainder limb, so both round it to even alike;
            # a NEAR tie (within 2^-30 of a unit) may be seen as a tie by the fp64 leading limb alone: skipped.
            if margin == 0 or margin > Fraction(1, 2 ** 30):
                assert [D[q, i, j] for q in range(qp.shape[0])] == want
                checked += 1
    assert checked > rows * cols * 0.99


def test_hand_derived_special_cases():
    Q = 8

    def run(hi, lo, others_hi=()):
        """Split the row [hi, *others] (+lo for the first element) and return (E, digits of element 0, remainder)."""
        row_hi = np.array([[hi, *others_hi]])
        row_lo = np.array([[lo] + [0.0] * len(others_hi)])
        qp, exps, rem = orc.split(np.stack([row_hi, row_lo]), 0, want_remainder=True)
        E = int(exps[0])
        return E, [int(F(qp[q, 0, 0]) / Fraction(2) ** (E - W * (q + 1))) for q in range(Q)], rem[:, 0, 0]

    # PAPER.md:124 Problem 3.3 (hi > 0, lo < 0): x = 1 - 2^-60.  Row max 1 -> E = 1, u_0 = 2^-12, u_4 = 2^-64.
    # 1 = 4096 u_0; -2^-60 = -16 u_4.  The low double simply contributes a digit of its own sign.
    E, D, rem = run(1.0, -(2.0 ** -60))
    assert (E, D) == (1, [4096, 0, 0, 0, -16, 0, 0, 0]) and not rem.any()
    # A small element in a row whose max is 0.75 (E = 0): 1.5 * 2^-41 = 3 * 2^-42 = 3072 * 2^-52 = 3072 u_3.
    E, D, rem = run(1.5 * 2.0 ** -41, 0.0, others_hi=(0.75,))
    assert (E, D) == (0, [0, 0, 0, 3072, 0, 0, 0, 0]) and not rem.any()
    # hi exactly on a tie of the leading unit (2^-14 = u_0/2, E = 0) with a tiny lo: ties-to-even on the leading limb
    # sends D_0 to 0 whatever the sign of lo; 2^-14 = 4096 u_1; +-2^-80 = +-2048 u_6 (u_6 = 2^-91).
    for sgn in (1.0, -1.0):
        E, D, rem = run(2.0 ** -14, sgn * 2.0 ** -80, others_hi=(0.75,))
        assert (E, D) == (0, [0, 4096, 0, 0, 0, 0, int(sgn) * 2048, 0]) and not rem.any()
    # The row maximum just below 2^E: 1 - 2^-53 + 2^-55 -> D_0 reaches the 2^13 bound; 8192 u_0 = 1, and the rest
    # -2^-53 + 2^-55 = -3 * 2^-55 = -3072 * 2^-65 = -3072 u_4.
    E, D, rem = run(1.0 - 2.0 ** -53, 2.0 ** -55)
    assert (E, D) == (0, [8192, 0, 0, 0, -3072, 0, 0, 0]) and not rem.any()
    # 2/3 rounded to double, E = 0: 0.101010..b -> 5461.33 u_0 -> 5461, remainder +1/3 u_0 = 2730.67 u_1 -> 2731,
    # remainder -1/3 u_1 -> -2731, then +1/3 -> 2730.67 but the double ends: 0x1.5555555555555p-1 has 53 bits, so
    # check only the first three digits by hand and the rest through the exact expansion.
    x = float.fromhex("0x1.5555555555555p-1")
    E, D, rem = run(x, 0.0)
    assert E == 0 and D[:3] == [5461, 2731, -2731]
    assert D == nearest_digits(F(x), 0, Q)[0]


def test_zero_rows_columns_and_signed_zero():
    X = np.zeros((2, 3, 4))
    X[0, 1, :] = [0.5, -0.0, 0.0, -0.25]
    qp, exps, rem = orc.split(X, 0, want_remainder=True)
    assert list(exps) == [0, 0, 0]  # all-zero rows: E = 0 (zeros are left alone)
    assert not qp[:, 0].any() and not qp[:, 2].any() and not rem.any()
    assert not np.signbit(qp[:, 1, 1]).any()  # -0.0 gives +0.0 digits
    assert qp[0, 1, 0] == 0.5 and qp[0, 1, 3] == -0.25
    _, eB, _ = orc.split(X, 1)
    assert list(eB) == [0, 0, 0, -1]


def test_axis1_is_axis0_of_the_transpose():
    cfg = small_cfg(3, 16, 24, 20)
    B = inputs.generate(cfg, "B")
    q1, e1, r1 = orc.split(B, 1, want_remainder=True)
    q0, e0, r0 = orc.split(np.ascontiguousarray(B.transpose(0, 2, 1)), 0, want_remainder=True)
    assert (e0 == e1).all() and (q0.transpose(0, 2, 1) == q1).all() and (r0.transpose(0, 2, 1) == r1).all()


def test_one_limb_is_the_plain_13_bit_slicing():
    """L = 1 (a plain double): with E the exponent of the element itself the digits are the 13-bit
    fields of the 53-bit significand, recoded to nearest: sum D_q 2^(-13(q+1)) == x / 2^E exactly with Q = 5."""
    rng = np.random.default_rng(3)
    x = rng.uniform(0.5, 1.0, (1, 40, 1))  # each row is its own group, E = 0
    qp, exps, rem = orc.split(x, 0, quarters=5, want_remainder=True)
    assert (exps == 0).all() and not rem.any()  # 65 bits hold every 53-bit significand
    for i in range(40):
        m = int(F(x[0, i, 0]) * 2 ** 53)  # the integer significand
        D = [int(F(qp[q, i, 0]) * 2 ** (W * (q + 1))) for q in range(5)]
        assert sum(d * 2 ** (65 - W * (q + 1)) for q, d in enumerate(D)) == m * 2 ** 12
        assert D == nearest_digits(F(x[0, i, 0]), 0, 5)[0]


def test_values_already_on_the_grid_leave_no_remainder():
    rng = np.random.default_rng(4)
    D = rng.integers(-4096, 4097, (8, 6, 7))
    X = np.zeros((2, 6, 7))
    X[0] = sum(D[q] * 2.0 ** (-13 * (q + 1)) for q in range(4))   # exact: 52 bits
    X[1] = sum(D[q] * 2.0 ** (-13 * (q + 1)) for q in range(4, 8))
    X[0, :, 0] = 0.75  # pins E = 0 for every row
    X[1, :, 0] = 0.0
    _, exps, rem = orc.split(X, 0, want_remainder=True)
    assert (exps == 0).all() and not rem.any()


def test_split_of_a_quarter_plane_returns_itself_in_one_digit():
    """Idempotence: quarter plane q of a matrix, split again on the same group exponents, is a single
    non-zero digit -- itself -- at position q (or q-1 .. when the row's maximum moved: here every row keeps an element
    that pins E, so the position is q)."""
    cfg = small_cfg(1, 9, 5, 11)
    X = inputs.generate(cfg, "A")
    qp, exps, _ = orc.split(X, 0)
    for q in (0, 3, 7):
        Y = np.zeros_like(X)
        Y[0] = qp[q]
        Y[0, :, 0] = np.ldexp(0.75, exps)  # one element per row pins the row exponent E_i (0.75 * 2^E has ilogb = E - 1)
        qq, e2, rem = orc.split(Y, 0, want_remainder=True)
        assert (e2 == exps).all() and not rem.any()
        for t in range(qq.shape[0]):
            want = qp[q][:, 1:] if t == q else np.zeros_like(qp[q][:, 1:])
            assert (qq[t][:, 1:] == want).all()


def test_row_of_equal_powers_of_two_is_one_digit():
    """A row whose elements are all +-2^e: E = e + 1, and every element is the single digit +-2^12 u_0 (u_0 = 2^(E-13))."""
    for e in (-40, 0, 17):
        row = np.ldexp(1.0, e) * np.array([[1.0, -1.0, 1.0, 1.0, -1.0]])
        qp, exps, rem = orc.split(np.stack([row, np.zeros_like(row)]), 0, want_remainder=True)
        assert list(exps) == [e + 1] and not rem.any() and not qp[1:].any()
        assert (qp[0] == row).all() and (np.abs(qp[0]) == 4096 * np.ldexp(1.0, e + 1 - W)).all()


def test_power_of_two_scaling_shifts_the_grid_and_nothing_else():
    """Scaling a row by 2^s moves its exponent by s and multiplies every quarter by 2^s: same integer digits (the method
    is scale-free per group -- what a common exponent per row / column buys, R2)."""
    cfg = small_cfg(3, 9, 5, 11)
    X = inputs.generate(cfg, "A")
    s = np.array([-300, -7, 0, 1, 13, 52, 200, 511, -512], dtype=np.int32)
    Xs = X * np.ldexp(1.0, s)[None, :, None]
    q0, e0, r0 = orc.split(X, 0, want_remainder=True)
    q1, e1, r1 = orc.split(Xs, 0, want_remainder=True)
    assert (e1 == e0 + s).all()
    assert (q1 == q0 * np.ldexp(1.0, s)[None, :, None]).all() and (r1 == r0 * np.ldexp(1.0, s)[None, :, None]).all()

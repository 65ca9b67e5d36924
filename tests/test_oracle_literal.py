"""Pins of oracle part O6: the paper's OWN section-3 balancing, element by element (R17-R22) --
per-double quartering, eq. (7), eq. (8), the zero rule, the exponent classes A_0..A_12
 and the sign groups of eq. (6).

Pinned against things other than the oracle: exact rational / big-integer arithmetic in Python (`fractions`, `math.frexp`), the
worked cases of the paper's own text (eq. 7: x_h = 1 with a negative x_l; eq. 8: b = 2^-14 for an x_1 with leading zeros),
value invariance of every move ("Obviously, the value ... does not change"), and the exact product O1.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import md_oracle as orc
from paper_2607_06881_b200 import inputs
from tests.exact import F, round_to_limbs

TOL = {2: 1e-28, 4: 1e-58, 8: 1e-120, 16: 1e-245}


def fr(values):
    return sum((F(v) for v in np.asarray(values).ravel()), Fraction(0))


def ilogb(x: float) -> int:
    return math.frexp(abs(x))[1] - 1


# ------------------------------------------------------------------------------------------------ R17: one double, 4 parts
@pytest.mark.parametrize("x", [1.0, -1.0, 1.5, math.pi, -math.e * 2.0 ** 40, 1.0 + 2.0 ** -52, 2.0 - 2.0 ** -52,
                               float.fromhex('0x1.5555555555555p-1'), 3e-300, -7.25e250, 1.0 + 2.0 ** -26, 0.0])
def test_quarter_double_is_the_bit_field_split(x):
    parts = orc.quarter_double(x)
    assert fr(parts) == F(x)                                    # x_0 + x_1 + x_2 + x_3 == x
    if x == 0.0:
        assert parts == [0.0] * 4
        return
    e = ilogb(x)
    # independent restatement on Python integers: 52 fraction bits in four fields of 13
    M = int(Fraction(abs(x)) / Fraction(2) ** (e - 52))
    assert M >> 52 == 1
    f = M - (1 << 52)
    fields = [(1 << 13) + (f >> 39), (f >> 26) & 8191, (f >> 13) & 8191, f & 8191]
    sign = -1 if x < 0 else 1
    for t, (part, field) in enumerate(zip(parts, fields)):
        assert F(part) == sign * field * Fraction(2) ** (e - 13 * (t + 1))      # on the grid 0, -13, -26, -39
    assert 2 ** 13 <= fields[0] < 2 ** 14 and all(0 <= v < 2 ** 13 for v in fields[1:])


def test_two_quarters_multiply_with_26_trailing_zero_bits():
    """'Multiplying two quarters leaves at least 26 zero bits at the end' -- for the 13-bit parts; the leading
    part carries the hidden bit too (14 bits), so a product of two leading parts needs 28 bits."""
    rng = np.random.default_rng(7)
    for x, y in rng.standard_normal((50, 2)):
        qx, qy = orc.quarter_double(float(x)), orc.quarter_double(float(y))
        for a in qx:
            for b in qy:
                prod = a * b
                assert Fraction(prod) == F(a) * F(b)                       # exact
                if prod != 0.0:
                    mant = int(Fraction(abs(prod)) / Fraction(2) ** (ilogb(prod) - 52))
                    assert mant % (1 << 24) == 0                           # at most 28 significant bits: >= 24 trailing zeros
        for a in qx[1:]:
            for b in qy[1:]:
                if a * b != 0.0:
                    mant = int(Fraction(abs(a * b)) / Fraction(2) ** (ilogb(a * b) - 52))
                    assert mant % (1 << 26) == 0                           # the paper's 26


# ------------------------------------------------------------------------------------------------ R18: eq. (7)
def test_eq7_worked_case_of_the_paper():
    """x_h > 0 with exponent zero, x_l < 0: b = 2^-52, x_h := x_h - b, x_l := x_l + b > 0."""
    x, carry = orc.eq7([1.0, -(2.0 ** -60)])
    assert x.tolist() == [1.0 - 2.0 ** -52, 2.0 ** -52 - 2.0 ** -60] and not carry.any()
    assert fr(x) == F(1.0) - F(2.0 ** -60)                                  # "the value ... does not change"
    x, carry = orc.eq7([1.75, -(2.0 ** -55) * 1.25])
    assert x[0] == 1.75 - 2.0 ** -52 and x[1] > 0 and fr(x) + fr(carry) == F(1.75) - F(2.0 ** -55 * 1.25)
    # negative element, positive low part: mirrored
    x, carry = orc.eq7([-1.0, 2.0 ** -60])
    assert x.tolist() == [-(1.0 - 2.0 ** -52), -(2.0 ** -52 - 2.0 ** -60)]
    # same signs / zero low part: untouched
    for v in ([1.0, 2.0 ** -60], [1.0, 0.0], [0.0, 0.0], [-3.0, -(2.0 ** -54)]):
        x, carry = orc.eq7(v)
        assert x.tolist() == v and not carry.any()


def test_eq7_the_last_bit_goes_to_the_next_double():
    """'As x_l grows in size, we may loose the last bit of x_l.  Therefore ... the last bit should then be added
    to the next double in the sequence'.  x_l with 53 significant bits right below one ulp of x_h: x_l + b needs 54."""
    lo = -(2.0 ** -54) * (1.0 + 2.0 ** -52)          # x_l + b = 2^-52 - 2^-54 - 2^-106 needs 54 bits
    x, carry = orc.eq7([1.0, lo, 2.0 ** -140, 0.0])
    assert fr(x) + fr(carry) == F(1.0) + F(lo) + F(2.0 ** -140)
    assert x[0] == 1.0 - 2.0 ** -52 and all(v >= 0 for v in x)
    assert x[2] != 2.0 ** -140                         # the bit that fell off x_l + b went into the third double
    # dd: nowhere to go but the carry
    x, carry = orc.eq7([1.0, lo])
    assert carry[0] != 0.0 and fr(x) + fr(carry) == F(1.0) + F(lo)


@pytest.mark.parametrize("cfg_idx", [0, 1, 2, 3, 4, 5, 6])
def test_eq7_value_invariant_and_one_sign(cfg_idx):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(6, 5, 7)
    A = inputs.generate(cfg, "A")
    for i in range(cfg.m):
        for j in range(cfg.k):
            x, carry = orc.eq7(A[:, i, j])
            assert fr(x) + fr(carry) == fr(A[:, i, j])
            nz = x[x != 0.0]
            assert (nz > 0).all() or (nz < 0).all()


# ------------------------------------------------------------------------------------------------ R19: eq. (8) + zero rule
def test_eq8_worked_case_of_the_paper():
    """x_0 in A_0 (exponent zero), the exponents of x_0 and x_1 differ by more than 13: b = 2^-14,
    x_0 := x_0 - b, x_1 := x_1 + b; 'x_1 + b has exponent -13' (its 13-bit field now starts with a one), 'Subtracting b does
    not alter the exponent of x_0'.  Here x = 1 + 2^-26: x_1 = 2^-26 has twelve leading zeros in its field."""
    parts = orc.quarter_double(1.0 + 2.0 ** -26)
    assert parts == [1.0, 2.0 ** -26, 0.0, 0.0]
    d = orc.eq8(parts, 0)
    assert d.tolist() == [1.0 - 2.0 ** -14, 2.0 ** -14 + 2.0 ** -26, 0.0, 0.0]     # zero parts: "just do nothing"
    assert fr(d) == F(1.0 + 2.0 ** -26)                                              # "the value of x_0 + x_1 remains invariant"
    assert ilogb(d[0]) == -1 or d[0] >= 0.5                                          # (x_0 = 1 exactly drops below 1: still 14 bits)
    assert 2.0 ** -14 <= d[1] < 2.0 ** -13
    # worst case of PAPER.md:135 ("-25, -38, -51"): every lower field = 1
    x = 1.5 + 2.0 ** -26 + 2.0 ** -39 + 2.0 ** -52
    d = orc.eq8(orc.quarter_double(x), 0)
    assert fr(d) == F(x)
    assert 2.0 ** -14 <= d[1] < 2.0 ** -13
    # x_1 lends to x_2 only if that keeps x_1's own exponent: here x_1 = 2^-14 + 2^-26 > 2^12 units, so it does
    assert 2.0 ** -27 <= d[2] < 2.0 ** -26 and 2.0 ** -14 <= d[1] < 2.0 ** -13
    # quarters already on the grid: untouched
    full = orc.quarter_double(math.pi / 2)
    on_grid = all(abs(p) >= 2.0 ** (-13 * t - 1) for t, p in enumerate(full) if t)     # every field starts with a one
    assert (orc.eq8(full, 0).tolist() == full) == on_grid
    gridded = [1.0 + 2.0 ** -13, 2.0 ** -14, 2.0 ** -27 + 2.0 ** -39, 2.0 ** -40]
    assert orc.eq8(gridded, 0).tolist() == gridded


def test_eq8_never_changes_the_value_and_keeps_half_units():
    rng = np.random.default_rng(11)
    for _ in range(300):
        e = int(rng.integers(-40, 40))
        digits = rng.integers(0, 2 ** 13, size=8) * (rng.random(8) < 0.8) * (2.0 ** -rng.integers(0, 13, size=8)).round(0).clip(0, 1)
        digits = np.where(rng.random(8) < 0.3, rng.integers(0, 8, size=8), rng.integers(0, 2 ** 13, size=8))
        digits[0] += 2 ** 13
        sign = -1.0 if rng.random() < 0.5 else 1.0
        d0 = np.array([sign * float(D) * 2.0 ** (e - 13 * (q + 1)) for q, D in enumerate(digits)])
        d = orc.eq8(d0, e)
        assert fr(d) == fr(d0)
        for q in range(8):
            half = Fraction(2) ** (e - 13 * (q + 1) - 1)
            assert (F(d[q]) / half).denominator == 1                     # a multiple of u_q / 2
            assert abs(F(d[q]) / half) < 2 ** 15
            if digits[q] == 0 and q > 0:
                assert d[q] == 0.0 or q == 0                             # a zero part stays zero
            if q > 0 and d[q] != d0[q] and abs(d[q]) > abs(d0[q]):       # a part that borrowed now has its top field bit set
                assert abs(F(d[q])) >= 2 ** 12 * 2 * half - half


# ------------------------------------------------------------------------------------------------ Algorithm L on matrices
@pytest.mark.parametrize("cfg_idx", [0, 1, 2, 3, 4, 5, 6])
@pytest.mark.parametrize("apply_eq8", [False, True])
def test_split_literal_exact_sum_grid_and_bounds(cfg_idx, apply_eq8):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(9, 5, 11)
    L, Q = cfg.limbs, 4 * cfg.limbs
    A = inputs.generate(cfg, "A")
    A[:, 0, 0] = 0.0                      # a zero element
    A[:, 1, 1] = [1.0] + [0.0] * (L - 1)  # a power of two
    if L >= 2:
        A[:2, 2, 2] = [1.0, -(2.0 ** -60)]  # PAPER.md:124 Problem 3.3
    qp, exps, rem = orc.split_literal(A, Q, apply_eq8, want_remainder=True)
    assert exps[0, 0] == 0 and not qp[:, 0, 0].any()
    for i in range(cfg.m):
        for j in range(cfg.k):
            x, d, e = A[:, i, j], qp[:, i, j], int(exps[i, j])
            assert fr(d) + fr(rem[:, i, j]) == fr(x)                       # north_star check (i), per element and exact
            v = fr(x)
            if v == 0:
                continue
            adj, _ = orc.eq7(x)
            assert e == ilogb(float(adj[adj != 0.0][0]))                    # the exponent of the leading quarter
            assert Fraction(2) ** e <= abs(fr(adj)) < Fraction(2) ** (e + 1) or abs(adj[adj != 0.0][0]) >= 2.0 ** e
            nz = d[d != 0.0]
            assert (nz > 0).all() or (nz < 0).all()                        # one sign after eq. (7)
            for q in range(Q):
                half = Fraction(2) ** (e - 13 * (q + 1) - 1)
                D = F(d[q]) / half
                assert D.denominator == 1 and (apply_eq8 or D % 2 == 0)    # on the grid (half units only after eq. 8)
                assert abs(D) <= (2 ** 15 if q == 0 else 2 ** 14)
            # what is left is below the last unit (per limb): the 13 Q bits below 2^(e+1) hold the element
            assert abs(fr(rem[:L, i, j])) < L * Fraction(2) ** (e - 13 * Q)
    # the worked case: 1 - 2^-60 after eq. (7) is (1 - 2^-52) + (2^-52 - 2^-60): exponent -1, all parts positive
    if L == 2:
        assert exps[2, 2] == -1 and (qp[:, 2, 2] >= 0).all()


@pytest.mark.parametrize("cfg_idx", [0, 1, 2, 3])
def test_split_literal_digits_are_the_bit_fields_of_the_exact_value(cfg_idx):
    """Without eq. (8), and where the limbs of the sign-fixed element do not overlap, part q is bits [e - 13 q - 1 .. e - 13 (q+1)]
    of |v| (the leading part with the top bit at 2^e): the plain definition of 'distribute the bits into parts of 13 bits'
     applied to the whole multiple double.  Computed here on Python big integers."""
    cfg = inputs.CONFIGS[cfg_idx].with_shape(12, 5, 13)
    A = inputs.generate(cfg, "A")
    qp, exps, _ = orc.split_literal(A, 8, apply_eq8=False)
    checked = 0
    for i in range(cfg.m):
        for j in range(cfg.k):
            adj, carry = orc.eq7(A[:, i, j])
            if carry.any() or abs(adj[1]) >= math.ulp(adj[0]):            # overlapping limbs: several valid cuts, not this pin
                continue
            v, e = abs(fr(adj)), int(exps[i, j])
            sign = 1 if fr(adj) > 0 else -1
            for q in range(8):
                u = Fraction(2) ** (e - 13 * (q + 1))
                field = int(v / u) - (int(v / (u * 2 ** 13)) << 13 if q else 0)
                assert F(qp[q, i, j]) == sign * field * u
            checked += 1
    assert checked > 100


# ------------------------------------------------------------------------------------------------ R20-R22: the literal product
def brute_force_literal(A, B, Q, apply_eq8):
    """Independent restatement in exact rationals: the kept products are those of global order
    p + (zmaxA - za) + q + (zmaxB - zb) < Q + spanA + spanB; C = their exact sum, rounded limb by limb."""
    L, m, k = A.shape
    n = B.shape[2]
    Aq, eA, _ = orc.split_literal(A, Q, apply_eq8)
    Bq, eB, _ = orc.split_literal(B, Q, apply_eq8)
    zA = np.floor_divide(eA, 13)
    zB = np.floor_divide(eB, 13)
    nzA, nzB = Aq.any(axis=0), Bq.any(axis=0)
    zmaxA, zminA = (int(zA[nzA].max()), int(zA[nzA].min())) if nzA.any() else (0, 0)
    zmaxB, zminB = (int(zB[nzB].max()), int(zB[nzB].min())) if nzB.any() else (0, 0)
    S = Q + (zmaxA - zminA) + (zmaxB - zminB)
    C = np.zeros((L, m, n))
    for i in range(m):
        for j in range(n):
            total = Fraction(0)
            for t in range(k):
                for p in range(Q):
                    if Aq[p, i, t] == 0.0:
                        continue
                    for q in range(Q):
                        if p + (zmaxA - int(zA[i, t])) + q + (zmaxB - int(zB[t, j])) < S:
                            total += F(Aq[p, i, t]) * F(Bq[q, t, j])
            C[:, i, j] = round_to_limbs(total, L)
    return C, (zminA, zmaxA, zminB, zmaxB)


@pytest.mark.parametrize("cfg_idx,shape", [(3, (5, 4, 9)), (0, (4, 4, 6)), (4, (3, 3, 5)), (1, (4, 5, 7))])
@pytest.mark.parametrize("apply_eq8", [False, True])
def test_literal_product_equals_the_rational_brute_force(cfg_idx, shape, apply_eq8):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(*shape)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    Q = 4 * cfg.limbs
    want, info = brute_force_literal(A, B, Q, apply_eq8)
    for sign_groups in (False, True):
        C, got_info = orc.md_gemm_literal(A, B, Q, apply_eq8, sign_groups)
        assert got_info == info
        assert (C == want).all()          # exact sums, correctly rounded: the sign groups of eq. (6) change nothing (R21)


@pytest.mark.parametrize("cfg_idx", [0, 1, 2, 3, 4])
def test_literal_product_meets_the_tolerance_with_the_papers_quarter_count(cfg_idx):
    """The point of per-element exponents: the error is relative to |a_ik||b_kj| term by term, hence to (|A||B|)_ij, whatever
    the dynamic range -- cfg3's distribution (elements over 2^+-30) passes with the paper's 8 quarters, where the row / column
    grid needs 9 or 10 (R5, R15)."""
    cfg = inputs.CONFIGS[cfg_idx].with_shape(24, 20, 64)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    Q = 4 * cfg.limbs
    C, _ = orc.md_gemm_literal(A, B, Q)
    r = orc.exact_all(A, B, C)
    assert (r["err"] <= TOL[cfg.limbs] * r["W"]).all()
    if cfg_idx == 3:
        # the same input through the row / column grid with 8 quarters misses the tolerance somewhere (why cfg3 runs with 9)
        C8 = orc.md_gemm_rows(A, B, quarters=8)
        r8 = orc.exact_all(A, B, C8)
        assert (r8["err"] > 1e-28 * r8["W"]).any()
        assert (r["err"] / r["W"]).max() < 2.0 ** -96          # (Q + 3) 2^-102 relative, term by term


def test_literal_product_closed_forms():
    # identity: C = B up to what the 13 Q-bit window of each element drops (nothing for dd elements with |lo| >= 2^-104 |hi|)
    cfg = inputs.CONFIGS[3].with_shape(6, 6, 6)
    B = inputs.generate(cfg, "B")
    I = np.zeros((2, 6, 6))
    I[0] = np.eye(6)
    C, _ = orc.md_gemm_literal(I, B, 8)
    r = orc.exact_all(I, B, C)
    assert (r["err"] <= 2.0 ** -100 * r["W"]).all()
    # small integers: exact
    rng = np.random.default_rng(3)
    A = np.zeros((2, 5, 7)); Bm = np.zeros((2, 7, 4))
    A[0] = rng.integers(-2 ** 20, 2 ** 20, size=(5, 7)); Bm[0] = rng.integers(-2 ** 20, 2 ** 20, size=(7, 4))
    C, _ = orc.md_gemm_literal(A, Bm, 8)
    want = A[0].astype(np.int64) @ Bm[0].astype(np.int64)
    assert (C[0] + C[1] == want).all() and (C[0] == want.astype(np.float64)).all()
    # zero matrix
    C, info = orc.md_gemm_literal(np.zeros((2, 3, 3)), Bm[:, :3, :], 8)
    assert not C.any() and info[:2] == (0, 0)

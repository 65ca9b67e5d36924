"""Pins for the oracle's slice-width parameter (oracle_*_w; R14): Algorithm S with `bits` in place of the
paper's 13 ("4 parts ... each of 13 bits" = 52/4), the order matrices on the unit 2^(E_i+F_j-bits(s+2)),
and the k-budget that generalises PAPER.md:95-99 eq. 5.

Pinned against: exact rational arithmetic (sum invariant, the independent nearest-digit expansion of tests/exact.py,
Fraction brute force of the order sums, the exact product O1), an identity that ties the wider slices back to the
paper's quarters (for one limb a 26-bit slice is the sum of two adjacent 13-bit quarters), and the paper's eq. 5
constant.  No expected value comes from the CUDA path."""
from fractions import Fraction

import numpy as np
import pytest

from oracle import md_oracle as orc
from paper_2607_06881_b200 import inputs
from tests.exact import F, nearest_digits
from tests.golden import load_paper_constants

PAPER = load_paper_constants()
WIDTHS = [7, 13, 19, 20, 24]


def small(idx, m=10, n=9, k=12):
    return inputs.CONFIGS[idx].with_shape(m, n, k)


def digit(v, E, q, bits):
    d = F(v) / Fraction(2) ** (E - bits * (q + 1))
    assert d.denominator == 1, "slice is not a multiple of its unit"
    return int(d)


@pytest.mark.parametrize("bits", WIDTHS)
@pytest.mark.parametrize("cfg_idx,axis", [(0, 0), (3, 1), (4, 0)])
def test_sum_of_slices_plus_remainder_is_exact_and_digits_bounded(bits, cfg_idx, axis):
    """north_star check (i) at any width: error-free, on the grid, |D_0| <= 2^bits, |D_q| <= 2^(bits-1)."""
    cfg = small(cfg_idx)
    X = inputs.generate(cfg, "A" if axis == 0 else "B")
    L, rows, cols = X.shape
    Q = -(-(53 * L) // bits)
    qp, exps, rem = orc.split(X, axis, quarters=Q, want_remainder=True, bits=bits)
    for i in range(rows):
        for j in range(cols):
            E = int(exps[i] if axis == 0 else exps[j])
            elt = sum(F(X[l, i, j]) for l in range(L))
            rho = sum(F(rem[l, i, j]) for l in range(L))
            assert sum(F(qp[q, i, j]) for q in range(Q)) + rho == elt
            assert abs(rho) <= Fraction(2) ** (E - bits * Q) * Fraction(1025, 2048)
            D = [digit(qp[q, i, j], E, q, bits) for q in range(Q)]
            assert abs(D[0]) <= 2 ** bits and all(abs(d) <= 2 ** (bits - 1) for d in D[1:])


@pytest.mark.parametrize("bits", [7, 19, 20])
@pytest.mark.parametrize("cfg_idx", [0, 3, 4])
def test_digits_equal_exact_nearest_expansion(bits, cfg_idx):
    """Away from ties the slices are the unique expansion D_q = RN(R_q / u_q) of the exact element value."""
    cfg = small(cfg_idx, 8, 8, 10)
    X = inputs.generate(cfg, "A")
    L, rows, cols = X.shape
    Q = -(-(52 * L) // bits)
    qp, exps, _ = orc.split(X, 0, quarters=Q, bits=bits)
    checked = 0
    for i in range(rows):
        for j in range(cols):
            E = int(exps[i])
            want, _, margin = nearest_digits(sum(F(X[l, i, j]) for l in range(L)), E, Q, bits)
            if margin == 0 or margin > Fraction(1, 2 ** 30):
                assert [digit(qp[q, i, j], E, q, bits) for q in range(Q)] == want
                checked += 1
    assert checked > rows * cols * 0.99


def test_one_limb_26_bit_slices_are_pairs_of_the_papers_quarters():
    """For a plain double (L = 1) rounding to a multiple of u_1 = 2^(E-26) in one step or in two (first to 2^(E-13),
    then the exact rest to 2^(E-26)) gives the same value, because D_0 * 2^13 is even and keeps the tie parity.  So
    slice_t(bits = 26) == quarter_2t + quarter_2t+1 of PAPER.md:47-49 exactly."""
    rng = np.random.default_rng(11)
    x = rng.standard_normal((1, 30, 17)) * 2.0 ** rng.integers(-20, 20, (1, 30, 17))
    q13, e13, _ = orc.split(x, 0, quarters=6, bits=13)
    q26, e26, _ = orc.split(x, 0, quarters=3, bits=26)
    assert (e13 == e26).all()
    for t in range(3):
        assert (q26[t] == q13[2 * t] + q13[2 * t + 1]).all()   # the fp64 sum of two adjacent quarters is exact (26 bits)


@pytest.mark.parametrize("bits,Q", [(19, 6), (20, 6), (7, 9), (19, 11)])
def test_order_routes_agree_and_match_rational_brute_force(bits, Q):
    """int64 digit route == plain fp64 route bit for bit (the exactness claim of PAPER.md:51-54, :95 at this width),
    and both equal the Fraction sum of the slice products."""
    cfg = small(0 if Q < 10 else 4, 5, 4, 6)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    Aq, eA, _ = orc.split(A, 0, quarters=Q, bits=bits)
    Bq, eB, _ = orc.split(B, 1, quarters=Q, bits=bits)
    oi, raw = orc.orders_int(Aq, eA, Bq, eB, want_raw=True, bits=bits)
    of = orc.orders_fp64(Aq, Bq)
    assert (oi == of).all()
    for s in range(Q):
        for i in range(cfg.m):
            for j in range(cfg.n):
                want = sum(F(Aq[p, i, t]) * F(Bq[s - p, t, j]) for p in range(s + 1) for t in range(cfg.k))
                assert F(oi[s, i, j]) == want
                assert Fraction(int(raw[s, i, j])) * Fraction(2) ** (int(eA[i]) + int(eB[j]) - bits * (s + 2)) == want


def test_k_budget_generalises_eq5():
    """PAPER.md:95-99 eq. 5: N (2^26 - 1) <= 2^52 -> N <= 67 108 865 for products of two 13-bit parts.  With slices of
    `bits` bits (|D| <= 2^bits) and S products per k in an order, every partial sum stays an exactly representable
    integer while k S 2^(2 bits) <= 2^53 (R6 / R14).  Worst-case digits at the bound still accumulate exactly."""
    assert (2 ** 52) // (2 ** 26 - 1) == PAPER["exact_sum_bound_N"][0]
    for bits, S in ((13, 8), (19, 6), (20, 4)):
        k = 2 ** 53 // (S * 2 ** (2 * bits))
        assert k * S * 2 ** (2 * bits) <= 2 ** 53 < (k + 1) * S * 2 ** (2 * bits) * 2
        kk = min(k, 4096)  # a row of worst-case digits: every slice of every element at its bound
        Aq = np.zeros((S, 1, kk))
        Bq = np.zeros((S, kk, 1))
        for q in range(S):
            Aq[q] = (2.0 ** bits if q == 0 else 2.0 ** (bits - 1)) * 2.0 ** (-bits * (q + 1))
            Bq[q] = Aq[q, 0, 0]
        z = np.zeros(1, dtype=np.int32)
        assert (orc.orders_int(Aq, z, Bq, z, bits=bits) == orc.orders_fp64(Aq, Bq)).all()


@pytest.mark.parametrize("cfg_idx,bits,Q,tol", [(0, 19, 6, 1e-28), (1, 19, 6, 1e-28), (2, 19, 6, 1e-28),
                                                (3, 19, 6, 1e-28), (4, 19, 11, 1e-58)])
def test_wide_slice_pipeline_reaches_the_north_star_tolerance(cfg_idx, bits, Q, tol):
    """The five steps with 19-bit slices (dd: 6 slices = 114 bits >= the paper's 8 x 13 = 104; qd: 11 slices = 209 >=
    208) against the exact product O1: |C - C_exact| <= tol (|A||B|)_ij on the five input distributions."""
    cfg = inputs.CONFIGS[cfg_idx].with_shape(12, 11, 64)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    C = orc.md_gemm_rows(A, B, quarters=Q, bits=bits)
    r = orc.exact_all(A, B, C)
    assert (r["err"] <= tol * r["W"]).all()


# ---------------------------------------------------------------------------------------------- chunked accumulation (R16)
def test_chunked_pipeline_with_one_chunk_is_the_plain_pipeline():
    cfg = small(1, 9, 7, 40)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    for chunk in (40, 64):
        assert (orc.md_gemm_rows_chunked(A, B, chunk, 6, 19) == orc.md_gemm_rows(A, B, quarters=6, bits=19)).all()


@pytest.mark.parametrize("cfg_idx", [0, 1, 2])
def test_chunked_pipeline_reaches_the_tolerance_beyond_the_whole_k_budget(cfg_idx):
    """5 slices of 21 bits (105 bits >= the paper's 104): the budget k S 2^(2W) <= 2^53 allows 409 indices, so k = 1000 is
    cut into chunks of 408; every chunk's order sums are exact (int64 route == fp64 route), and the result is within
    1e-28 (|A||B|)_ij of the exact product O1."""
    cfg = inputs.CONFIGS[cfg_idx].with_shape(6, 5, 1000)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    assert 408 * 5 * 2 ** 42 <= 2 ** 53 < 1000 * 5 * 2 ** 42
    C = orc.md_gemm_rows_chunked(A, B, 408, 5, 21)
    r = orc.exact_all(A, B, C)
    assert (r["err"] <= 1e-28 * r["W"]).all()
    Aq, eA, _ = orc.split(A, 0, quarters=5, bits=21)
    Bq, eB, _ = orc.split(B, 1, quarters=5, bits=21)
    for k0 in (0, 408, 816):
        a, b = np.ascontiguousarray(Aq[:, :, k0:k0 + 408]), np.ascontiguousarray(Bq[:, k0:k0 + 408])
        assert (orc.orders_int(a, eA, b, eB, bits=21) == orc.orders_fp64(a, b)).all()

"""Pins for the oracle's order matrices C^(s) = sum_{p+q=s} A_p B_q (eq. 3-4).

Pinned against: numpy's int64 matmul on the digits (a library routine, independent of the C++ loops), exact
rationals on tiny cases, the paper's own claims (26 trailing zero bits, eq. 5 constant), and special cases
(k = 1 outer product, A = I)."""
from fractions import Fraction

import numpy as np
import pytest

from oracle import md_oracle as orc
from paper_2607_06881_b200 import inputs
from tests.exact import F
from tests.golden import load_paper_constants

PAPER = load_paper_constants()


def split_pair(cfg):
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    Aq, eA, _ = orc.split(A, 0)
    Bq, eB, _ = orc.split(B, 1)
    return A, B, Aq, eA, Bq, eB


def int_digits(Xq, exps, axis):
    Q = Xq.shape[0]
    e = exps[:, None] if axis == 0 else exps[None, :]
    D = np.stack([np.ldexp(Xq[q], -(e - 13 * (q + 1))) for q in range(Q)])
    assert (D == np.rint(D)).all()
    return D.astype(np.int64)


@pytest.mark.parametrize("cfg_idx,shape", [(0, (64, 64, 64)), (1, (40, 48, 96)), (2, (40, 48, 96)),
                                           (3, (40, 48, 96)), (4, (24, 20, 40))])
def test_integer_route_equals_fp64_route_bit_for_bit(cfg_idx, shape):
    """The paper's exactness claim: fp64 accumulation of quarter products loses no bits, so
    it must equal integer accumulation of the digits, bit for bit."""
    cfg = inputs.CONFIGS[cfg_idx].with_shape(*shape)
    _, _, Aq, eA, Bq, eB = split_pair(cfg)
    via_int, raw = orc.orders_int(Aq, eA, Bq, eB, want_raw=True)
    via_f64 = orc.orders_fp64(Aq, Bq)
    assert (via_int == via_f64).all()
    # raw integer sums against numpy's int64 matmul of the digit matrices
    DA, DB = int_digits(Aq, eA, 0), int_digits(Bq, eB, 1)
    Q = DA.shape[0]
    for s in range(Q):
        want = sum(DA[p] @ DB[s - p] for p in range(s + 1))
        assert (raw[s] == want).all()
        scale = eA[:, None].astype(np.int64) + eB[None, :] - 13 * (s + 2)
        assert (via_int[s] == np.ldexp(want.astype(np.float64), scale.astype(np.int32))).all()
    assert np.abs(raw).max() < 2 ** 53


def test_tiny_brute_force_with_rationals():
    cfg = inputs.CONFIGS[3].with_shape(5, 4, 6)
    _, _, Aq, eA, Bq, eB = split_pair(cfg)
    got = orc.orders_fp64(Aq, Bq)
    Q = Aq.shape[0]
    for s in range(Q):
        for i in range(5):
            for j in range(4):
                want = sum(F(Aq[p, i, t]) * F(Bq[s - p, t, j]) for p in range(s + 1) for t in range(6))
                assert F(got[s, i, j]) == want


def test_every_quarter_product_is_exact_with_26_trailing_zero_bits():
    """north_star check (ii) and PAPER.md:53: a product of two quarters is exact and leaves >= 26 zero bits at the
    end of the 53-bit significand (it is a <= 27-bit integer times a power of two; the paper's count ignores the hidden
    bit of the leading quarter, R1)."""
    zero_bits = PAPER["product_trailing_zero_bits"][0]
    cfg = inputs.CONFIGS[1].with_shape(16, 16, 16)
    _, _, Aq, eA, Bq, eB = split_pair(cfg)
    for p in range(8):
        for q in range(8):
            a, b = Aq[p][:, :, None], Bq[q][None, :, :]
            prod = (a * b).ravel()
            for x, y, z in zip(np.broadcast_to(a, (16, 16, 16)).ravel()[::37], np.broadcast_to(b, (16, 16, 16)).ravel()[::37], prod[::37]):
                assert F(x) * F(y) == F(z)
                if z != 0.0:
                    m = F(z).numerator  # odd part times power of two; strip the power of two
                    m = abs(m)
                    while m % 2 == 0:
                        m //= 2
                    assert m.bit_length() <= 53 - zero_bits


def test_eq5_constant_and_k_budget():
    """PAPER.md:95-99 eq. (5): N (2^26 - 1) <= 2^52 gives N <= 67,108,865."""
    assert 2 ** 52 // (2 ** 26 - 1) == PAPER["exact_sum_bound_N"][0]
    assert PAPER["exact_sum_bound_N"][0] * (2 ** 26 - 1) <= 2 ** 52 < (PAPER["exact_sum_bound_N"][0] + 1) * (2 ** 26 - 1)


def test_k_equals_one_is_an_outer_product_convolution():
    cfg = inputs.CONFIGS[0].with_shape(7, 9, 1)
    _, _, Aq, eA, Bq, eB = split_pair(cfg)
    got = orc.orders_int(Aq, eA, Bq, eB)
    for s in range(8):
        want = sum(Aq[p][:, 0][:, None] * Bq[s - p][0, :][None, :] for p in range(s + 1))  # exact in fp64: <= 30-bit sums
        assert (got[s] == want).all()


def test_identity_A_reproduces_the_quarters_of_B():
    """A = I (hi = identity, lo = 0): row max 1 -> E = 1, A_0 = I and A_p = 0 for p > 0, hence C^(s) = B_s."""
    cfg = inputs.CONFIGS[1].with_shape(32, 24, 32)
    B = inputs.generate(cfg, "B")
    A = np.zeros((2, 32, 32))
    A[0] = np.eye(32)
    Aq, eA, _ = orc.split(A, 0)
    Bq, eB, _ = orc.split(B, 1)
    assert (eA == 1).all() and (Aq[0] == np.eye(32)).all() and not Aq[1:].any()
    assert (orc.orders_int(Aq, eA, Bq, eB) == Bq).all()
    assert (orc.orders_fp64(Aq, Bq) == Bq).all()


def test_fewer_orders_than_quarters_and_more():
    cfg = inputs.CONFIGS[0].with_shape(6, 5, 8)
    _, _, Aq, eA, Bq, eB = split_pair(cfg)
    full = orc.orders_int(Aq, eA, Bq, eB, orders=15)  # all 2Q-1 orders
    assert (full[:8] == orc.orders_int(Aq, eA, Bq, eB)).all()
    assert (full == orc.orders_fp64(Aq, Bq, orders=15)).all()
    # sum over all orders == (sum of quarters of A) * (sum of quarters of B), exactly
    for i in range(6):
        for j in range(5):
            want = sum(sum(F(Aq[p, i, t]) for p in range(8)) * sum(F(Bq[q, t, j]) for q in range(8)) for t in range(8))
            assert sum(F(full[s, i, j]) for s in range(15)) == want


def test_sampled_route_equals_the_full_route():
    cfg = inputs.CONFIGS[3].with_shape(20, 18, 33)
    _, _, Aq, eA, Bq, eB = split_pair(cfg)
    full = orc.orders_int(Aq, eA, Bq, eB)
    si, sj = inputs.sample_indices(cfg, 50)
    got = orc.orders_int_samples(Aq, eA, Bq, eB, si, sj)
    assert (got == full[:, si, sj].T).all()

"""Pins of oracle part O7: Householder QR in multiple-double arithmetic (the paper's announced application;
ref [18] PAPER.md:235).  Pinned against exact rational arithmetic (residual A - QR and orthogonality Q^T Q - I evaluated in
`fractions` at n <= 8), closed forms (an upper triangular A with positive diagonal is its own R; a 3-4-5 column), numpy's
double-precision QR on the leading limbs, and the scalar operations against correctly rounded rationals."""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import md_oracle as orc
from paper_2607_06881_b200 import inputs
from tests.exact import F, round_to_limbs


def val(x):
    return sum((F(v) for v in x), Fraction(0))


@pytest.mark.parametrize("limbs", [2, 4, 8])
def test_scalar_operations_against_rationals(limbs):
    rng = np.random.default_rng(limbs)
    eps = Fraction(2) ** -(53 * limbs - 6)
    for _ in range(40):
        a = round_to_limbs(Fraction(int(rng.integers(1, 2 ** 62)), int(rng.integers(1, 2 ** 62))) * (-1) ** int(rng.integers(0, 2)), limbs)
        b = round_to_limbs(Fraction(int(rng.integers(1, 2 ** 62)), int(rng.integers(1, 2 ** 62))), limbs)
        va, vb = val(a), val(b)
        for op, want in (("add", va + vb), ("sub", va - vb), ("mul", va * vb), ("div", va / vb)):
            got = val(orc.mdx_op(op, a, b))
            assert abs(got - want) <= eps * max(abs(want), abs(va), abs(vb)), op
        r = val(orc.mdx_op("sqrt", b))
        assert abs(r * r - vb) <= 4 * eps * vb
    assert orc.mdx_op("sqrt", [25.0] + [0.0] * (limbs - 1)).tolist() == [5.0] + [0.0] * (limbs - 1)
    assert not orc.mdx_op("sqrt", [0.0] * limbs).any()


def exact_checks(A, Q, R, limbs):
    """max |A - QR|, max |Q^T Q - I| in exact rationals, relative to max |A| resp. 1."""
    L, m, n = A.shape
    Af = [[val(A[:, i, j]) for j in range(n)] for i in range(m)]
    Qf = [[val(Q[:, i, j]) for j in range(n)] for i in range(m)]
    Rf = [[val(R[:, i, j]) for j in range(n)] for i in range(n)]
    amax = max(abs(v) for row in Af for v in row)
    res = max(abs(Af[i][j] - sum(Qf[i][t] * Rf[t][j] for t in range(n))) for i in range(m) for j in range(n))
    orth = max(abs(sum(Qf[t][i] * Qf[t][j] for t in range(m)) - (1 if i == j else 0)) for i in range(n) for j in range(n))
    return res / amax, orth


@pytest.mark.parametrize("cfg_idx,shape", [(0, (8, 8)), (3, (8, 6)), (4, (7, 7)), (1, (5, 3)), (5, (6, 4)), (2, (1, 1))])
def test_qr_residual_and_orthogonality_in_exact_arithmetic(cfg_idx, shape):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(shape[0], 3, shape[1])
    A = inputs.generate(cfg, "A")
    L = cfg.limbs
    Q, R = orc.md_qr(A)
    res, orth = exact_checks(A, Q, R, L)
    bar = shape[0] * Fraction(2) ** -(53 * L - 8)
    assert res <= bar and orth <= bar, (float(res), float(orth), float(bar))
    assert not np.tril(R[0], -1).any() and all(not np.tril(R[l], -1).any() for l in range(L))   # upper triangular
    assert (np.diagonal(R[0]) >= 0).all()                                                          # the sign convention
    # the leading limbs against the library routine in double precision (same sign convention)
    q, r = np.linalg.qr(A.sum(axis=0))
    sgn = np.sign(np.diagonal(r))
    sgn[sgn == 0] = 1
    scale = np.abs(A[0]).max()
    kappa = np.linalg.cond(A.sum(axis=0))
    assert np.abs(Q[0] - q * sgn[None, :]).max() <= 1e-13 * kappa and np.abs(R[0] - r * sgn[:, None]).max() <= 1e-13 * scale * kappa


def test_qr_closed_forms():
    # an upper triangular A with positive diagonal: Q = I, R = A, exactly (every reflection is the identity)
    rng = np.random.default_rng(5)
    A = np.zeros((2, 6, 6))
    A[0] = np.triu(rng.standard_normal((6, 6)))
    A[0][np.diag_indices(6)] = np.abs(np.diagonal(A[0])) + 1.0
    A[1] = A[0] * 2.0 ** -55 * np.triu(rng.uniform(-1, 1, (6, 6)))
    Q, R = orc.md_qr(A)
    assert (R == A).all() and (Q[0] == np.eye(6)).all() and not Q[1].any()
    # negative diagonal entry: the sign moves into Q
    A2 = A.copy()
    A2[:, 2, :] = -A2[:, 2, :]
    Q2, R2 = orc.md_qr(A2)
    assert (R2 == A).all() and Q2[0, 2, 2] == -1.0
    # the 3-4-5 column: R_11 = 5 exactly, Q = (3/5, 4/5) to full precision
    A3 = np.zeros((2, 2, 1))
    A3[0, :, 0] = [3.0, 4.0]
    Q3, R3 = orc.md_qr(A3)
    assert R3[0, 0, 0] == 5.0 and R3[1, 0, 0] == 0.0
    assert abs(val(Q3[:, 0, 0]) - Fraction(3, 5)) <= Fraction(2) ** -104 and abs(val(Q3[:, 1, 0]) - Fraction(4, 5)) <= Fraction(2) ** -104
    # orthogonal input: R = I up to rounding
    c, s_ = Fraction(3, 5), Fraction(4, 5)
    A4 = np.zeros((2, 2, 2))
    for (i, j), v in {(0, 0): c, (0, 1): -s_, (1, 0): s_, (1, 1): c}.items():
        A4[:, i, j] = round_to_limbs(v, 2)
    Q4, R4 = orc.md_qr(A4)
    assert abs(val(R4[:, 0, 0]) - 1) <= Fraction(2) ** -100 and abs(val(R4[:, 0, 1])) <= Fraction(2) ** -100

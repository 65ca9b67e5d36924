"""Pins for the oracle on the two wider formats of the paper's Table 2: octo double (8 limbs, 32
quarters) and hexa double (16 limbs, 64 quarters) -- SURVEY.md section 8(f) next-1.

The oracle's code is generic in `limbs`; these tests pin it at L = 8, 16 the same way the L = 2, 4 tests do: exact rational
arithmetic (tests/exact.py), numpy's int64 matmul on the digits, the Table 2 dimensions the paper prints
(tests/golden/paper_constants.txt), and the tolerance DESIGN.md section 3 R13 derives for these formats."""
from fractions import Fraction

import numpy as np
import pytest

from oracle import md_oracle as orc
from paper_2607_06881_b200 import inputs
from tests.exact import F, nearest_digits, round_to_limbs
from tests.golden import load_paper_constants

PAPER = load_paper_constants()
WIDE = [5, 6]                       # inputs.CONFIGS indices: od_1024, hd_512
TOL = {8: 1e-120, 16: 1e-245}       # DESIGN.md R13: 2^-(52 L - 18), rounded down to a power of ten


def test_table2_dimensions_are_the_quarter_counts():
    """PAPER.md:196-205 Table 2: the top-down 8192 x 4096 double matrix represents a (8192/Q) x (4096/Q) md matrix with
    Q = 4 * limbs quarters per element: dd 1024 x 512, qd 512 x 256, od 256 x 128, hd 128 x 64."""
    rows, cols = PAPER["table2_rows_A"], PAPER["table2_cols_A"]  # d dd qd od hd
    for t, limbs in enumerate((2, 4, 8, 16), start=1):
        assert (rows[0] // (4 * limbs), cols[0] // (4 * limbs)) == (rows[t], cols[t])
    assert [inputs.CONFIGS[i].quarters for i in WIDE] == [32, 64]
    assert [inputs.CONFIGS[i].products for i in WIDE] == [528, 2080]


@pytest.mark.parametrize("cfg_idx", WIDE)
@pytest.mark.parametrize("axis", [0, 1])
def test_sum_of_quarters_plus_remainder_is_exact(cfg_idx, axis):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(7, 6, 9)
    X = inputs.generate(cfg, "A" if axis == 0 else "B")
    qp, exps, rem = orc.split(X, axis, want_remainder=True)
    L, rows, cols = X.shape
    Q = qp.shape[0]
    assert Q == 4 * L
    for i in range(rows):
        for j in range(cols):
            E = int(exps[i] if axis == 0 else exps[j])
            elt = sum(F(X[l, i, j]) for l in range(L))
            rho = sum(F(rem[l, i, j]) for l in range(L))
            assert sum(F(qp[q, i, j]) for q in range(Q)) + rho == elt
            assert abs(rho) <= Fraction(2) ** (E - 13 * Q) * Fraction(1025, 2048)
            # digits: on the grid, bounded, and equal to the exact nearest expansion away from near-ties
            D = []
            for q in range(Q):
                v = F(qp[q, i, j]) / Fraction(2) ** (E - 13 * (q + 1))
                assert v.denominator == 1 and abs(v) <= (2 ** 13 if q == 0 else 2 ** 12)
                D.append(int(v))
            want, _, margin = nearest_digits(elt, E, Q)
            if margin == 0 or margin > Fraction(1, 2 ** 30):
                assert D == want


def test_hand_derived_wide_case():
    """x = 1 - 2^-400 as an octo double (1, -2^-400, 0, ...) in a row whose maximum is 1: E = 1, u_q = 2^(1-13(q+1)).
    1 = 4096 u_0.  -2^-400: u_30 = 2^(1-403) = 2^-402, so -2^-400 = -4 u_30.  Problem 3.3 of the paper (PAPER.md:124,
    hi > 0, lo < 0) across 30 quarters: the low limb just contributes a digit of its own sign."""
    X = np.zeros((8, 1, 2))
    X[0, 0] = [1.0, 0.5]
    X[1, 0, 0] = -(2.0 ** -400)
    qp, exps, rem = orc.split(X, 0, want_remainder=True)
    assert int(exps[0]) == 1 and not rem.any()
    D = [int(F(qp[q, 0, 0]) / Fraction(2) ** (1 - 13 * (q + 1))) for q in range(32)]
    assert D == [4096] + [0] * 29 + [-4, 0]


@pytest.mark.parametrize("cfg_idx,shape", [(5, (10, 9, 40)), (6, (6, 5, 24))])
def test_integer_route_equals_fp64_route_and_numpy_matmul(cfg_idx, shape):
    """accumulation of quarter products is exact -> fp64 route == int64 route == numpy int matmul."""
    cfg = inputs.CONFIGS[cfg_idx].with_shape(*shape)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    Aq, eA, _ = orc.split(A, 0)
    Bq, eB, _ = orc.split(B, 1)
    via_int, raw = orc.orders_int(Aq, eA, Bq, eB, want_raw=True)
    assert (via_int == orc.orders_fp64(Aq, Bq)).all()
    Q = cfg.quarters
    DA = np.stack([np.ldexp(Aq[q], -(eA[:, None] - 13 * (q + 1))) for q in range(Q)]).astype(np.int64)
    DB = np.stack([np.ldexp(Bq[q], -(eB[None, :] - 13 * (q + 1))) for q in range(Q)]).astype(np.int64)
    for s in range(Q):
        want = sum(DA[p] @ DB[s - p] for p in range(s + 1))
        assert (raw[s] == want).all()
        scale = (eA[:, None].astype(np.int64) + eB[None, :] - 13 * (s + 2)).astype(np.int32)
        assert (via_int[s] == np.ldexp(want.astype(np.float64), scale)).all()
    assert np.abs(raw).max() < 2 ** 53


@pytest.mark.parametrize("limbs", [8, 16])
def test_renorm_is_the_exact_sum_rounded_limb_by_limb(limbs):
    rng = np.random.default_rng(limbs)
    S = 4 * limbs
    ord_planes = np.stack([np.ldexp(rng.integers(-2 ** 40, 2 ** 40, (3, 4)).astype(np.float64), -13 * (s + 2))
                           for s in range(S)])
    C = orc.renorm(ord_planes, limbs)
    for i in range(3):
        for j in range(4):
            want = round_to_limbs(sum(F(ord_planes[s, i, j]) for s in range(S)), limbs)
            assert [C[l, i, j] for l in range(limbs)] == want


@pytest.mark.parametrize("cfg_idx", WIDE)
def test_exact_samples_against_rationals(cfg_idx):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(4, 3, 5)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    L = cfg.limbs
    r = orc.exact_all(A, B, out_limbs=L + 1)
    for i in range(4):
        for j in range(3):
            tot = sum(sum(F(A[l, i, t]) for l in range(L)) * sum(F(B[l, t, j]) for l in range(L)) for t in range(5))
            w = sum(abs(sum(F(A[l, i, t]) for l in range(L))) * abs(sum(F(B[l, t, j]) for l in range(L))) for t in range(5))
            assert list(r["exact"][i, j]) == round_to_limbs(tot, L + 1)
            assert r["W"][i, j] == float(w)


@pytest.mark.parametrize("cfg_idx,shape", [(5, (12, 12, 96)), (6, (8, 8, 64))])
def test_five_step_pipeline_reaches_the_derived_tolerance(cfg_idx, shape):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(*shape)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    C = orc.md_gemm_rows(A, B)
    r = orc.exact_all(A, B, C)
    assert (r["err"] <= TOL[cfg.limbs] * r["W"]).all(), float((r["err"] / r["W"]).max())
    _, eA, _ = orc.split(A, 0)
    _, eB, _ = orc.split(B, 1)
    Q = cfg.quarters  # the any-input bound of DESIGN.md R5
    bound = cfg.k * (Q + 3) * np.ldexp(1.0, (eA[:, None] + eB[None, :] - 13 * Q - 2).astype(np.int32))
    assert (r["err"] <= bound + np.abs(C[0]) * 2.0 ** (-53 * cfg.limbs + 1)).all()
    for l in range(cfg.limbs - 1):
        assert (np.abs(C[l + 1]) <= np.spacing(np.abs(C[l])) / 2).all()
    # north_star check (iv): the classical md GEMM agrees to its own working precision
    Cc = orc.classic_gemm(A, B)
    rc = orc.exact_all(A, B, Cc)
    assert (rc["err"] <= 4 * cfg.k * 2.0 ** -(53 * cfg.limbs - 2) * rc["W"]).all()

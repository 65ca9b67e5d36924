"""Pins for the oracle's recombination (O4), exact product (O1), classical md GEMM (O5) and the
five-step pipeline -- against exact rationals, numpy integer matmul, textbook TwoSum, and the
tolerance BASELINE.json north_star states."""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import md_oracle as orc
from paper_2607_06881_b200 import inputs
from tests.exact import F, round_to_limbs
from tests.golden import load_paper_constants

TOL = {2: 1e-28, 4: 1e-58}  # BASELINE.json north_star: |C - C_exact|_ij <= TOL * (|A||B|)_ij


def exact_product_fraction(A, B, i, j):
    L, _, k = A.shape
    tot, w = Fraction(0), Fraction(0)
    for t in range(k):
        a = sum(F(A[l, i, t]) for l in range(L))
        b = sum(F(B[l, t, j]) for l in range(L))
        tot += a * b
        w += abs(a) * abs(b)
    return tot, w


# ---------------------------------------------------------------- O4
@pytest.mark.parametrize("limbs", [2, 4])
def test_renorm_is_the_exact_sum_rounded_limb_by_limb(limbs):
    rng = np.random.default_rng(limbs)
    S = 4 * limbs
    ord_planes = np.stack([np.ldexp(rng.integers(-2 ** 40, 2 ** 40, (6, 5)).astype(np.float64), -13 * (s + 2))
                           for s in range(S)])
    C = orc.renorm(ord_planes, limbs)
    for i in range(6):
        for j in range(5):
            want = round_to_limbs(sum(F(ord_planes[s, i, j]) for s in range(S)), limbs)
            assert [C[l, i, j] for l in range(limbs)] == want
            for l in range(limbs - 1):  # Definition 1.1: non-overlapping
                assert abs(C[l + 1, i, j]) <= math.ulp(C[l, i, j]) / 2


def test_renorm_special_cases():
    x = np.array([[[1.0, -2.5, 0.0]]])
    assert (orc.renorm(x, 2) == np.array([[[1.0, -2.5, 0.0]], [[0.0, 0.0, 0.0]]])).all()  # S = 1: a copy
    a, b = 1.0, 2.0 ** -70 + 2.0 ** -100
    C = orc.renorm(np.array([[[a]], [[b]]]), 2)  # S = 2: TwoSum by definition: hi = fl(a+b), lo = a+b-hi
    assert C[0, 0, 0] == a + b and F(C[1, 0, 0]) == F(a) + F(b) - F(a + b)


# ---------------------------------------------------------------- O1
@pytest.mark.parametrize("cfg_idx", [0, 3, 4])
def test_exact_samples_against_rationals(cfg_idx):
    """north_star check (iii): tiny-n brute force in exact rational arithmetic."""
    cfg = inputs.CONFIGS[cfg_idx].with_shape(6, 5, 9)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    L = cfg.limbs
    rng = np.random.default_rng(0)
    C = rng.uniform(-1, 1, (L, 6, 5)) * np.array([2.0 ** (-53 * l) for l in range(L)])[:, None, None]
    r = orc.exact_all(A, B, C, out_limbs=L + 1)
    for i in range(6):
        for j in range(5):
            tot, w = exact_product_fraction(A, B, i, j)
            assert list(r["exact"][i, j]) == round_to_limbs(tot, L + 1)
            assert r["W"][i, j] == float(w)
            assert r["err"][i, j] == float(abs(sum(F(C[l, i, j]) for l in range(L)) - tot))


def test_exact_product_of_small_integer_matrices_is_numpy_int_matmul():
    rng = np.random.default_rng(1)
    Ai, Bi = rng.integers(-2 ** 20, 2 ** 20, (9, 17)), rng.integers(-2 ** 20, 2 ** 20, (17, 8))
    A, B = np.zeros((2, 9, 17)), np.zeros((2, 17, 8))
    A[0], B[0] = Ai, Bi
    r = orc.exact_all(A, B, out_limbs=2)
    assert (r["exact"][..., 0] == (Ai @ Bi).astype(np.float64)).all() and not r["exact"][..., 1].any()
    assert (r["W"] == (np.abs(Ai) @ np.abs(Bi)).astype(np.float64)).all()


# ---------------------------------------------------------------- pipeline and O5
@pytest.mark.parametrize("cfg_idx,shape", [(0, (64, 64, 64)), (1, (24, 24, 200)), (2, (24, 24, 200)),
                                           (3, (32, 32, 128)), (4, (16, 16, 64))])
def test_five_step_pipeline_reaches_the_stated_tolerance(cfg_idx, shape):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(*shape)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    C = orc.md_gemm_rows(A, B, quarters=cfg.quarters)  # 4 per limb, 9 for config 3 (R5)
    r = orc.exact_all(A, B, C)
    assert (r["err"] <= TOL[cfg.limbs] * r["W"]).all(), float((r["err"] / r["W"]).max())
    for l in range(cfg.limbs - 1):
        assert (np.abs(C[l + 1]) <= np.spacing(np.abs(C[l])) / 2).all()


@pytest.mark.parametrize("cfg_idx,Q", [(0, 8), (3, 8), (3, 9), (4, 16)])
def test_error_bound_relative_to_the_group_exponents(cfg_idx, Q):
    """What the common-exponent reading guarantees for ANY input (R5): per (i,j,k) the neglected part is
    rho_a*b + a*rho_b + sum_{p+q>=Q} a_p b_q, at most (Q+3) * 2^(E_i+F_j-13Q-2) in magnitude (2 + (Q-1) + 2 units: DESIGN.md R5), so
    |C - C_exact|_ij <= k (Q+3) 2^(E_i + F_j - 13 Q - 2) (+ the final rounding).  Relative to (|A||B|)_ij this can
    exceed 1e-28 when (|A||B|)_ij << 2^(E_i+F_j): config 3's distribution at Q = 8 is the example."""
    cfg = inputs.CONFIGS[cfg_idx].with_shape(32, 32, 128)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    C = orc.md_gemm_rows(A, B, quarters=Q)
    _, eA, _ = orc.split(A, 0)
    _, eB, _ = orc.split(B, 1)
    r = orc.exact_all(A, B, C)
    bound = cfg.k * (Q + 3) * np.ldexp(1.0, (eA[:, None] + eB[None, :] - 13 * Q - 2).astype(np.int32))
    bound = bound + np.abs(C[0]) * 2.0 ** (-53 * cfg.limbs + 1)
    assert (r["err"] <= bound).all()


@pytest.mark.parametrize("cfg_idx,shape", [(0, (48, 40, 64)), (3, (24, 24, 96)), (4, (16, 12, 48))])
def test_classical_md_gemm_agrees_to_working_precision(cfg_idx, shape):
    """north_star check (iv) / the paper's own validation (eq. 9): quarter path vs a classical
    multiple-double GEMM.  Threshold 4k * 2^-(53L-2) * W: the classical product's own error bound."""
    cfg = inputs.CONFIGS[cfg_idx].with_shape(*shape)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    Cc = orc.classic_gemm(A, B)
    r = orc.exact_all(A, B, Cc)
    thr = 4 * cfg.k * 2.0 ** -(53 * cfg.limbs - 2)
    assert (r["err"] <= thr * r["W"]).all(), float((r["err"] / r["W"]).max() / thr)
    Cq = orc.md_gemm_rows(A, B, quarters=cfg.quarters)
    diff = np.abs(sum((Cq[l] - Cc[l]) for l in reversed(range(cfg.limbs))))
    assert (diff <= 2 * thr * r["W"]).all()


def test_eps_max_has_the_papers_order_of_magnitude():
    """PAPER.md:188 (Table 1): eps_max = 3.5e-28 at n = 1024 (dd), growing with n.  Inputs differ (unspecified
    in the paper), so only the order of magnitude is a sanity check: at n = 96 it must be well below 3.5e-28 * 10."""
    paper = load_paper_constants()["eps_max_dd"][0]
    cfg = inputs.CONFIGS[0].with_shape(96, 96, 96)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    Cq, Cc = orc.md_gemm_rows(A, B), orc.classic_gemm(A, B)
    eps = np.abs((Cq[0] - Cc[0]) + (Cq[1] - Cc[1])).max()
    assert eps < 10 * paper


def test_identity_and_integer_products_are_exact():
    cfg = inputs.CONFIGS[0].with_shape(16, 16, 16)
    B = inputs.generate(cfg, "B")
    A = np.zeros((2, 16, 16))
    A[0] = np.eye(16)
    C = orc.md_gemm_rows(A, B)
    # C = B up to the remainder of B's split: |rho| <= 2^(F_j - 104) / 2 * (1 + 2^-27)
    _, eB, _ = orc.split(B, 1)
    assert (np.abs((C[0] - B[0]) + (C[1] - B[1])) <= np.ldexp(1.0, eB - 104)[None, :]).all()
    rng = np.random.default_rng(2)
    Ai, Bi = rng.integers(-2 ** 20, 2 ** 20, (12, 30)), rng.integers(-2 ** 20, 2 ** 20, (30, 10))
    A, B = np.zeros((2, 12, 30)), np.zeros((2, 30, 10))
    A[0], B[0] = Ai, Bi
    C = orc.md_gemm_rows(A, B)
    assert (C[0] == (Ai @ Bi).astype(np.float64)).all() and not C[1].any()

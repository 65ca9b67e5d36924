"""GPU parity of md_plan_quarters (include/mdgemm.h; R15) against the oracle's plan.  The spread D is an
integer decided by fp64 sums whose rounding depends on the summation order, so D may differ by one where a sum sits on a
power of two (several results are valid); what is unique is checked exactly (Q is the smallest count for the D the GPU
measured), and the plan is checked for what it promises: with it md_gemm is inside the tolerance at every position."""
import numpy as np
import pytest
import torch

from oracle import md_oracle as orc
from paper_2607_06881_b200 import binding as md
from paper_2607_06881_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = {2: 1e-28, 4: 1e-58, 8: 1e-120, 16: 1e-245}


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def smallest_Q(k, limbs, bits, D, tol):
    Q = -(-(52 * limbs) // bits)
    while k * (Q + 3) * 2.0 ** (D - bits * Q - 2) > tol:
        Q += 1
    return Q


@pytest.mark.parametrize("cfg_idx,shape", [(0, (64, 64, 64)), (1, (150, 70, 90)), (2, (37, 51, 77)), (3, (96, 80, 200)),
                                           (4, (70, 45, 91)), (3, (1, 1, 1)), (5, (40, 30, 20)), (6, (20, 10, 12))])
def test_plan_matches_oracle(cfg_idx, shape):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(*shape)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    Q, D = md.md_plan_quarters(dev(A), dev(B))
    Qo, Do = orc.plan_quarters(A, B, TOL[cfg.limbs])
    assert abs(D - Do) <= 1
    assert Q == smallest_Q(cfg.k, cfg.limbs, 13, D, TOL[cfg.limbs])
    if D == Do:
        assert Q == Qo


def test_plan_with_wide_slices_and_explicit_tolerance():
    cfg = inputs.CONFIGS[3].with_shape(64, 64, 128)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    md.md_set_option(md.MD_OPT_SLICE_BITS, 19)
    try:
        Q, D = md.md_plan_quarters(dev(A), dev(B), 1e-25)
    finally:
        md.md_set_option(md.MD_OPT_SLICE_BITS, 0)
    Qo, Do = orc.plan_quarters(A, B, 1e-25, bits=19)
    assert abs(D - Do) <= 1 and Q == smallest_Q(cfg.k, 2, 19, D, 1e-25)


def test_zero_product_needs_the_minimum():
    Q, D = md.md_plan_quarters(torch.zeros((2, 5, 7), dtype=torch.float64, device="cuda"),
                               torch.zeros((2, 7, 3), dtype=torch.float64, device="cuda"))
    assert (Q, D) == (8, -2 ** 31)


def test_planned_count_delivers_the_tolerance_on_the_wide_range_input():
    """Config 3's distribution at k = 256: the paper's 8 quarters miss 1e-28 (|A||B|)_ij at ~100 positions (by up to 49x),
    the planned count (10, which has a kernel) misses none."""
    cfg = inputs.CONFIGS[3].with_shape(96, 80, 256)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    Q, D = md.md_plan_quarters(dev(A), dev(B))
    assert Q == 10 and 14 <= D <= 16, (Q, D)
    with md.Workspace(cfg.m, cfg.n, cfg.k, 2, 8):
        r8 = orc.exact_all(A, B, md.md_gemm(dev(A), dev(B)).cpu().numpy())
    assert (r8["err"] > 1e-28 * r8["W"]).any()
    with md.Workspace(cfg.m, cfg.n, cfg.k, 2, Q):
        rq = orc.exact_all(A, B, md.md_gemm(dev(A), dev(B)).cpu().numpy())
    assert (rq["err"] <= 1e-28 * rq["W"]).all()


def test_full_size_config3_plan():
    """BASELINE.json configs[3] (8192 x 8192 x 2048, "stresses balancing/quarter count"): the count bench.py runs it with
    (inputs.CONFIGS[3].quarters = 9) against the any-input guarantee of the plan."""
    cfg = inputs.CONFIGS[3]
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    Q, D = md.md_plan_quarters(dev(A), dev(B))
    print(f"cfg3 full size: D = {D}, guaranteed Q = {Q} (run with {cfg.quarters})")
    assert cfg.quarters <= Q <= cfg.quarters + 1

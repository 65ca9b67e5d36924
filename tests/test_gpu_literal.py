"""GPU parity of the paper's own section-3 balancing (R17-R22; include/mdgemm.h md_split_literal,
md_gemm_literal) against oracle part O6: Algorithm L bit-exact (parts and per-element exponents), the exponent-class product
equal to the oracle's up to the recombination (R9) and inside 1e-28 (|A||B|)_ij on cfg3's wide-range distribution
WITH THE PAPER'S 8 QUARTERS -- where the row / column grid of md_gemm needs 9 or 10."""
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


def host(t):
    return t.cpu().numpy()


@pytest.mark.parametrize("cfg_idx", [0, 1, 2, 3, 4, 5, 6])
@pytest.mark.parametrize("shape", [(64, 64), (37, 77), (1, 1), (3, 500)])
@pytest.mark.parametrize("eq8", [True, False])
def test_split_literal_bit_exact(cfg_idx, shape, eq8):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(shape[0], 5, shape[1])
    X = inputs.generate(cfg, "A")
    X[:, 0, 0] = 0.0
    for Q in (4 * cfg.limbs, 4 * cfg.limbs + 1):
        qp, exps = md.md_split_literal(dev(X), Q, 0 if eq8 else md.MD_LITERAL_NO_EQ8)
        want_q, want_e, _ = orc.split_literal(X, Q, eq8)
        assert (host(exps) == want_e).all()
        assert bool((host(qp) == want_q).all())


def test_split_literal_worked_cases_of_the_paper_on_gpu():
    """PAPER.md:124-131 (x_h = 1, x_l = -2^-60) and PAPER.md:133-140 (x_1 with twelve leading zeros: b = 2^-14)."""
    hi = np.array([[1.0, 1.0 + 2.0 ** -26, -1.0, 0.0]])
    lo = np.array([[-(2.0 ** -60), 0.0, 2.0 ** -60, 0.0]])
    qp, exps = md.md_split_literal(dev(np.stack([hi, lo])), 8)
    q, e = host(qp)[:, 0, :], host(exps)[0]
    assert e.tolist() == [-1, 0, -1, 0]
    assert q[0, 1] == 1.0 - 2.0 ** -14 and q[1, 1] == 2.0 ** -14 + 2.0 ** -26 and not q[2:, 1].any()   # eq. (8), zero rule
    assert (q[:, 0] >= 0).all() and q[:, 0].sum() == 1.0 - 2.0 ** -60                                    # eq. (7): one sign
    assert (q[:, 2] == -q[:, 0]).all() and not q[:, 3].any()


@pytest.mark.parametrize("cfg_idx,shape", [(3, (70, 45, 52)), (0, (64, 64, 64)), (1, (37, 51, 77)), (2, (33, 20, 40)), (4, (20, 17, 33)),
                                           (3, (1, 1, 1)), (3, (150, 70, 9))])
@pytest.mark.parametrize("flags", [0, md.MD_LITERAL_NO_EQ8, md.MD_LITERAL_SIGN_GROUPS])
def test_literal_product_against_the_oracle_and_the_exact_product(cfg_idx, shape, flags):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(*shape)
    L = cfg.limbs
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    C, info = md.md_gemm_literal(dev(A), dev(B), flags=flags)
    C = host(C)
    want, oinfo = orc.md_gemm_literal(A, B, 4 * L, not (flags & md.MD_LITERAL_NO_EQ8), bool(flags & md.MD_LITERAL_SIGN_GROUPS))
    assert (info["zminA"], info["zmaxA"], info["zminB"], info["zmaxB"]) == oinfo
    spanA, spanB = oinfo[1] - oinfo[0], oinfo[3] - oinfo[2]
    assert info["planes"] == 4 * L + max(spanA, spanB) and info["orders"] == 4 * L + spanA + spanB and info["pairs"] >= 1
    r = orc.exact_all(A, B, C)
    assert (r["err"] <= TOL[L] * r["W"]).all()                      # the paper's quarter count, any dynamic range
    # against the oracle's own (exactly summed, correctly rounded) result: the recombination's slack, relative to |A||B|
    assert (np.abs((C - want).sum(axis=0)) <= np.ldexp(r["W"], -(53 * L - 8))).all()
    if cfg_idx == 3 and cfg.k >= 40:
        with md.Workspace(cfg.m, cfg.n, cfg.k, 2, 8):               # the row / column grid with the same 8 quarters misses it
            r8 = orc.exact_all(A, B, host(md.md_gemm(dev(A), dev(B))))
        assert (r8["err"] > 1e-28 * r8["W"]).any()


def test_literal_product_errors_and_limits():
    cfg = inputs.CONFIGS[3].with_shape(16, 16, 16)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    A2 = A * np.ldexp(1.0, np.where(np.arange(16)[None, :] % 2 == 0, 150, -150))[None]   # levels spanning far more than 8
    with pytest.raises(md.MdError) as e:
        md.md_gemm_literal(dev(A2), dev(B))
    assert e.value.status == md.MD_ERR_UNSUPPORTED
    lib = md.lib()
    assert lib.md_literal_scratch_bytes(0, 4, 4, 2, 0, 0) == 0 and lib.md_literal_scratch_bytes(4, 4, 4, 3, 0, 0) == 0
    assert lib.md_gemm_literal(4, 4, 4, 2, None, None, None, None, 0, 0, None, None) == md.MD_ERR_BAD_ARG
    assert lib.md_split_literal(4, 4, 3, 8, 0, None, None, None, None) == md.MD_ERR_BAD_ARG
    # zero operands
    Z = torch.zeros((2, 5, 6), dtype=torch.float64, device="cuda")
    C, info = md.md_gemm_literal(Z, dev(inputs.generate(cfg.with_shape(6, 4, 4), "A")))
    assert not host(C).any() and info["pairs"] == 0

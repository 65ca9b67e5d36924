"""GPU parity for the wider formats of the paper's Table 2: octo double
(8 limbs, 32 quarters, T = 528) and hexa double (16 limbs, 64 quarters, T = 2080) through qgemm_wide.cu.

Same bars as tests/test_gpu_parity.py: split and order matrices BIT-EXACT against the oracle; md_renorm within
2^-(53L-3) sum_s|C^(s)| of the oracle's correctly rounded sum; final C within 1e-120 (od) / 1e-245 (hd) of the exact product
relative to (|A||B|)_ij (R13 derives these; the paper and north_star state none for od / hd); the fused epilogue
(for hd a chain over four warps) equal to the standalone md_renorm bit for bit.
Sizes span several CTA tiles (32x16 od, 16x8 hd) with ragged tails in m, n, k, and more tiles than SMs (stream-K tail)."""
import numpy as np
import pytest
import torch

from oracle import md_oracle as orc
from paper_2607_06881_b200 import binding as md
from paper_2607_06881_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = {8: 1e-120, 16: 1e-245}
WIDE = [5, 6]


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def host(t):
    return t.cpu().numpy()


def gen(cfg_idx, m, n, k):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(m, n, k)
    return cfg, inputs.generate(cfg, "A"), inputs.generate(cfg, "B")


@pytest.mark.parametrize("cfg_idx", WIDE)
@pytest.mark.parametrize("shape", [(64, 64), (37, 77), (1, 1), (3, 200), (200, 3)])
@pytest.mark.parametrize("axis", [0, 1])
def test_split_bit_exact(cfg_idx, shape, axis):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(shape[0], 5, shape[1])
    X = inputs.generate(cfg, "A")
    qp, exps = md.md_split(dev(X), axis, cfg.quarters)
    want_q, want_e, _ = orc.split(X, axis, cfg.quarters)
    assert (host(exps) == want_e).all()
    assert bool((host(qp) == want_q).all())


def test_split_hand_derived_wide_case_on_gpu():
    """x = 1 - 2^-400 as an octo double: D = [4096, 0 x 29, -4, 0] (tests/test_oracle_wide.py derives it)."""
    X = np.zeros((8, 1, 2))
    X[0, 0] = [1.0, 0.5]
    X[1, 0, 0] = -(2.0 ** -400)
    qp, exps = md.md_split(dev(X), 0, 32)
    assert int(host(exps)[0]) == 1
    D = [float(np.ldexp(host(qp)[q, 0, 0], -(1 - 13 * (q + 1)))) for q in range(32)]
    assert D == [4096.0] + [0.0] * 29 + [-4.0, 0.0]


SHAPES = [(64, 64, 64), (70, 45, 52), (33, 17, 9), (8, 8, 4), (1, 1, 1), (130, 190, 36)]


@pytest.mark.parametrize("cfg_idx", WIDE)
@pytest.mark.parametrize("shape", SHAPES)
def test_order_matrices_bit_exact(cfg_idx, shape):
    cfg, A, B = gen(cfg_idx, *shape)
    with md.Workspace(cfg.m, cfg.n, cfg.k, cfg.limbs, cfg.quarters):
        got = host(md.md_gemm_orders(dev(A), dev(B)))
        assert md.md_read_flags() == 0
    Aq, eA, _ = orc.split(A, 0, cfg.quarters)
    Bq, eB, _ = orc.split(B, 1, cfg.quarters)
    want = orc.orders_int(Aq, eA, Bq, eB)
    assert got.shape == want.shape and bool((got == want).all())


@pytest.mark.parametrize("cfg_idx", WIDE)
@pytest.mark.parametrize("shape", [(64, 64, 64), (70, 45, 52), (130, 190, 36)])
def test_gemm_within_derived_tolerance_and_equal_to_standalone_renorm(cfg_idx, shape):
    cfg, A, B = gen(cfg_idx, *shape)
    L = cfg.limbs
    with md.Workspace(cfg.m, cfg.n, cfg.k, L, cfg.quarters):
        dA, dB = dev(A), dev(B)
        C = host(md.md_gemm(dA, dB))
        orders = md.md_gemm_orders(dA, dB)
        assert md.md_read_flags() == 0
    # the fused epilogue (hd: accumulator chained through four warps) == the standalone md_renorm, bit for bit
    assert bool((C == host(md.md_renorm(orders, L))).all())
    r = orc.exact_all(A, B, C)
    assert (r["err"] <= TOL[L] * r["W"]).all(), float((r["err"] / r["W"]).max())
    for l in range(L - 1):  # Definition 1.1: non-overlapping
        assert (np.abs(C[l + 1]) <= np.spacing(np.abs(C[l])) / 2).all()
    Co = orc.md_gemm_rows(A, B)  # the oracle's own five-step result, up to the last limb's rounding
    assert bool((C[: L - 1] == Co[: L - 1]).all())


@pytest.mark.parametrize("limbs", [8, 16])
def test_renorm_against_oracle(limbs):
    cfg, A, B = gen(5 if limbs == 8 else 6, 30, 26, 40)
    Aq, eA, _ = orc.split(A, 0)
    Bq, eB, _ = orc.split(B, 1)
    ord_planes = orc.orders_int(Aq, eA, Bq, eB)
    got = host(md.md_renorm(dev(ord_planes), limbs))
    want = orc.renorm(ord_planes, limbs)
    diff = np.abs(sum((got[l] - want[l]) for l in reversed(range(limbs))))
    assert (diff <= 2.0 ** -(53 * limbs - 3) * np.abs(ord_planes).sum(axis=0)).all()
    assert bool((got[: limbs - 1] == want[: limbs - 1]).all())


@pytest.mark.parametrize("cfg_idx", WIDE)
def test_identity_and_small_integer_products(cfg_idx):
    cfg = inputs.CONFIGS[cfg_idx]
    L = cfg.limbs
    rng = np.random.default_rng(cfg_idx)
    Ai, Bi = rng.integers(-2 ** 20, 2 ** 20, (40, 50)), rng.integers(-2 ** 20, 2 ** 20, (50, 30))
    A, B = np.zeros((L, 40, 50)), np.zeros((L, 50, 30))
    A[0], B[0] = Ai, Bi
    with md.Workspace(40, 30, 50, L):
        C = host(md.md_gemm(dev(A), dev(B)))
    assert bool((C[0] == (Ai @ Bi).astype(np.float64)).all()) and not C[1:].any()
    # A = I: the order matrices reproduce the quarter planes of B (A_0 = I on the grid E = 1, A_p = 0 for p > 0)
    _, _, Bm = gen(cfg_idx, 48, 20, 48)
    I = np.zeros((L, 48, 48))
    I[0] = np.eye(48)
    with md.Workspace(48, 20, 48, L):
        got = host(md.md_gemm_orders(dev(I), dev(Bm)))
    assert bool((got == orc.split(Bm, 1)[0]).all())


@pytest.mark.parametrize("cfg_idx", WIDE)
def test_recombination_when_only_some_lanes_carry_something(cfg_idx):
    """The recombination of the wide formats stops a TwoSum cascade once EVERY lane of the warp carries zero (renorm_add2).  Rows
    of zeros, rows with a single power of two and exactly cancelling pairs next to dense rows put lanes that carry nothing beside
    lanes that do, in one 8 x 8 tile: the fused result must still equal the standalone md_renorm of the dumped orders bit for bit
    (which adds every order through the whole cascade) and meet the tolerance against the exact product."""
    cfg, A, B = gen(cfg_idx, 40, 24, 36)
    L = cfg.limbs
    A[:, 0::4, :] = 0.0                                  # zero rows
    A[:, 1::4, :] = 0.0
    A[0, 1::4, 5] = 2.0 ** -7                            # a single power of two: one non-zero order per element
    A[:, 2::4, 1::2] = -A[:, 2::4, 0::2]                 # a_{2j+1} = -a_{2j} ...
    B[:, 1::2, :8] = B[:, 0::2, :8]                      # ... against b_{2j+1} = b_{2j} in the first 8 columns: exact zeros
    with md.Workspace(cfg.m, cfg.n, cfg.k, L, cfg.quarters):
        dA, dB = dev(A), dev(B)
        C = host(md.md_gemm(dA, dB))
        orders = md.md_gemm_orders(dA, dB)
        assert md.md_read_flags() == 0
    assert bool((C == host(md.md_renorm(orders, L))).all())
    assert not C[:, 0::4, :].any() and not C[:, 2::4, :8].any()
    r = orc.exact_all(A, B, C)
    assert (r["err"] <= TOL[L] * r["W"]).all()
    Aq, eA, _ = orc.split(A, 0)
    Bq, eB, _ = orc.split(B, 1)
    assert bool((host(orders) == orc.orders_int(Aq, eA, Bq, eB)).all())


@pytest.mark.parametrize("shape", [(200, 160, 40), (600, 300, 20), (600, 300, 3), (33, 17, 5)])
def test_hexa_double_passes_kernel_whole_tiles_and_stream_k_parts(shape):
    """Hexa double runs one order range at a time (qgemm_hd_passes_kernel: 32 x 16 CTA tiles, four passes over the contraction, the
    stream-K schedule over a virtual contraction of 4 KS slabs).  (200, 160): 70 tiles on 148 CTAs, every tile cut, the cuts fall
    inside and between passes; (600, 300): 19 x 19 = 361 tiles = two whole waves + 65 cut tiles; k = 3: one real k-slab, so a pass
    is a single virtual slab; (33, 17): ragged edge tiles.  Order matrices bit-exact against the oracle, C within tolerance of
    the exact product and equal to the standalone md_renorm of the dumped orders bit for bit."""
    cfg, A, B = gen(6, *shape)
    with md.Workspace(cfg.m, cfg.n, cfg.k, 16):
        orders = md.md_gemm_orders(dev(A), dev(B))
        C = host(md.md_gemm(dev(A), dev(B)))
        assert md.md_read_flags() == 0
    assert bool((C == host(md.md_renorm(orders, 16))).all())
    got = host(orders)
    si, sj = inputs.sample_indices(cfg, 300)
    Aq, eA, _ = orc.split(A, 0)
    Bq, eB, _ = orc.split(B, 1)
    want = orc.orders_int_samples(Aq, eA, Bq, eB, si, sj)
    assert bool((got[:, si, sj].T == want).all())
    r = orc.exact_samples(A, B, si, sj, C)
    assert (r["err"] <= TOL[16] * r["W"]).all()


@pytest.mark.parametrize("cfg_idx,shape", [(6, (200, 160, 40)), (6, (600, 300, 12)), (5, (300, 200, 24))])
def test_md_qgemm_on_oracle_quarters_with_both_outputs(cfg_idx, shape):
    """The public md_qgemm on PLAIN quarter planes (the oracle's) for the wide formats: they are repacked into the workspace in the
    tile shape of the kernel that runs them (hexa double: 32 x 16, one order range at a time), and one launch writes BOTH the order
    matrices and C -- whole tiles and stream-K parts.  Orders bit-exact against the oracle, C == md_renorm of them."""
    cfg, A, B = gen(cfg_idx, *shape)
    L, Q = cfg.limbs, cfg.quarters
    Aq, eA, _ = orc.split(A, 0)
    Bq, eB, _ = orc.split(B, 1)
    with md.Workspace(cfg.m, cfg.n, cfg.k, L, Q):
        orders, C = md.md_qgemm(dev(Aq), dev(Bq), L, want_orders=True, want_C=True)
    assert bool((host(orders) == orc.orders_int(Aq, eA, Bq, eB)).all())
    assert bool((C == md.md_renorm(orders, L)).all())


def test_unsupported_and_budget_errors():
    cfg, A, B = gen(5, 16, 16, 16)
    with md.Workspace(16, 16, 16, 8):
        md.md_set_option(md.MD_OPT_QUARTERS, 41)  # octo double: tuned kernels for 32 / 22, the generic one up to 40 quarters
        with pytest.raises(md.MdError) as e:
            md.md_gemm(dev(A), dev(B))
        assert e.value.status == md.MD_ERR_UNSUPPORTED
        md.md_set_option(md.MD_OPT_QUARTERS, 0)
    Aq, Bq = dev(np.zeros((32, 8, 8))), dev(np.zeros((32, 8, 8)))
    with pytest.raises(md.MdError) as e:  # md_qgemm repacks octo / hexa double planes into the registered workspace: none here
        md.md_qgemm(Aq, Bq, 8)
    assert e.value.status == md.MD_ERR_WORKSPACE

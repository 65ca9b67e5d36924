"""GPU parity of the k-adaptive slice variant (MD_OPT_SLICE_BITS; R14): slices of W != 13
bits, fewer of them.  Same bars as the paper's quarters: split and order matrices BIT-EXACT against the oracle's
oracle_*_w functions, final C within 1e-28 / 1e-58 (|A||B|)_ij of the exact product.  Small cases span several CTA tiles
with ragged tails; the full-size cases run BASELINE.json's shapes with the (W, Q) md_plan_slices picks, checked on samples."""
import numpy as np
import pytest
import torch

from oracle import md_oracle as orc
from paper_2607_06881_b200 import binding as md
from paper_2607_06881_b200 import inputs
from tests.test_gpu_fullsize import sample_positions

pytestmark = pytest.mark.gpu

TOL = {2: 1e-28, 4: 1e-58, 8: 1e-120, 16: 1e-245}
# (config index, W, Q): the plans md_plan_slices gives at the BASELINE sizes, and a few others with kernels
CASES = [(0, 19, 6), (1, 19, 6), (2, 19, 6), (3, 19, 6), (3, 16, 7), (4, 19, 11), (4, 18, 12), (5, 19, 22), (6, 19, 44)]
SHAPES = [(64, 64, 64), (150, 70, 90), (37, 51, 77), (1, 1, 1)]


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("bits", [7, 16, 19, 20, 24])
@pytest.mark.parametrize("cfg_idx,axis,shape", [(0, 0, (37, 77)), (3, 1, (150, 90)), (4, 0, (64, 64)), (3, 0, (1000, 3))])
def test_split_bit_exact_at_any_width(bits, cfg_idx, axis, shape):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(shape[0], 5, shape[1])
    X = inputs.generate(cfg, "A")
    Q = -(-(53 * cfg.limbs) // bits)
    md.md_set_option(md.MD_OPT_SLICE_BITS, bits)
    try:
        qp, exps = md.md_split(dev(X), axis, Q)
    finally:
        md.md_set_option(md.MD_OPT_SLICE_BITS, 0)
    want_q, want_e, _ = orc.split(X, axis, Q, bits=bits)
    assert (exps.cpu().numpy() == want_e).all()
    assert bool((qp.cpu().numpy() == want_q).all())


@pytest.mark.parametrize("cfg_idx,bits,Q", CASES)
@pytest.mark.parametrize("shape", SHAPES)
def test_orders_bit_exact_and_C_within_tolerance(cfg_idx, bits, Q, shape):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(*shape)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    with md.Workspace(cfg.m, cfg.n, cfg.k, cfg.limbs, Q, bits=bits):
        orders = md.md_gemm_orders(dev(A), dev(B))
        C = md.md_gemm(dev(A), dev(B))
        assert md.md_read_flags() == 0
        assert bool((C == md.md_renorm(orders, cfg.limbs)).all())  # fused epilogue == standalone renorm
    Aq, eA, _ = orc.split(A, 0, Q, bits=bits)
    Bq, eB, _ = orc.split(B, 1, Q, bits=bits)
    want = orc.orders_int(Aq, eA, Bq, eB, bits=bits)
    assert bool((orders.cpu().numpy() == want).all())
    Ch = C.cpu().numpy()
    r = orc.exact_all(A, B, Ch)
    if cfg_idx == 3:
        # the 2^[-30,30] element range at a SMALL k makes (|A||B|)_ij << 2^(E_i+F_j) common; there the common-exponent
        # reading guarantees the any-input bound (R5 with W in place of 13).  The full-size config 3 is held to
        # 1e-28 (|A||B|)_ij below.
        bound = cfg.k * (Q + 1) * np.ldexp(1.0, (eA[:, None] + eB[None, :] - bits * Q - 2).astype(np.int32))
        assert (r["err"] <= bound + np.abs(Ch[0]) * 2.0 ** (-53 * cfg.limbs + 1)).all()
    else:
        assert (r["err"] <= TOL[cfg.limbs] * r["W"]).all()


def test_k_budget_follows_the_slice_width():
    """k * S * 2^(2W) <= 2^53 (R14): W = 19, S = 6 allows k <= 5461."""
    A = torch.zeros((2, 8, 5462), dtype=torch.float64, device="cuda")
    B = torch.zeros((2, 5462, 8), dtype=torch.float64, device="cuda")
    with md.Workspace(8, 8, 5462, 2, 6, bits=19):
        with pytest.raises(md.MdError) as e:
            md.md_gemm(A, B)
        assert e.value.status == md.MD_ERR_K_TOO_LARGE
        md.md_gemm(A[:, :, :5461].contiguous(), B[:, :5461].contiguous())


@pytest.mark.parametrize("cfg_idx", [2, 3, 4])
def test_full_size_with_planned_slices(cfg_idx):
    """BASELINE.json's full shapes in the launch configuration `bench.py --slices adaptive` times."""
    cfg = inputs.CONFIGS[cfg_idx]
    L = cfg.limbs
    bits, Q = md.md_plan_slices(cfg.k, L)
    assert (bits, Q) == ((19, 6) if L == 2 else (19, 11))
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    dA, dB = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    Aq_o, eA_o, _ = orc.split(A, 0, Q, bits=bits)
    Bq_o, eB_o, _ = orc.split(B, 1, Q, bits=bits)
    si, sj = sample_positions(cfg, dA, dB, 512 if L == 2 else 192, 64)
    with md.Workspace(cfg.m, cfg.n, cfg.k, L, Q, bits=bits):
        orders = md.md_gemm_orders(dA, dB)
        got_orders = orders[:, torch.from_numpy(si).cuda(), torch.from_numpy(sj).cuda()].cpu().numpy().T
        fused_vs_unfused = md.md_renorm(orders, L)
        del orders
        C = md.md_gemm(dA, dB)
        assert md.md_read_flags() == 0
        assert bool((C == fused_vs_unfused).all())
        Ch = C.cpu().numpy()
    assert (got_orders == orc.orders_int_samples(Aq_o, eA_o, Bq_o, eB_o, si, sj, bits=bits)).all()
    r = orc.exact_samples(A, B, si, sj, Ch)
    ratio = r["err"] / (TOL[L] * r["W"])
    print(f"cfg{cfg_idx} W={bits} Q={Q}: max err/(tol*W) = {ratio.max():.3g} over {si.size} samples")
    assert (ratio <= 1.0).all()

"""GPU parity of the ONE-LAUNCH path (fused_small.cu, MD_OPT_ONE_LAUNCH; SURVEY.md 8(f) NEXT-3 "no quarter planes in HBM"):
every CTA derives the exponents of its rows / columns, splits its operand slabs into shared memory
(Algorithm S) and issues the quarter products; a thread-block cluster shares a tile along k.
Bars: order matrices BIT-EXACT against the oracle's int64 route, C bit-identical to the two-launch path and within the north_star
tolerance of the exact product, one kernel launch per call, the status flags of the separate preparation."""
import numpy as np
import pytest
import torch

from oracle import md_oracle as orc
from paper_2607_06881_b200 import binding as md
from paper_2607_06881_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = {2: 1e-28, 4: 1e-58}


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def host(t):
    return t.cpu().numpy()


def gen(cfg_idx, m, n, k):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(m, n, k)
    return cfg, inputs.generate(cfg, "A"), inputs.generate(cfg, "B")


def run(cfg, A, B, one_launch):
    md.md_set_option(md.MD_OPT_ONE_LAUNCH, one_launch)
    try:
        with md.Workspace(cfg.m, cfg.n, cfg.k, cfg.limbs, 4 * cfg.limbs):
            before = md.md_launch_count()
            orders = host(md.md_gemm_orders(dev(A), dev(B)))
            C = host(md.md_gemm(dev(A), dev(B)))
            launches = md.md_launch_count() - before
            flags = md.md_read_flags()
    finally:
        md.md_set_option(md.MD_OPT_ONE_LAUNCH, 0)
    return orders, C, launches, flags


# shapes: cluster sizes 8 / 4 / 2 / 1, ragged tails in m, n and k, odd n (unvectorised stores), a single element, k below one
# slab, more k-slabs than chunks of two, more tiles than SMs (forced mode: several waves of clusters)
SHAPES = [(64, 64, 64), (128, 128, 128), (192, 192, 100), (256, 256, 256), (70, 45, 90), (33, 21, 9), (1, 1, 1), (37, 51, 77),
          (150, 70, 3), (8, 8, 4), (500, 330, 41)]


@pytest.mark.parametrize("cfg_idx", [0, 1, 3, 4])
@pytest.mark.parametrize("shape", SHAPES)
def test_one_launch_path_orders_bit_exact_and_C_identical(cfg_idx, shape):
    cfg, A, B = gen(cfg_idx, *shape)
    L, Q = cfg.limbs, 4 * cfg.limbs
    orders, C, launches, flags = run(cfg, A, B, 1)
    assert launches == 2 and flags == 0                                  # one launch per call (md_gemm_orders + md_gemm)
    Aq, eA, _ = orc.split(A, 0, Q)
    Bq, eB, _ = orc.split(B, 1, Q)
    assert bool((orders == orc.orders_int(Aq, eA, Bq, eB)).all())        # a1 + a2 + a3 bit-exact
    orders2, C2, launches2, _ = run(cfg, A, B, 2)
    assert launches2 >= 4
    assert bool((orders == orders2).all()) and bool((C == C2).all())     # a4: the same epilogue, the same bits
    r = orc.exact_all(A, B, C)
    if cfg_idx in (0, 4):                                                 # well-scaled data: the north_star tolerance
        assert (r["err"] <= TOL[L] * r["W"]).all()
    # any input (cfg1 / cfg3 spread their elements over 2^+-8 / 2^+-30): the bound of DESIGN.md R5, relative to 2^(E_i + F_j)
    bound = cfg.k * (Q + 3) * np.ldexp(1.0, (eA[:, None] + eB[None, :] - 13 * Q - 2).astype(np.int32))
    assert (r["err"] <= bound + np.ldexp(np.abs(C[0]), -(53 * L - 3))).all()


def test_automatic_choice_and_launch_count():
    cfg, A, B = gen(0, 64, 64, 64)
    with md.Workspace(64, 64, 64, 2, 8):
        before = md.md_launch_count()
        md.md_gemm(dev(A), dev(B))
        assert md.md_launch_count() - before == 1                        # BASELINE.json configs[0] runs in one launch
    cfg, A, B = gen(2, 1024, 1024, 64)
    with md.Workspace(1024, 1024, 64, 2, 8):
        before = md.md_launch_count()
        md.md_gemm(dev(A), dev(B))
        assert md.md_launch_count() - before >= 2                        # 2048 tiles: the persistent kernel on pre-split operands


def test_status_flags_of_the_one_launch_path():
    cfg, A, B = gen(0, 70, 45, 90)
    md.md_set_option(md.MD_OPT_ONE_LAUNCH, 1)
    try:
        bad = A.copy()
        bad[1, 3, 5] = np.inf                                            # a non-finite LOW limb: only the splitter sees it
        with md.Workspace(70, 45, 90, 2, 8):
            md.md_gemm(dev(bad), dev(B))
            assert md.md_read_flags() & 1
        big = B * 2.0 ** 950                                             # column exponents beyond the documented range
        with md.Workspace(70, 45, 90, 2, 8):
            md.md_gemm(dev(A), dev(big))
            assert md.md_read_flags() & 2
        with md.Workspace(70, 45, 90, 2, 8):
            md.md_gemm(dev(A), dev(B))
            assert md.md_read_flags() == 0
    finally:
        md.md_set_option(md.MD_OPT_ONE_LAUNCH, 0)


def test_zero_groups_scaling_and_capture_in_a_graph():
    """Zero rows / columns (E = 0), power-of-two scaling of a row (digits unchanged), and the launch is an
    ordinary (cluster) kernel launch: capturable in a CUDA graph, replayed bit for bit."""
    cfg, A, B = gen(1, 64, 48, 72)
    A[:, 5, :] = 0.0
    B[:, :, 7] = 0.0
    A[:, 9, :] *= 2.0 ** 40
    orders, C, _, flags = run(cfg, A, B, 1)
    orders2, C2, _, _ = run(cfg, A, B, 2)
    assert flags == 0 and bool((orders == orders2).all()) and bool((C == C2).all())
    assert not C[:, 5, :].any() and not C[:, :, 7].any()
    md.md_set_option(md.MD_OPT_ONE_LAUNCH, 1)
    try:
        with md.Workspace(cfg.m, cfg.n, cfg.k, 2, 8):
            dA, dB = dev(A), dev(B)
            out = torch.zeros((2, cfg.m, cfg.n), dtype=torch.float64, device="cuda")
            s = torch.cuda.Stream()
            s.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(s):
                md.md_gemm(dA, dB, out)  # warm-up on the side stream
                graph = torch.cuda.CUDAGraph()
                out.zero_()
                with torch.cuda.graph(graph, stream=s):
                    md.md_gemm(dA, dB, out)
                graph.replay()
            s.synchronize()
            assert bool((host(out) == C).all())
    finally:
        md.md_set_option(md.MD_OPT_ONE_LAUNCH, 0)

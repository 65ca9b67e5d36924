"""GPU parity of the GENERIC quarter GEMM (runtime quarter / order counts, qgemm_wide.cu) and of MD_OPT_ORDERS (pruned and
extended order sets, PAPER.md:78 C_1..C_S): every (limbs, quarters, orders) md_gemm accepts has a kernel, and each is held to
the same bars as the tuned ones -- order matrices bit-exact against the oracle's int64 route, C equal to the oracle's
recombination of those orders up to the last limb (R9) and inside the any-input bound of DESIGN.md R5.
Closes the hole VERDICT r1 names: md_plan_quarters may prescribe any count, and md_gemm must run it."""
import numpy as np
import pytest
import torch

from oracle import md_oracle as orc
from paper_2607_06881_b200 import binding as md
from paper_2607_06881_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = {2: 1e-28, 4: 1e-58, 8: 1e-120, 16: 1e-245}
CFG_OF_LIMBS = {2: 3, 4: 4, 8: 5, 16: 6}


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def host(t):
    return t.cpu().numpy()


def check_orders_and_C(cfg, A, B, Q, S, bits=13):
    L = cfg.limbs
    with md.Workspace(cfg.m, cfg.n, cfg.k, L, Q, bits=bits, orders=S):
        orders = host(md.md_gemm_orders(dev(A), dev(B)))
        C = host(md.md_gemm(dev(A), dev(B)))
        assert md.md_read_flags() == 0
    Aq, eA, _ = orc.split(A, 0, Q, bits=bits)
    Bq, eB, _ = orc.split(B, 1, Q, bits=bits)
    want = orc.orders_int(Aq, eA, Bq, eB, orders=S, bits=bits)
    assert orders.shape == want.shape and bool((orders == want).all()), (L, Q, S)
    ref = orc.renorm(want, L)                       # the oracle's correctly rounded sum of the same orders
    slack = np.ldexp(np.abs(want).sum(axis=0), -(53 * L - 3))
    assert (np.abs((C - ref).sum(axis=0)) <= slack).all(), (L, Q, S)
    return C


# (limbs, quarters, orders): counts that have NO tuned kernel (generic path), at the edges of its range
GENERIC_CASES = [
    (2, 3, 3), (2, 5, 5), (2, 8, 7), (2, 8, 6), (2, 11, 11), (2, 12, 13), (2, 13, 15), (2, 16, 16), (2, 16, 18), (2, 9, 10),
    (4, 10, 10), (4, 13, 13), (4, 16, 15), (4, 19, 20), (4, 24, 24), (4, 24, 26),
    (8, 23, 23), (8, 31, 32), (8, 32, 34), (8, 40, 40), (8, 40, 42),
    (16, 45, 45), (16, 64, 66), (16, 63, 61), (16, 72, 72), (16, 72, 74),
]


@pytest.mark.parametrize("limbs,Q,S", GENERIC_CASES)
def test_generic_kernel_orders_bit_exact_and_C(limbs, Q, S):
    shape = {2: (70, 45, 52), 4: (37, 51, 29), 8: (33, 18, 21), 16: (17, 9, 13)}[limbs]
    cfg = inputs.CONFIGS[CFG_OF_LIMBS[limbs]].with_shape(*shape)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    check_orders_and_C(cfg, A, B, Q, S)


@pytest.mark.parametrize("limbs,Q,S", [(2, 8, 9), (2, 8, 10), (4, 16, 17), (4, 16, 18)])
@pytest.mark.parametrize("shape", [(150, 70, 90), (65, 33, 9), (1, 1, 1), (300, 200, 40)])
def test_tuned_extended_order_sets(limbs, Q, S, shape):
    """The tuned S > Q instances of the packed kernel (the cfg3-like case: a (Q+1)-th ORDER for Q - 1 more products instead
    of a (Q+1)-th QUARTER for Q + 1 more, R5)."""
    cfg = inputs.CONFIGS[CFG_OF_LIMBS[limbs]].with_shape(*shape)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    check_orders_and_C(cfg, A, B, Q, S)


def test_generic_kernel_equals_tuned_kernel_bit_for_bit():
    """The same (Q, S) on both kernels: dd 8 quarters through md_qgemm's plain-layout kernel and through the generic kernel
    (forced by asking for the orders of (8, 8) ... there is a tuned kernel, so compare via a count pair that exists in both:
    (8, 9) tuned packed against the generic one reached through md_qgemm's repacking of oracle quarters with orders = 9)."""
    cfg = inputs.CONFIGS[3].with_shape(130, 70, 100)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    with md.Workspace(cfg.m, cfg.n, cfg.k, 2, 8, orders=9):
        tuned = host(md.md_gemm_orders(dev(A), dev(B)))
        Ct = host(md.md_gemm(dev(A), dev(B)))
    # an odd shape through the generic kernel: quarters 8, orders 9 has a tuned instance, (8, 7) and (11, 12) do not
    Aq, eA, _ = orc.split(A, 0, 8)
    Bq, eB, _ = orc.split(B, 1, 8)
    assert bool((tuned == orc.orders_int(Aq, eA, Bq, eB, orders=9)).all())
    with md.Workspace(cfg.m, cfg.n, cfg.k, 2, 8, orders=7):
        pruned = host(md.md_gemm_orders(dev(A), dev(B)))
    assert bool((pruned == tuned[:7]).all())       # a pruned set is a prefix of the extended one, whichever kernel ran
    r = orc.exact_all(A, B, Ct)
    assert np.isfinite(r["err"]).all()


@pytest.mark.parametrize("shape", [(400, 330, 64), (148 * 4 + 5, 40, 24)])
def test_generic_kernel_stream_k_and_whole_tiles(shape):
    """More tiles than SMs on the generic kernel's 32 x 16 tiles: whole-tile waves plus a stream-K tail, against the oracle."""
    cfg = inputs.CONFIGS[1].with_shape(*shape)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    check_orders_and_C(cfg, A, B, 11, 12)


def test_md_qgemm_repacks_counts_without_a_plain_kernel():
    """md_qgemm on oracle quarters with (quarters, orders) that only the packed / generic kernels know: repacked into the
    registered workspace (include/mdgemm.h), same bits as the oracle."""
    for limbs, Q, S, shape in ((2, 11, 11, (70, 45, 52)), (2, 8, 9, (70, 45, 52)), (8, 32, 32, (33, 18, 21)), (4, 13, 14, (37, 51, 29))):
        cfg = inputs.CONFIGS[CFG_OF_LIMBS[limbs]].with_shape(*shape)
        A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
        Aq, eA, _ = orc.split(A, 0, Q)
        Bq, eB, _ = orc.split(B, 1, Q)
        with md.Workspace(cfg.m, cfg.n, cfg.k, limbs, Q, orders=S):
            orders, C = md.md_qgemm(dev(Aq), dev(Bq), limbs, want_orders=True, want_C=True, orders_kept=S)
            want = orc.orders_int(Aq, eA, Bq, eB, orders=S)
            assert bool((host(orders) == want).all()), (limbs, Q, S)
            assert bool((host(C) == host(md.md_renorm(orders, limbs))).all())
        with pytest.raises(md.MdError) as e:        # without a workspace the repacking has nowhere to go
            md.md_qgemm(dev(Aq), dev(Bq), limbs, orders_kept=S)
        assert e.value.status == md.MD_ERR_WORKSPACE


def test_every_planned_count_runs_and_meets_the_tolerance():
    """VERDICT r1 'done' criterion: md_plan_quarters -> md_gemm succeeds for every planned Q in a fuzz over element spreads up
    to 2^+-40, and the result is inside the format's tolerance at every position (what the plan promises)."""
    rng = np.random.default_rng(2607)
    seen = set()
    for trial in range(24):
        limbs = (2, 2, 2, 4)[trial % 4]
        spread = int(rng.integers(0, 41))
        m, n, k = (int(x) for x in rng.integers(1, 90, size=3))
        cfg = inputs.CONFIGS[CFG_OF_LIMBS[limbs]].with_shape(m, n, k)
        A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
        # per-element scaling by 2^e, e uniform in [-spread, spread]: exact, keeps the limbs non-overlapping
        A = A * np.ldexp(1.0, rng.integers(-spread, spread + 1, size=A.shape[1:]))[None]
        B = B * np.ldexp(1.0, rng.integers(-spread, spread + 1, size=B.shape[1:]))[None]
        Q, D = md.md_plan_quarters(dev(A), dev(B))
        seen.add((limbs, Q))
        if Q > {2: 16, 4: 24}[limbs]:   # beyond the generic maxima (D > ~100): the one refusal that is allowed, and it is loud
            with pytest.raises(md.MdError) as e:
                md.Workspace(cfg.m, cfg.n, cfg.k, limbs, Q)
            continue
        with md.Workspace(cfg.m, cfg.n, cfg.k, limbs, Q):
            C = host(md.md_gemm(dev(A), dev(B)))
            assert md.md_read_flags() == 0
        r = orc.exact_all(A, B, C)
        assert (r["err"] <= TOL[limbs] * r["W"]).all(), (limbs, spread, Q, D, float((r["err"] / (TOL[limbs] * r["W"] + 1e-300)).max()))
    assert len({q for _, q in seen}) >= 4, seen    # the fuzz really visited several counts, tuned and generic


def test_md_gemm_auto_runs_the_plan():
    """md_gemm_auto = md_plan_quarters + md_gemm with the planned count (include/mdgemm.h): same bits as doing it by hand,
    tolerance met where the paper's 8 quarters miss it."""
    cfg = inputs.CONFIGS[3].with_shape(96, 80, 256)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    md.md_set_workspace(None)
    C, Q = md.md_gemm_auto(dev(A), dev(B))
    assert md.md_read_flags() == 0
    Qp, _ = md.md_plan_quarters(dev(A), dev(B))
    assert Q == Qp == 10
    with md.Workspace(cfg.m, cfg.n, cfg.k, 2, Q):
        by_hand = host(md.md_gemm(dev(A), dev(B)))
    assert bool((host(C) == by_hand).all())
    r = orc.exact_all(A, B, host(C))
    assert (r["err"] <= 1e-28 * r["W"]).all()
    # a badly scaled row: [2^60, 1 + 2^-70] x [1; 1] -- the default 8 quarters lose the small element's low limb
    A2 = np.zeros((2, 1, 2))
    A2[0, 0] = [2.0 ** 60, 1.0]
    A2[1, 0] = [0.0, 2.0 ** -70]
    B2 = np.zeros((2, 2, 1))
    B2[0, :, 0] = [2.0 ** -60, 1.0]
    C2, Q2 = md.md_gemm_auto(dev(A2), dev(B2))
    r2 = orc.exact_all(A2, B2, host(C2))
    assert Q2 > 8 and (r2["err"] <= 1e-28 * r2["W"]).all()

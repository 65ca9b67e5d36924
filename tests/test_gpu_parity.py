"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element on the same seeded
inputs.  Bars (BASELINE.json north_star): split and order matrices BIT-EXACT; final C within 1e-28 (|A||B|)_ij (double
double) / 1e-58 (|A||B|)_ij (quad double) of the exact product; md_renorm within 2^-(53L-3) sum_s|C^(s)| of the oracle's
correctly rounded sum (several results are correct there, R9) and non-overlapping.
Sizes span several CTA tiles (64x32 / 32x16) with ragged tails in m, n and k, odd n / k (unvectorised loaders)."""
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


def bits_equal(a, b):
    """== on values (so that -0.0 == +0.0, R10) and no NaNs."""
    return bool((a == b).all())


SHAPES = [(64, 64, 64), (150, 70, 90), (65, 33, 9), (37, 51, 77), (8, 8, 4), (1, 1, 1), (129, 31, 130)]


# ------------------------------------------------------------------------------------------------ a1 + a2: md_split
@pytest.mark.parametrize("cfg_idx", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("shape", [(64, 64), (150, 90), (37, 77), (1, 1), (3, 1000), (1000, 3)])
@pytest.mark.parametrize("axis", [0, 1])
def test_split_bit_exact(cfg_idx, shape, axis):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(shape[0], 5, shape[1])
    X = inputs.generate(cfg, "A")
    for Q in (cfg.quarters, cfg.quarters + 1):
        qp, exps = md.md_split(dev(X), axis, Q)
        want_q, want_e, _ = orc.split(X, axis, Q)
        assert (host(exps) == want_e).all()
        assert bits_equal(host(qp), want_q)


def test_split_one_limb_zero_groups_and_signed_zero():
    X = np.zeros((1, 5, 6))
    X[0, 1] = [0.5, -0.0, 0.0, -0.25, 3e-9, 1.0 - 2.0 ** -53]
    X[0, 3, 2] = -7.0
    for axis in (0, 1):
        qp, exps = md.md_split(dev(X), axis, 5)
        want_q, want_e, _ = orc.split(X, axis, 5)
        assert (host(exps) == want_e).all() and bits_equal(host(qp), want_q)
        assert not np.signbit(host(qp)[:, 1, 1]).any()


def test_split_hand_derived_cases_on_gpu():
    """The special cases of tests/test_oracle_split.py (PAPER.md:124 Problem 3.3 etc.), straight on the GPU."""
    hi = np.array([[1.0, 0.0], [1.5 * 2.0 ** -41, 0.75], [2.0 ** -14, 0.75], [1.0 - 2.0 ** -53, 0.0]])
    lo = np.array([[-(2.0 ** -60), 0.0], [0.0, 0.0], [-(2.0 ** -80), 0.0], [2.0 ** -55, 0.0]])
    qp, exps = md.md_split(dev(np.stack([hi, lo])), 0, 8)
    E = host(exps)
    D = np.stack([np.ldexp(host(qp)[q, :, 0], -(E - 13 * (q + 1))) for q in range(8)]).T
    assert list(E) == [1, 0, 0, 0]
    assert D.tolist() == [[4096, 0, 0, 0, -16, 0, 0, 0], [0, 0, 0, 3072, 0, 0, 0, 0],
                          [0, 4096, 0, 0, 0, 0, -2048, 0], [8192, 0, 0, 0, -3072, 0, 0, 0]]


def test_split_idempotent_on_a_quarter_plane_and_powers_of_two_on_gpu():
    """a quarter plane split again is itself in one digit; a row of equal powers of two is one digit."""
    cfg, A, _ = gen(1, 40, 8, 36)
    qp, exps = md.md_split(dev(A), 0, 8)
    E = host(exps)
    Y = np.zeros_like(A)
    Y[0] = host(qp)[3]
    Y[0, :, 0] = np.ldexp(0.75, E)
    qq, e2 = md.md_split(dev(Y), 0, 8)
    assert (host(e2) == E).all()
    got = host(qq)
    assert bits_equal(got[3][:, 1:], host(qp)[3][:, 1:]) and not got[[0, 1, 2, 4, 5, 6, 7]][:, :, 1:].any()
    row = np.ldexp(1.0, -40) * np.array([[1.0, -1.0, 1.0, 1.0, -1.0]])
    q2, e3 = md.md_split(dev(np.stack([row, np.zeros_like(row)])), 0, 8)
    assert host(e3).tolist() == [-39] and bits_equal(host(q2)[0], row) and not host(q2)[1:].any()


# ------------------------------------------------------------------------------------------------ a3: order matrices
@pytest.mark.parametrize("cfg_idx", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("shape", SHAPES)
def test_order_matrices_bit_exact(cfg_idx, shape):
    cfg, A, B = gen(cfg_idx, *shape)
    with md.Workspace(cfg.m, cfg.n, cfg.k, cfg.limbs, cfg.quarters):
        got = host(md.md_gemm_orders(dev(A), dev(B)))
    Aq, eA, _ = orc.split(A, 0, cfg.quarters)
    Bq, eB, _ = orc.split(B, 1, cfg.quarters)
    want = orc.orders_int(Aq, eA, Bq, eB)
    assert got.shape == want.shape and bits_equal(got, want)


@pytest.mark.parametrize("limbs,Q", [(2, 8), (2, 9), (2, 10), (4, 16), (4, 17), (4, 18)])
def test_qgemm_on_oracle_quarters_bit_exact(limbs, Q):
    """Isolates the GEMM kernel: quarter planes come from the oracle."""
    cfg, A, B = gen(3 if limbs == 2 else 4, 70, 45, 52)
    Aq, eA, _ = orc.split(A, 0, Q)
    Bq, eB, _ = orc.split(B, 1, Q)
    orders, C = md.md_qgemm(dev(Aq), dev(Bq), limbs, want_orders=True, want_C=True)
    want = orc.orders_int(Aq, eA, Bq, eB)
    assert bits_equal(host(orders), want)
    # the fused epilogue is the same arithmetic as the standalone md_renorm
    assert bits_equal(host(C), host(md.md_renorm(orders, limbs)))


def test_identity_A_reproduces_quarters_of_B():
    cfg, _, B = gen(1, 96, 40, 96)
    A = np.zeros((2, 96, 96))
    A[0] = np.eye(96)
    with md.Workspace(96, 40, 96, 2):
        got = host(md.md_gemm_orders(dev(A), dev(B)))
    Bq, _, _ = orc.split(B, 1)
    assert bits_equal(got, Bq)


# ------------------------------------------------------------------------------------------------ a4: md_renorm
@pytest.mark.parametrize("cfg_idx", [0, 3, 4])
def test_renorm_against_oracle(cfg_idx):
    cfg, A, B = gen(cfg_idx, 50, 36, 120)
    Aq, eA, _ = orc.split(A, 0, cfg.quarters)
    Bq, eB, _ = orc.split(B, 1, cfg.quarters)
    ord_planes = orc.orders_int(Aq, eA, Bq, eB)
    got = host(md.md_renorm(dev(ord_planes), cfg.limbs))
    want = orc.renorm(ord_planes, cfg.limbs)
    L = cfg.limbs
    diff = np.abs(sum((got[l] - want[l]) for l in reversed(range(L))))
    assert (diff <= 2.0 ** -(53 * L - 3) * np.abs(ord_planes).sum(axis=0)).all()
    assert bits_equal(got[: L - 1], want[: L - 1])  # all but the last limb are in fact identical
    for l in range(L - 1):  # Definition 1.1: non-overlapping
        assert (np.abs(got[l + 1]) <= np.spacing(np.abs(got[l])) / 2).all()


def test_renorm_special_cases():
    x = np.array([[[1.0, -2.5, 0.0, 3.0]]])
    assert bits_equal(host(md.md_renorm(dev(x), 2)), np.stack([x[0], np.zeros_like(x[0])]))
    a, b = 1.0, 2.0 ** -70 + 2.0 ** -100
    C = host(md.md_renorm(dev(np.array([[[a]], [[b]]])), 2))
    assert C[0, 0, 0] == a + b and C[1, 0, 0] == (b - ((a + b) - a))  # TwoSum of (a, b), |a| > |b|
    # interior zeros: 1 + 2^-200 needs the second limb to jump over 150 bits of zeros
    C = host(md.md_renorm(dev(np.array([[[1.0]], [[0.0]], [[2.0 ** -200]]])), 4))
    assert C[:, 0, 0].tolist() == [1.0, 2.0 ** -200, 0.0, 0.0]


# ------------------------------------------------------------------------------------------------ the whole path
@pytest.mark.parametrize("cfg_idx", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("shape", [(64, 64, 64), (96, 80, 200), (37, 51, 77)])
def test_gemm_within_stated_tolerance_of_exact_product(cfg_idx, shape):
    cfg, A, B = gen(cfg_idx, *shape)
    # Config 3's 2^[-30,30] element range at a SMALL k makes (|A||B|)_ij << 2^(E_i+F_j) common, where the common-exponent
    # reading only guarantees the bound below (R5); one more quarter restores 1e-28 (|A||B|)_ij at these sizes.
    # The full-size config 3 (k = 2048, Q = 9) is checked against 1e-28 (|A||B|)_ij in tests/test_gpu_fullsize.py.
    Q = cfg.quarters + (1 if cfg_idx == 3 else 0)
    with md.Workspace(cfg.m, cfg.n, cfg.k, cfg.limbs, Q):
        C = host(md.md_gemm(dev(A), dev(B)))
        assert md.md_read_flags() == 0
    r = orc.exact_all(A, B, C)
    assert (r["err"] <= TOL[cfg.limbs] * r["W"]).all(), float((r["err"] / r["W"]).max())
    for l in range(cfg.limbs - 1):
        assert (np.abs(C[l + 1]) <= np.spacing(np.abs(C[l])) / 2).all()
    # and it is the oracle's own five-step result up to the last limb's rounding
    Co = orc.md_gemm_rows(A, B, quarters=Q)
    assert bits_equal(C[: cfg.limbs - 1], Co[: cfg.limbs - 1])


@pytest.mark.parametrize("cfg_idx,Q", [(0, 8), (3, 8), (3, 9), (3, 10), (4, 16)])
def test_gemm_error_bound_relative_to_group_exponents(cfg_idx, Q):
    """The guarantee for ANY input (include/mdgemm.h md_gemm; R5):
    |C - A*B|_ij <= k (Q+3) 2^(E_i+F_j-13Q-2) + 2^-(53L-1) |C|_ij."""
    cfg, A, B = gen(cfg_idx, 64, 64, 64)
    with md.Workspace(cfg.m, cfg.n, cfg.k, cfg.limbs, Q):
        C = host(md.md_gemm(dev(A), dev(B)))
    _, eA, _ = orc.split(A, 0)
    _, eB, _ = orc.split(B, 1)
    r = orc.exact_all(A, B, C)
    bound = cfg.k * (Q + 3) * np.ldexp(1.0, (eA[:, None] + eB[None, :] - 13 * Q - 2).astype(np.int32))
    assert (r["err"] <= bound + np.abs(C[0]) * 2.0 ** (-53 * cfg.limbs + 1)).all()


def test_small_integer_and_power_of_two_matrices_are_exact():
    rng = np.random.default_rng(7)
    Ai, Bi = rng.integers(-2 ** 20, 2 ** 20, (70, 130)), rng.integers(-2 ** 20, 2 ** 20, (130, 50))
    A, B = np.zeros((2, 70, 130)), np.zeros((2, 130, 50))
    A[0], B[0] = Ai, Bi
    with md.Workspace(70, 50, 130, 2):
        C = host(md.md_gemm(dev(A), dev(B)))
        assert bits_equal(C[0], (Ai @ Bi).astype(np.float64)) and not C[1].any()
        A[0] = np.ldexp(1.0, rng.integers(-20, 20, (70, 130)).astype(np.int32)) * rng.choice([-1.0, 1.0], (70, 130))
        B[0] = np.ldexp(1.0, rng.integers(-20, 20, (130, 50)).astype(np.int32))
        C = host(md.md_gemm(dev(A), dev(B)))
    r = orc.exact_all(A, B, C)
    assert not r["err"].any()


def test_zero_matrices_and_k_equal_one():
    with md.Workspace(40, 24, 1, 2):
        C = host(md.md_gemm(dev(np.zeros((2, 40, 1))), dev(np.zeros((2, 1, 24)))))
        assert not C.any()
        cfg, A, B = gen(0, 40, 24, 1)
        C = host(md.md_gemm(dev(A), dev(B)))
    r = orc.exact_all(A, B, C)
    assert (r["err"] <= 1e-28 * r["W"]).all()


def test_host_entry_point_matches_device_entry_point():
    cfg, A, B = gen(1, 130, 66, 100)
    with md.Workspace(cfg.m, cfg.n, cfg.k, 2):
        C = host(md.md_gemm(dev(A), dev(B)))
    Ah, Bh = torch.from_numpy(A).pin_memory(), torch.from_numpy(B).pin_memory()
    Ch = torch.empty((2, cfg.m, cfg.n), dtype=torch.float64).pin_memory()
    scratch = torch.empty(md.md_host_scratch_bytes(cfg.m, cfg.n, cfg.k, 2), dtype=torch.uint8, device="cuda")
    before = md.md_launch_count()
    md.md_gemm_host(Ah, Bh, Ch, scratch)
    assert md.md_launch_count() - before == 1  # one block of a single-wave problem: the one-launch kernel (MD_OPT_ONE_LAUNCH)
    assert bits_equal(Ch.numpy(), C)


@pytest.mark.parametrize("cfg_idx,shape,blocks", [(1, (300, 200, 100), 6), (3, (129, 31, 130), 16), (4, (100, 90, 40), 8),
                                                  (2, (640, 96, 24), 3), (5, (70, 50, 20), 4)])
def test_host_entry_point_pipelined_over_blocks_is_bit_identical(cfg_idx, shape, blocks):
    """md_gemm_host cuts C into row-panel x column-panel blocks and overlaps copies with kernels (include/mdgemm.h): a
    row's / column's exponent depends on that row / column only, so the blocks reproduce md_gemm bit for bit."""
    cfg, A, B = gen(cfg_idx, *shape)
    L = cfg.limbs
    with md.Workspace(cfg.m, cfg.n, cfg.k, L, cfg.quarters):
        C = host(md.md_gemm(dev(A), dev(B)))
        Ah, Bh = torch.from_numpy(A).pin_memory(), torch.from_numpy(B).pin_memory()
        Ch = torch.full((L, cfg.m, cfg.n), float("nan"), dtype=torch.float64).pin_memory()
        scratch = torch.empty(md.md_host_scratch_bytes(cfg.m, cfg.n, cfg.k, L), dtype=torch.uint8, device="cuda")
        md.md_set_option(md.MD_OPT_HOST_BLOCKS, blocks)
        try:
            md.md_gemm_host(Ah, Bh, Ch, scratch)
            md.md_gemm_host(Ah, Bh, Ch, scratch)  # a second call reuses the library's streams and events
        finally:
            md.md_set_option(md.MD_OPT_HOST_BLOCKS, 0)
    assert bits_equal(Ch.numpy(), C)


def test_flags_and_runtime_errors():
    cfg, A, B = gen(0, 16, 16, 16)
    A[0, 3, 4] = np.inf
    with md.Workspace(16, 16, 16, 2):
        md.md_gemm(dev(A), dev(B))
        assert md.md_read_flags() & 1
    with pytest.raises(md.MdError) as e:  # no workspace registered
        md.md_gemm(dev(A), dev(B))
    assert e.value.status == md.MD_ERR_WORKSPACE
    with md.Workspace(8, 8, 8, 2):  # too small for 1500 x 1500 x 64
        cfg2, A2, B2 = gen(0, 1500, 1500, 64)
        with pytest.raises(md.MdError) as e2:
            md.md_gemm(dev(A2), dev(B2))
        assert e2.value.status == md.MD_ERR_WORKSPACE


@pytest.mark.parametrize("cfg_idx,shape", [
    (2, (100, 60, 140)),      # the one-launch kernel
    (2, (700, 500, 90)),      # cooperative preparation kernel + the GEMM behind it as a programmatic dependent launch
    (4, (1100, 1500, 24)),    # quad double, 11 whole-tile waves: the hybrid tile schedule (queue counter cleared by a memset node)
])
def test_on_a_side_stream_and_in_a_cuda_graph(cfg_idx, shape):
    """md_gemm only enqueues: on a side stream, captured in a CUDA graph and REPLAYED TWICE (what a call leaves behind in the
    workspace -- counters, flags, the tile queue -- must not leak into the next replay)."""
    cfg, A, B = gen(cfg_idx, *shape)
    dA, dB = dev(A), dev(B)
    with md.Workspace(cfg.m, cfg.n, cfg.k, cfg.limbs, 4 * cfg.limbs):
        ref = md.md_gemm(dA, dB).clone()
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        out = torch.zeros_like(ref)
        with torch.cuda.stream(s):
            md.md_gemm(dA, dB, out)  # warm-up on the side stream
            graph = torch.cuda.CUDAGraph()
            out.zero_()
            with torch.cuda.graph(graph, stream=s):
                md.md_gemm(dA, dB, out)
            graph.replay()
            s.synchronize()
            assert bool((out == ref).all())
            out.zero_()
            graph.replay()
        s.synchronize()
        assert bool((out == ref).all())


@pytest.mark.parametrize("cfg_idx,shape", [(0, (64, 64, 64)), (1, (150, 70, 90)), (3, (37, 51, 77)), (4, (70, 45, 91)), (5, (40, 30, 20)),
                                           (2, (1, 1, 1)), (6, (20, 10, 12))])
def test_fused_preparation_is_bit_identical_to_the_separate_kernels(cfg_idx, shape):
    """MD_OPT_FUSED_PREP: exponent vectors and packed quarter planes of both operands in one launch (2 launches per md_gemm
    instead of 6) against the five separate launches: the order matrices and C must not differ in a bit."""
    cfg, A, B = gen(cfg_idx, *shape)
    out = {}
    for mode in (1, 2):
        md.md_set_option(md.MD_OPT_FUSED_PREP, mode)
        md.md_set_option(md.MD_OPT_ONE_LAUNCH, 2)   # the two-kernel path is what is compared here (tests/test_gpu_one_launch.py has the other)
        try:
            with md.Workspace(cfg.m, cfg.n, cfg.k, cfg.limbs, cfg.quarters):
                before = md.md_launch_count()
                C = md.md_gemm(dev(A), dev(B))
                launches = md.md_launch_count() - before
                out[mode] = (host(md.md_gemm_orders(dev(A), dev(B))), host(C), launches, md.md_read_flags())
        finally:
            md.md_set_option(md.MD_OPT_FUSED_PREP, 0)
            md.md_set_option(md.MD_OPT_ONE_LAUNCH, 0)
    assert out[1][2] == 2 and out[2][2] == 6 and out[1][3] == out[2][3] == 0
    assert bits_equal(out[1][0], out[2][0]) and bits_equal(out[1][1], out[2][1])
    Aq, eA, _ = orc.split(A, 0, cfg.quarters)
    Bq, eB, _ = orc.split(B, 1, cfg.quarters)
    assert bits_equal(out[1][0], orc.orders_int(Aq, eA, Bq, eB))


@pytest.mark.parametrize("shape", [(70001, 5, 3), (3, 70001, 5), (5, 3, 70001), (1, 40000, 1), (40000, 1, 1)])
def test_extreme_aspect_ratios(shape):
    """Tall, wide and deep degenerate shapes (one dimension 70 001, the others a handful): order matrices bit-exact, C
    within tolerance, host entry point bit-identical, with the paper's quarters and with 7 slices of 16 bits (whose
    whole-k budget, k <= 2^21 / 7, covers the deep shape; 19-bit slices stop at k = 5461)."""
    cfg, A, B = gen(0, *shape)
    for Q, W in ((8, 13), (7, 16)):
        with md.Workspace(cfg.m, cfg.n, cfg.k, 2, Q, bits=W):
            orders = host(md.md_gemm_orders(dev(A), dev(B)))
            C = md.md_gemm(dev(A), dev(B))
            assert md.md_read_flags() == 0
            Ch = torch.empty((2, cfg.m, cfg.n), dtype=torch.float64).pin_memory()
            scratch = torch.empty(md.md_host_scratch_bytes(cfg.m, cfg.n, cfg.k, 2), dtype=torch.uint8, device="cuda")
            md.md_gemm_host(torch.from_numpy(A).pin_memory(), torch.from_numpy(B).pin_memory(), Ch, scratch)
        assert bool((Ch == C.cpu()).all())
        Aq, eA, _ = orc.split(A, 0, Q, bits=W)
        Bq, eB, _ = orc.split(B, 1, Q, bits=W)
        assert bits_equal(orders, orc.orders_int(Aq, eA, Bq, eB, bits=W))
        si, sj = inputs.sample_indices(cfg, min(2000, cfg.m * cfg.n))
        r = orc.exact_samples(A, B, si, sj, host(C))
        assert (r["err"] <= 1e-28 * r["W"]).all()


@pytest.mark.parametrize("fused", [1, 2])
def test_exponent_range_flag_and_scaling_near_the_limits(fused):
    """include/mdgemm.h data preconditions: group exponents within [-900, 900] -- beyond, bit 1 of the status word is set
    (both preparation paths); inside, a problem scaled by 2^+-850 per operand is the same digits on a shifted grid, so C is
    the scaled C bit for bit; a group whose maximum is subnormal counts as a zero group."""
    cfg, A, B = gen(0, 40, 24, 32)
    md.md_set_option(md.MD_OPT_FUSED_PREP, fused)
    try:
        with md.Workspace(cfg.m, cfg.n, cfg.k, 2):
            C = host(md.md_gemm(dev(A), dev(B)))
            assert md.md_read_flags() == 0
            up, down = 2.0 ** 850, 2.0 ** -850
            Cs = host(md.md_gemm(dev(A * up), dev(B * down)))   # rows of A at 2^850, columns of B at 2^-850: C unchanged
            assert md.md_read_flags() == 0 and bits_equal(Cs, C)
            Cu = host(md.md_gemm(dev(A * 2.0 ** 400), dev(B * 2.0 ** 400)))
            assert md.md_read_flags() == 0 and bits_equal(Cu, C * 2.0 ** 800)
        with md.Workspace(cfg.m, cfg.n, cfg.k, 2):
            md.md_gemm(dev(A * 2.0 ** 950), dev(B))
            assert md.md_read_flags() == 2          # exponent out of range (bit 1), nothing non-finite (bit 0)
        with md.Workspace(cfg.m, cfg.n, cfg.k, 2):
            A2 = A.copy()
            A2[:, 3, :] = 0.0
            A2[0, 3, 5] = 5e-320                    # a subnormal row maximum: the row counts as zero
            C2 = host(md.md_gemm(dev(A2), dev(B)))
            assert not C2[:, 3, :].any() and bits_equal(np.delete(C2, 3, axis=1), np.delete(C, 3, axis=1))
    finally:
        md.md_set_option(md.MD_OPT_FUSED_PREP, 0)


@pytest.mark.parametrize("cfg_idx,shape,Q,W", [(0, (64, 64, 64), 8, 13), (1, (150, 70, 90), 8, 13), (3, (37, 51, 77), 8, 13),
                                               (2, (129, 31, 130), 6, 19), (2, (1, 1, 1), 8, 13), (1, (300, 200, 100), 6, 19)])
def test_small_tile_instance_is_bit_identical_to_the_large_one(cfg_idx, shape, Q, W):
    """MD_OPT_TILE: the 32 x 16 CTA tile instance of the double-double kernel (picked automatically when the 64 x 32 tiles
    would not fill the SMs) against the 64 x 32 one: order matrices and C must not differ in a bit, and both preparation
    paths must feed it."""
    cfg, A, B = gen(cfg_idx, *shape)
    out = {}
    for tile in (1, 2):
        for fused in (1, 2):
            md.md_set_option(md.MD_OPT_TILE, tile)
            md.md_set_option(md.MD_OPT_FUSED_PREP, fused)
            md.md_set_option(md.MD_OPT_ONE_LAUNCH, 2)
            try:
                with md.Workspace(cfg.m, cfg.n, cfg.k, 2, Q, bits=W):
                    out[tile, fused] = (host(md.md_gemm_orders(dev(A), dev(B))), host(md.md_gemm(dev(A), dev(B))), md.md_read_flags())
            finally:
                md.md_set_option(md.MD_OPT_TILE, 0)
                md.md_set_option(md.MD_OPT_FUSED_PREP, 0)
                md.md_set_option(md.MD_OPT_ONE_LAUNCH, 0)
    Aq, eA, _ = orc.split(A, 0, Q, bits=W)
    Bq, eB, _ = orc.split(B, 1, Q, bits=W)
    want = orc.orders_int(Aq, eA, Bq, eB, bits=W)
    for key, (orders, C, flags) in out.items():
        assert flags == 0 and bits_equal(orders, want), key
        assert bits_equal(C, out[2, 2][1]), key


@pytest.mark.parametrize("world", [2, 3, 8])
@pytest.mark.parametrize("cfg_idx,shape", [(3, (203, 77, 130)), (4, (70, 45, 91))])
def test_row_sharded_md_gemm_is_bit_identical_to_the_unsharded_call(world, cfg_idx, shape):
    """SURVEY.md 8(e) / DESIGN.md section 8: the path shards by rows of A with no collective.  Every rank's block
    (shard.row_block) through md_gemm on this one GPU, concatenated, must equal the unsharded md_gemm bit for bit: E_i and the
    quarters of a row depend on that row only, F_j on B only.  Ragged m (not a multiple of world or of the tile), cfg3's
    wide-range distribution and quad double."""
    from paper_2607_06881_b200 import shard
    cfg, A, B = gen(cfg_idx, *shape)
    dA, dB = dev(A), dev(B)
    with md.Workspace(cfg.m, cfg.n, cfg.k, cfg.limbs, cfg.quarters):
        whole = host(md.md_gemm(dA, dB))
        whole_orders = host(md.md_gemm_orders(dA, dB))
        parts, parts_orders = [], []
        for rank in range(world):
            r0, r1 = shard.row_block(cfg.m, world, rank)
            if r1 == r0:
                continue
            blk = dA[:, r0:r1, :].contiguous()
            parts.append(host(md.md_gemm(blk, dB)))
            parts_orders.append(host(md.md_gemm_orders(blk, dB)))
        assert md.md_read_flags() == 0
    assert bits_equal(np.concatenate(parts, axis=1), whole)
    assert bits_equal(np.concatenate(parts_orders, axis=1), whole_orders)


@pytest.mark.parametrize("cfg_idx,shape,Q,S,schedule", [
    (1, (1000, 700, 200), 8, 8, 1),     # dd, 64 x 32 tiles: 16 x 22 = 352 = 2.4 waves of 148; ragged m, n; 25 slabs in units of 2
    (3, (1000, 700, 72), 9, 9, 1),      # cfg3's distribution with the ninth quarter
    (3, (700, 1000, 40), 8, 9, 1),      # an extended order set
    (4, (400, 300, 90), 16, 16, 2),     # qd, 32 x 16 tiles: 13 x 19 = 247 tiles
    (4, (700, 500, 40), 16, 16, 1),     # qd, 22 x 32 = 704 tiles = 4.8 waves: static waves, then the queue
    (0, (1600, 1600, 64), 8, 8, 2),     # 25 x 50 = 1250 tiles = 8.4 waves, the queue from the first tile on
    (2, (1601, 1530, 8), 8, 8, 1),      # one slab per tile: the units are whole tiles; 7 static waves first
    (2, (1024, 1024, 7), 6, 6, 1),      # 6 slices of 19 bits
    (4, (1100, 1500, 24), 16, 16, 0),   # qd, 35 x 47 = 1645 tiles = 11.1 waves: the AUTOMATIC rule takes the hybrid here
])
def test_dynamic_tile_schedule_is_bit_identical_to_the_static_lists(cfg_idx, shape, Q, S, schedule):
    """MD_OPT_TILE_SCHEDULE: the CTAs of the persistent kernel claim k-units of the last tiles (hybrid: 1, and 0 from many waves
    on) or every tile (2) from a queue counter instead of walking static lists (3) -- DESIGN.md section 6.  Every partial order sum is exact (R6), so the order matrices
    and C must not differ in a bit from the static schedule, whichever CTA computed what -- repeated, because the assignment
    differs from run to run -- and the order matrices must equal the oracle's."""
    cfg, A, B = gen(cfg_idx, *shape)
    W = 19 if Q == 6 else 13
    dA, dB = dev(A), dev(B)
    out = {}
    try:
        with md.Workspace(cfg.m, cfg.n, cfg.k, cfg.limbs, Q, bits=W, orders=S):
            md.md_set_option(md.MD_OPT_TILE_SCHEDULE, 3)
            out["static"] = (host(md.md_gemm_orders(dA, dB)), host(md.md_gemm(dA, dB)))
            md.md_set_option(md.MD_OPT_TILE_SCHEDULE, schedule)
            for rep in range(3):
                out[rep] = (host(md.md_gemm_orders(dA, dB)), host(md.md_gemm(dA, dB)))
            assert md.md_read_flags() == 0
    finally:
        md.md_set_option(md.MD_OPT_TILE_SCHEDULE, 0)
    for rep in range(3):
        assert bits_equal(out[rep][0], out["static"][0]) and bits_equal(out[rep][1], out["static"][1]), rep
    si, sj = inputs.sample_indices(cfg, 4096, salt=7)
    Aq, eA, _ = orc.split(A, 0, Q, bits=W)
    Bq, eB, _ = orc.split(B, 1, Q, bits=W)
    want = orc.orders_int_samples(Aq, eA, Bq, eB, si, sj, orders=S, bits=W)
    assert bits_equal(out[0][0][:, si, sj].T, want)

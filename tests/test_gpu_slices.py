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
        bound = cfg.k * (Q + 3) * np.ldexp(1.0, (eA[:, None] + eB[None, :] - bits * Q - 2).astype(np.int32))
        assert (r["err"] <= bound + np.abs(Ch[0]) * 2.0 ** (-53 * cfg.limbs + 1)).all()
    else:
        assert (r["err"] <= TOL[cfg.limbs] * r["W"]).all()


def test_k_budget_follows_the_slice_width():
    """k * S * 2^(2W) <= 2^53 (R14): W = 19, S = 6 allows k <= 5461."""
    A = torch.zeros((2, 8, 5462), dtype=torch.float64, device="cuda")
    B = torch.zeros((2, 5462, 8), dtype=torch.float64, device="cuda")
    with md.Workspace(8, 8, 5462, 2, 6, bits=19):
        with pytest.raises(md.MdError) as e:
            md.md_gemm_orders(A, B)
        assert e.value.status == md.MD_ERR_K_TOO_LARGE
        md.md_gemm_orders(A[:, :, :5461].contiguous(), B[:, :5461].contiguous())
        md.md_gemm(A, B)  # md_gemm chunks the contraction instead (R16)


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


# ---------------------------------------------------------------------------------------------- chunked accumulation (R16)
def last_limb_close(C, Co, L):
    """all but the last limb bit-identical, the last within the renormalisation bound of DESIGN.md R9"""
    return bool((C[: L - 1] == Co[: L - 1]).all()) and bool((np.abs(C[L - 1] - Co[L - 1]) <= 2.0 ** -(53 * L - 3) * np.abs(Co[0]) * 64).all())


@pytest.mark.parametrize("cfg_idx,shape", [(0, (64, 64, 1000)), (1, (150, 70, 900)), (2, (37, 51, 1700)), (2, (200, 100, 40))])
def test_chunked_accumulation_with_planned_wide_slices(cfg_idx, shape):
    """5 slices of 21 bits, chunks of 408 (md_plan_slices_chunked): C within 1e-28 (|A||B|)_ij of the exact product and equal
    to the oracle's chunked pipeline up to the last limb's rounding."""
    cfg = inputs.CONFIGS[cfg_idx].with_shape(*shape)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    W, Q, chunk = md.md_plan_slices_chunked(4096, 2, 256)
    assert (W, Q, chunk) == (21, 5, 408)
    with md.Workspace(cfg.m, cfg.n, cfg.k, 2, Q, bits=W):
        C = md.md_gemm(dev(A), dev(B)).cpu().numpy()
        assert md.md_read_flags() == 0
    r = orc.exact_all(A, B, C)
    assert (r["err"] <= 1e-28 * r["W"]).all()
    assert last_limb_close(C, orc.md_gemm_rows_chunked(A, B, 408, Q, W), 2)


@pytest.mark.parametrize("Q,W", [(8, 13), (6, 19)])
def test_forced_short_chunks_agree_with_the_unchunked_path(Q, W):
    """MD_OPT_K_CHUNK = 64 on a contraction of 300 (5 chunks, the last one ragged), the paper's quarters and the 19-bit
    slices: same result as the exact-order path up to the last limb, host entry point included."""
    cfg = inputs.CONFIGS[1].with_shape(130, 66, 300)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    with md.Workspace(cfg.m, cfg.n, cfg.k, 2, Q, bits=W):
        C0 = md.md_gemm(dev(A), dev(B)).cpu().numpy()
    md.md_set_option(md.MD_OPT_K_CHUNK, 64)  # before the workspace is sized: the chunked stream-K scratch depends on it
    try:
        with md.Workspace(cfg.m, cfg.n, cfg.k, 2, Q, bits=W):
            C1 = md.md_gemm(dev(A), dev(B)).cpu().numpy()
            Ch = torch.empty((2, cfg.m, cfg.n), dtype=torch.float64).pin_memory()
            scratch = torch.empty(md.md_host_scratch_bytes(cfg.m, cfg.n, cfg.k, 2), dtype=torch.uint8, device="cuda")
            md.md_gemm_host(torch.from_numpy(A).pin_memory(), torch.from_numpy(B).pin_memory(), Ch, scratch)
    finally:
        md.md_set_option(md.MD_OPT_K_CHUNK, 0)
    assert last_limb_close(C1, C0, 2) and bool((Ch.numpy() == C1).all())
    assert last_limb_close(C1, orc.md_gemm_rows_chunked(A, B, 64, Q, W), 2)
    r = orc.exact_all(A, B, C1)
    assert (r["err"] <= 1e-28 * r["W"]).all()


def test_full_size_chunked_dd_4096():
    """BASELINE.json configs[2] with the chunked plan (5 slices of 21 bits, chunks of 408), on samples."""
    cfg = inputs.CONFIGS[2]
    W, Q, chunk = md.md_plan_slices_chunked(cfg.k, 2, 256)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    dA, dB = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    si, sj = sample_positions(cfg, dA, dB, 512, 64)
    with md.Workspace(cfg.m, cfg.n, cfg.k, 2, Q, bits=W):
        Ch = md.md_gemm(dA, dB).cpu().numpy()
        assert md.md_read_flags() == 0
    r = orc.exact_samples(A, B, si, sj, Ch)
    ratio = r["err"] / (1e-28 * r["W"])
    print(f"cfg2 chunked W={W} Q={Q} chunk={chunk}: max err/(tol*W) = {ratio.max():.3g} over {si.size} samples")
    assert (ratio <= 1.0).all()
    assert (np.abs(Ch[1]) <= np.spacing(np.abs(Ch[0])) / 2).all()


def test_chunked_stream_k_tail_is_bit_identical_to_whole_tiles():
    """The chunked kernel's stream-K tail adds each chunk's exact sums into that chunk's scratch slot and the finishing CTA
    replays the renorm_add sequence, so cutting tiles along k must not change a bit: a 600 x 600 problem (190 tiles on 148
    CTAs: 42 tiles are cut) against the same rows computed as part of a problem whose tiles are all whole-wave (a 64 x 32
    block = 1 tile, processed whole)."""
    cfg = inputs.CONFIGS[2].with_shape(600, 600, 1000)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    W, Q = 21, 5
    with md.Workspace(cfg.m, cfg.n, cfg.k, 2, Q, bits=W):
        C = md.md_gemm(dev(A), dev(B)).cpu().numpy()
    for (r0, c0) in ((0, 0), (512, 576), (320, 96)):  # single-tile problems: never cut along k
        Ab, Bb = np.ascontiguousarray(A[:, r0:r0 + 64]), np.ascontiguousarray(B[:, :, c0:c0 + 32])
        mb, nb = Ab.shape[1], Bb.shape[2]
        with md.Workspace(mb, nb, cfg.k, 2, Q, bits=W):
            Cb = md.md_gemm(dev(Ab), dev(Bb)).cpu().numpy()
        assert bool((C[:, r0:r0 + mb, c0:c0 + nb] == Cb).all())
    r = orc.exact_samples(A, B, *inputs.sample_indices(cfg, 256), C)
    assert (r["err"] <= 1e-28 * r["W"]).all()


@pytest.mark.parametrize("shape", [(70, 45, 500), (130, 40, 90)])
def test_chunked_accumulation_quad_double(shape):
    """Quad double in 10 slices of 21 bits, chunks of 200 (md_plan_slices_chunked(2048, 4, 128)): C within 1e-58 (|A||B|)_ij
    and equal to the oracle's chunked pipeline up to the last limb."""
    assert md.md_plan_slices_chunked(2048, 4, 128) == (21, 10, 200)
    cfg = inputs.CONFIGS[4].with_shape(*shape)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    with md.Workspace(cfg.m, cfg.n, cfg.k, 4, 10, bits=21):
        C = md.md_gemm(dev(A), dev(B)).cpu().numpy()
        assert md.md_read_flags() == 0
    r = orc.exact_all(A, B, C)
    assert (r["err"] <= 1e-58 * r["W"]).all()
    assert last_limb_close(C, orc.md_gemm_rows_chunked(A, B, 200, 10, 21), 4)

"""Seeded differential test of the whole C-ABI surface against the oracle: random shapes (ragged in every dimension,
down to 1), formats, distributions, slice widths / counts, chunk lengths and host-block counts.  For every case: split
bit-exact, order matrices bit-exact (where the call provides them), C within the any-input bound (R5) and within
the format's tolerance of the exact product wherever the data-driven plan (R15) guarantees it, md_gemm_host bit-identical
to md_gemm."""
import numpy as np
import pytest
import torch

from oracle import md_oracle as orc
from paper_2607_06881_b200 import binding as md
from paper_2607_06881_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = {2: 1e-28, 4: 1e-58, 8: 1e-120, 16: 1e-245}
# (limbs, slice bits, slice count, chunked?) combinations that have kernels
VARIANTS = [(2, 13, 8, False), (2, 13, 9, False), (2, 13, 10, False), (2, 19, 6, False), (2, 16, 7, False), (2, 21, 5, True),
            (2, 13, 8, True), (2, 19, 6, True), (4, 21, 10, True), (4, 13, 16, False), (4, 13, 17, False), (4, 19, 11, False), (4, 18, 12, False),
            (8, 13, 32, False), (8, 19, 22, False), (16, 13, 64, False), (16, 19, 44, False)]
CFG_OF_LIMBS = {2: (0, 1, 2, 3), 4: (4,), 8: (5,), 16: (6,)}


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("case", range(128))
def test_random_case(case):
    rng = np.random.default_rng(1000 + case)
    L, W, Q, chunked = VARIANTS[case % len(VARIANTS)]
    big = L <= 4
    m, n = int(rng.integers(1, 200 if big else 60)), int(rng.integers(1, 150 if big else 40))
    k = int(rng.integers(1, 260 if big else 50))
    cfg_idx = int(rng.choice(CFG_OF_LIMBS[L]))
    cfg = inputs.CONFIGS[cfg_idx].with_shape(m, n, k)
    cfg = inputs.Config(cfg.index, cfg.name, m, n, k, L, 7000 + case, cfg.dist)  # a fresh seed per case
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    dA, dB = dev(A), dev(B)
    chunk = int(rng.choice([8, 16, 64])) if chunked else 0
    blocks = int(rng.choice([0, 1, 3, 6]))
    one_launch = int(rng.choice([0, 1, 2]))  # automatic / wherever the one-launch kernel exists / never: the same bits
    Aq_o, eA, _ = orc.split(A, 0, Q, bits=W)
    Bq_o, eB, _ = orc.split(B, 1, Q, bits=W)
    md.md_set_option(md.MD_OPT_K_CHUNK, chunk)
    md.md_set_option(md.MD_OPT_HOST_BLOCKS, blocks)
    md.md_set_option(md.MD_OPT_ONE_LAUNCH, one_launch)
    try:
        md.md_set_option(md.MD_OPT_SLICE_BITS, 0 if W == 13 else W)
        Aq, gA = md.md_split(dA, 0, Q)
        Bq, gB = md.md_split(dB, 1, Q)
        assert (gA.cpu().numpy() == eA).all() and (gB.cpu().numpy() == eB).all()
        assert bool((Aq.cpu().numpy() == Aq_o).all()) and bool((Bq.cpu().numpy() == Bq_o).all())
        with md.Workspace(m, n, k, L, Q, bits=W):
            C = md.md_gemm(dA, dB)
            assert md.md_read_flags() == 0
            if not (chunked and (Q in (5, 10) or k > chunk)):
                orders = md.md_gemm_orders(dA, dB)
                assert bool((orders.cpu().numpy() == orc.orders_int(Aq_o, eA, Bq_o, eB, bits=W)).all())
                if not chunked:
                    assert bool((C == md.md_renorm(orders, L)).all())
            Ch = torch.full((L, m, n), float("nan"), dtype=torch.float64).pin_memory()
            scratch = torch.empty(md.md_host_scratch_bytes(m, n, k, L), dtype=torch.uint8, device="cuda")
            md.md_gemm_host(torch.from_numpy(A).pin_memory(), torch.from_numpy(B).pin_memory(), Ch, scratch)
            assert bool((Ch == C.cpu()).all())
    finally:
        for key in (md.MD_OPT_K_CHUNK, md.MD_OPT_HOST_BLOCKS, md.MD_OPT_SLICE_BITS, md.MD_OPT_ONE_LAUNCH):
            md.md_set_option(key, 0)
    Cn = C.cpu().numpy()
    r = orc.exact_all(A, B, Cn)
    # the any-input bound (R5) always; the tolerance relative to (|A||B|)_ij wherever the data-driven plan
    # (R15) says this slice count guarantees it, and for the well-scaled distributions regardless
    bound = k * (Q + 3) * np.ldexp(1.0, (eA[:, None] + eB[None, :] - W * Q - 2).astype(np.int32))
    assert (r["err"] <= bound + np.abs(Cn[0]) * 2.0 ** (-53 * L + 1)).all()
    Q_needed, _ = orc.plan_quarters(A, B, TOL[L], bits=W)
    if Q >= Q_needed or cfg.dist in ("uniform", "normal"):
        assert (r["err"] <= TOL[L] * r["W"]).all(), float((r["err"] / (TOL[L] * r["W"])).max())
    for l in range(L - 1):
        assert (np.abs(Cn[l + 1]) <= np.spacing(np.abs(Cn[l])) / 2).all()


@pytest.mark.parametrize("case", range(20))
def test_random_multiwave_case(case):
    """Larger random shapes (short contractions, so that the oracle stays cheap): several to dozens of whole-tile waves on the
    persistent kernels.  Double / quad double: every tile schedule (MD_OPT_TILE_SCHEDULE automatic, hybrid, queue only) against
    the static lists bit for bit, C and order matrices; all formats: sampled order matrices against the oracle and the fused
    epilogue against the standalone md_renorm.  (A one-off run of this generator over 24 182 cases, incl. hexa double through
    its one-range-at-a-time kernel and md_gemm_static, found no difference.)"""
    rng = np.random.default_rng(5000 + case)
    kind = ("dd", "qd", "dd", "hd", "od")[case % 5]
    if kind == "dd":
        L, Q, cfg_idx = 2, int(rng.choice([8, 9])), int(rng.choice([0, 1, 2, 3]))
        m, n, k = int(rng.integers(1200, 4200)), int(rng.integers(1200, 4200)), int(rng.integers(1, 70))
    elif kind == "qd":
        L, Q, cfg_idx = 4, 16, 4
        m, n, k = int(rng.integers(700, 2400)), int(rng.integers(700, 2400)), int(rng.integers(1, 50))
    elif kind == "hd":
        L, Q, cfg_idx = 16, 64, 6
        m, n, k = int(rng.integers(33, 800)), int(rng.integers(17, 600)), int(rng.integers(1, 40))
    else:
        L, Q, cfg_idx = 8, 32, 5
        m, n, k = int(rng.integers(33, 1200)), int(rng.integers(17, 1000)), int(rng.integers(1, 40))
    S = Q + 1 if (kind == "dd" and Q == 8 and case % 2) else Q
    base = inputs.CONFIGS[cfg_idx]
    cfg = inputs.Config(base.index, base.name, m, n, k, L, 9000 + case, base.dist)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    dA, dB = dev(A), dev(B)
    schedules = (3, 0, 1, 2) if L <= 4 else (0,)
    res = {}
    try:
        with md.Workspace(m, n, k, L, Q, orders=(S if S != Q else 0)):
            for ts in schedules:
                md.md_set_option(md.MD_OPT_TILE_SCHEDULE, ts)
                res[ts] = (md.md_gemm(dA, dB), md.md_gemm_orders(dA, dB))
            assert md.md_read_flags() == 0
    finally:
        md.md_set_option(md.MD_OPT_TILE_SCHEDULE, 0)
    C, orders = res[schedules[0]]
    for ts in schedules[1:]:
        assert bool((res[ts][0] == C).all()) and bool((res[ts][1] == orders).all()), ts
    si, sj = rng.integers(0, m, 1500), rng.integers(0, n, 1500)
    Aq, eA, _ = orc.split(A, 0, Q)
    Bq, eB, _ = orc.split(B, 1, Q)
    want = orc.orders_int_samples(Aq, eA, Bq, eB, si, sj, orders=S)
    assert bool((orders[:, si, sj].T.cpu().numpy() == want).all())
    if S == Q:
        assert bool((C == md.md_renorm(orders, L)).all())
    r = orc.exact_samples(A, B, si[:200], sj[:200], C.cpu().numpy())
    bound = k * (Q + 3) * np.ldexp(1.0, (eA[si[:200]] + eB[sj[:200]] - 13 * Q - 2).astype(np.int32))
    assert (r["err"] <= bound + np.abs(C[0, si[:200], sj[:200]].cpu().numpy()) * 2.0 ** (-53 * L + 1)).all()

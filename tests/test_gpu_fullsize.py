"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (md_gemm with the config's
quarter count), checked on sampled outputs the oracle can compute one by one:
  * split: bit-exact on the WHOLE matrices (the oracle's split is elementwise and fast);
  * order matrices: bit-exact at sampled (i, j) (int64 digit route);
  * final C: |C - C_exact| <= tol * (|A||B|)_ij at sampled (i, j) -- uniformly random positions, two full rows / columns
    worth of positions, and the positions with the SMALLEST (|A||B|)_ij / 2^(E_i+F_j) estimate (most at risk, R5).
"""
import numpy as np
import pytest
import torch

from oracle import md_oracle as orc
from paper_2607_06881_b200 import binding as md
from paper_2607_06881_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = {2: 1e-28, 4: 1e-58}


def sample_positions(cfg, dA, dB, n_random, n_risky):
    si, sj = inputs.sample_indices(cfg, n_random)
    # a full row and a full column worth of positions, subsampled to 256 each
    r, c = int(si[0]), int(sj[0])
    cols = np.linspace(0, cfg.n - 1, 256).astype(np.int64)
    rows = np.linspace(0, cfg.m - 1, 256).astype(np.int64)
    si = np.concatenate([si, np.full(256, r), rows])
    sj = np.concatenate([sj, cols, np.full(256, c)])
    # the riskiest positions: smallest (|A_hi||B_hi|)_ij relative to the product of the group maxima (fp64 estimate,
    # used ONLY to choose where to look)
    W = dA[0].abs() @ dB[0].abs()
    rel = W / (dA[0].abs().amax(dim=1)[:, None] * dB[0].abs().amax(dim=0)[None, :])
    flat = torch.topk(rel.flatten(), n_risky, largest=False).indices.cpu().numpy()
    si = np.concatenate([si, flat // cfg.n])
    sj = np.concatenate([sj, flat % cfg.n])
    return si.astype(np.int64), sj.astype(np.int64)


@pytest.mark.parametrize("cfg_idx", [1, 2, 3, 4])
def test_full_size_config(cfg_idx):
    cfg = inputs.CONFIGS[cfg_idx]
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    dA, dB = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    Q, L = cfg.quarters, cfg.limbs

    # a1 + a2 on the whole matrices
    Aq_o, eA_o, _ = orc.split(A, 0, Q)
    Bq_o, eB_o, _ = orc.split(B, 1, Q)
    Aq, eA = md.md_split(dA, 0, Q)
    assert (eA.cpu().numpy() == eA_o).all() and bool((Aq.cpu() == torch.from_numpy(Aq_o)).all())
    del Aq
    Bq, eB = md.md_split(dB, 1, Q)
    assert (eB.cpu().numpy() == eB_o).all() and bool((Bq.cpu() == torch.from_numpy(Bq_o)).all())
    del Bq

    n_random = 512 if L == 2 else 192
    si, sj = sample_positions(cfg, dA, dB, n_random, 64)
    with md.Workspace(cfg.m, cfg.n, cfg.k, L, Q):
        orders = md.md_gemm_orders(dA, dB)
        got_orders = orders[:, torch.from_numpy(si).cuda(), torch.from_numpy(sj).cuda()].cpu().numpy().T
        fused_vs_unfused = md.md_renorm(orders, L)
        del orders
        C = md.md_gemm(dA, dB)
        assert md.md_read_flags() == 0
        assert bool((C == fused_vs_unfused).all())  # fused epilogue == standalone renorm of the dumped orders
        del fused_vs_unfused
        Ch = C.cpu().numpy()

    # a3 at the sampled positions, bit-exact
    want_orders = orc.orders_int_samples(Aq_o, eA_o, Bq_o, eB_o, si, sj)
    assert (got_orders == want_orders).all()

    # final C against the exact product
    r = orc.exact_samples(A, B, si, sj, Ch)
    ratio = r["err"] / (TOL[L] * r["W"])
    print(f"cfg{cfg_idx} Q={Q}: max err/(tol*W) = {ratio.max():.3g} over {si.size} samples "
          f"(riskiest 64: {ratio[-64:].max():.3g})")
    assert (ratio <= 1.0).all()
    for l in range(L - 1):
        assert (np.abs(Ch[l + 1]) <= np.spacing(np.abs(Ch[l])) / 2).all()

"""GPU parity of md_qr (include/mdgemm.h, ref [18] PAPER.md:235): blocked Householder QR with
the trailing updates through md_gemm, against oracle part O7 (unblocked, scalar multiple-double arithmetic) at small sizes and
against the definition at 512 and 2048: |A - Q R| and |Q^T Q - I| evaluated EXACTLY (the oracle's long accumulator, O1) at sampled
positions, at working precision; R upper triangular with diag(R) >= 0."""
import numpy as np
import pytest
import torch

from oracle import md_oracle as orc
from paper_2607_06881_b200 import binding as md
from paper_2607_06881_b200 import inputs

pytestmark = pytest.mark.gpu


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def host(t):
    return t.cpu().numpy()


def residual_and_orthogonality(A, Q, R, samples, seed):
    """(max |A - QR|_ij / (|Q||R|)_ij-scale, max |Q^T Q - I|_ij) on `samples` random positions each, exactly (oracle O1)."""
    L, m, n = A.shape
    rng = np.random.default_rng(seed)
    si, sj = rng.integers(0, m, samples), rng.integers(0, n, samples)
    r = orc.exact_samples(Q, R, si, sj, C=A)                    # |A - Q R|_ij exactly
    res = float((r["err"] / np.abs(A[0]).max()).max())
    ti, tj = rng.integers(0, n, samples), rng.integers(0, n, samples)
    ti[: min(n, samples // 2)] = tj[: min(n, samples // 2)]     # include diagonal positions
    Qt = np.ascontiguousarray(np.transpose(Q, (0, 2, 1)))
    I = np.zeros((L, n, n))
    I[0] = np.eye(n)
    o = orc.exact_samples(Qt, Q, ti, tj, C=I)
    return res, float(o["err"].max())


@pytest.mark.parametrize("cfg_idx,shape", [(0, (64, 64)), (3, (96, 40)), (1, (33, 33)), (2, (100, 7)), (4, (70, 45)), (0, (1, 1)), (4, (40, 33))])
def test_qr_against_the_oracle(cfg_idx, shape):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(shape[0], 3, shape[1])
    A = inputs.generate(cfg, "A")
    L = cfg.limbs
    Q, R = (host(t) for t in md.md_qr(dev(A)))
    Qo, Ro = orc.md_qr(A)
    kappa = np.linalg.cond(A.sum(axis=0))
    tol = shape[0] * kappa * 2.0 ** -(52 * L - 8)
    scale = np.abs(A[0]).max()
    assert np.abs((Q - Qo).sum(axis=0)).max() <= tol and np.abs((R - Ro).sum(axis=0)).max() <= tol * scale
    assert all(not np.tril(R[l], -1).any() for l in range(L)) and (np.diagonal(R[0]) >= 0).all()
    res, orth = residual_and_orthogonality(A, Q, R, 400, 1)
    bar = shape[0] * 2.0 ** -(52 * L - 6)
    assert res <= bar and orth <= bar, (res, orth, bar)


@pytest.mark.parametrize("n", [512, 2048])
def test_qr_at_working_precision_dd(n):
    """VERDICT r1 'done' criterion: 512 x 512 and 2048 x 2048 double double -- residual and orthogonality <= c n 2^-104."""
    cfg = inputs.CONFIGS[2].with_shape(n, 3, n)
    A = inputs.generate(cfg, "A")
    Qd, Rd, (total_ms, gemm_ms) = md.md_qr(dev(A), want_times=True)
    Q, R = host(Qd), host(Rd)
    assert not np.tril(R[0], -1).any() and not np.tril(R[1], -1).any() and (np.diagonal(R[0]) > 0).all()
    res, orth = residual_and_orthogonality(A, Q, R, 3000, n)
    bar = 8 * n * 2.0 ** -104
    print(f"md_qr dd {n}x{n}: |A-QR|/max|A| = {res:.3g}, |Q^TQ-I| = {orth:.3g} (bar {bar:.3g}); {total_ms:.1f} ms, {100 * gemm_ms / total_ms:.0f} % in md_gemm")
    assert res <= bar and orth <= bar, (res, orth, bar)
    # the leading limbs against the library routine in double precision (unique factorisation: diag(R) > 0)
    q, r = np.linalg.qr(A.sum(axis=0))
    s = np.sign(np.diagonal(r))
    assert np.abs(R[0] - r * s[:, None]).max() <= 1e-9 * np.abs(A[0]).max() * np.sqrt(n)


def test_qr_quad_double_and_tall():
    cfg = inputs.CONFIGS[4].with_shape(300, 3, 130)
    A = inputs.generate(cfg, "A")
    Q, R = (host(t) for t in md.md_qr(dev(A)))
    res, orth = residual_and_orthogonality(A, Q, R, 1500, 9)
    bar = 8 * 300 * 2.0 ** -208
    assert res <= bar and orth <= bar, (res, orth, bar)
    assert (np.diagonal(R[0]) > 0).all()


def test_qr_closed_forms_and_errors():
    rng = np.random.default_rng(5)
    A = np.zeros((2, 40, 40))
    A[0] = np.triu(rng.standard_normal((40, 40)))
    A[0][np.diag_indices(40)] = np.abs(np.diagonal(A[0])) + 1.0
    Q, R = (host(t) for t in md.md_qr(dev(A)))
    assert (R == A).all() and (Q[0] == np.eye(40)).all() and not Q[1].any()     # an upper triangular A is its own R, exactly
    lib = md.lib()
    assert lib.md_qr_scratch_bytes(4, 5, 2) == 0 and lib.md_qr_scratch_bytes(4, 4, 8) == 0
    assert lib.md_qr(4, 5, 2, None, None, None, None, 0, None, None) == md.MD_ERR_BAD_ARG

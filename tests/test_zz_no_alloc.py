"""md_gemm_static (include/mdgemm.h): md_gemm for callers that can not allocate -- the workspace is a 64 MiB file-scope device array
inside the library (csrc/static_gemm.cu).  Checked against the existing path (md_gemm with a registered workspace): the same
kernels run, so the results must not differ in a bit (the bar every path-against-path test of this suite uses), on two calls in a
row and with a call of another shape in between (the array keeps the last call's contents); plus the limit, the status word and
that the calls really allocate nothing.  Collected last on purpose (pytest -x): a failure here hides no other test."""
import numpy as np
import pytest
import torch

from oracle import md_oracle as orc
from paper_2607_06881_b200 import binding as md
from paper_2607_06881_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = {2: 1e-28, 4: 1e-58}
# (config, shape): the one-launch kernel (64^3), the two-launch path on small tiles with ragged edges, a problem of several waves
# with a stream-K tail on the large tiles, quad double
CASES = [(0, (64, 64, 64)), (1, (333, 257, 190)), (3, (448, 448, 448)), (4, (70, 45, 91)), (4, (256, 256, 256))]


def gen(cfg_idx, m, n, k):
    cfg = inputs.CONFIGS[cfg_idx].with_shape(m, n, k)
    return cfg, inputs.generate(cfg, "A"), inputs.generate(cfg, "B")


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def reset_options():
    for key in (md.MD_OPT_QUARTERS, md.MD_OPT_ORDERS, md.MD_OPT_SLICE_BITS, md.MD_OPT_K_CHUNK, md.MD_OPT_FUSED_PREP, md.MD_OPT_TILE,
                md.MD_OPT_ONE_LAUNCH, md.MD_OPT_TILE_SCHEDULE, md.MD_OPT_RASTER_GROUP):
        md.md_set_option(key, 0)


def reference(cfg, dA, dB):
    """the existing path: md_gemm on a registered, caller-owned workspace (the paper's quarter count, as md_gemm_static uses)"""
    with md.Workspace(cfg.m, cfg.n, cfg.k, cfg.limbs, 4 * cfg.limbs):
        C = md.md_gemm(dA, dB)
        assert md.md_read_flags() == 0
    return C


@pytest.mark.parametrize("cfg_idx,shape", CASES)
def test_two_calls_in_a_row_equal_md_gemm_bit_for_bit(cfg_idx, shape):
    reset_options()
    cfg, A, B = gen(cfg_idx, *shape)
    dA, dB = dev(A), dev(B)
    want = reference(cfg, dA, dB)
    assert md.md_gemm_static_bytes(cfg.m, cfg.n, cfg.k, cfg.limbs) <= md.md_static_scratch_bytes()
    C1, C2 = torch.full_like(want, float("nan")), torch.full_like(want, float("nan"))
    md.md_gemm_static(dA, dB, C1)      # no workspace is registered here
    md.md_gemm_static(dA, dB, C2)      # ... and the array now holds the first call's quarter planes, exponents and flags
    assert md.md_gemm_static_read_flags() == 0
    assert bool((C1 == want).all()) and bool((C2 == want).all())
    if cfg.m * cfg.n <= 100000:       # and the result is right, not just the same: against the exact product (oracle O1)
        r = orc.exact_all(A, B, C2.cpu().numpy())
        assert (r["err"] <= TOL[cfg.limbs] * r["W"]).all()


def test_a_call_of_another_shape_and_format_in_between_leaves_nothing_behind():
    reset_options()
    cfg, A, B = gen(1, 333, 257, 190)
    cfg2, A2, B2 = gen(4, 129, 200, 77)
    dA, dB, dA2, dB2 = dev(A), dev(B), dev(A2), dev(B2)
    want, want2 = reference(cfg, dA, dB), reference(cfg2, dA2, dB2)
    got = md.md_gemm_static(dA, dB)
    got2 = md.md_gemm_static(dA2, dB2)
    again = md.md_gemm_static(dA, dB)
    assert bool((got == want).all()) and bool((got2 == want2).all()) and bool((again == want).all())


def test_status_word_belongs_to_the_last_call():
    reset_options()
    cfg, A, B = gen(0, 96, 80, 200)
    bad = A.copy()
    bad[0, 5, 7] = np.nan
    md.md_gemm_static(dev(bad), dev(B))
    assert md.md_gemm_static_read_flags() & 1          # non-finite input
    C = md.md_gemm_static(dev(A), dev(B))
    assert md.md_gemm_static_read_flags() == 0         # cleared by the next call, not sticky
    assert bool((C == reference(cfg, dev(A), dev(B))).all())


def test_beyond_the_built_in_scratch_is_refused_with_its_own_status():
    reset_options()
    limit = md.md_static_scratch_bytes()
    assert limit == 64 << 20
    assert md.md_gemm_static_bytes(4096, 4096, 4096, 2) > limit
    assert 0 < md.md_gemm_static_bytes(448, 448, 448, 2) <= limit and 0 < md.md_gemm_static_bytes(256, 256, 256, 4) <= limit
    assert md.md_gemm_static_bytes(0, 4, 4, 2) == 0 and md.md_gemm_static_bytes(4, 4, 4, 3) == 0
    A = torch.zeros((2, 2048, 2048), dtype=torch.float64, device="cuda")
    C = torch.full((2, 2048, 2048), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(md.MdError) as exc:
        md.md_gemm_static(A, A, C)
    assert exc.value.status == md.MD_ERR_STATIC_LIMIT and "MD_ERR_STATIC_LIMIT" in str(exc.value)
    torch.cuda.synchronize()
    assert bool((C == 7.0).all())                      # nothing was enqueued


def test_the_calls_allocate_no_device_memory():
    reset_options()
    cfg, A, B = gen(1, 333, 257, 190)
    dA, dB = dev(A), dev(B)
    C = torch.empty((cfg.limbs, cfg.m, cfg.n), dtype=torch.float64, device="cuda")
    md.md_gemm_static(dA, dB, C)                       # first use: the module with the array and the kernels are loaded here
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(2):
        md.md_gemm_static(dA, dB, C)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_before - free_after < (1 << 20)        # device-wide free memory: a cudaMalloc inside the calls would show

"""CPU-only checks of the boundary: libmdgemm.so loads, exports every symbol include/mdgemm.h declares, and rejects bad
arguments before touching the GPU (no compute calls here)."""
import ctypes
import os
import re

import pytest

from paper_2607_06881_b200 import binding as md

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_06881_b200 import build
    build.build()
    return md.lib()


def header_symbols():
    text = open(os.path.join(ROOT, "include", "mdgemm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(md_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound(lib):
    declared = header_symbols()
    assert len(declared) >= 14
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(md.EXPORTED_SYMBOLS) == declared  # the binding covers exactly the header


def test_status_strings(lib):
    for code in (0, -1, -2, -3, -4, -5):
        assert lib.md_status_string(code)
    assert b"unknown" in lib.md_status_string(-99)


def test_argument_errors_need_no_gpu(lib):
    fake = ctypes.c_void_p(4096)  # non-null, aligned, never dereferenced: errors are argument-only
    assert lib.md_gemm(0, 4, 4, 2, fake, fake, fake, None) == md.MD_ERR_BAD_ARG
    assert lib.md_gemm(4, 4, 4, 3, fake, fake, fake, None) == md.MD_ERR_BAD_ARG
    assert lib.md_gemm(4, 4, 4, 2, None, fake, fake, None) == md.MD_ERR_BAD_ARG
    assert lib.md_gemm(4, 4, 4, 2, ctypes.c_void_p(4100), fake, fake, None) == md.MD_ERR_BAD_ARG  # misaligned
    # k budget: k * S <= 2^27 (eq. 5 generalised, R6): 2^24 passes the check, 2^24 + 1 does not
    # (md_gemm on double double chunks the contraction beyond it, R16; md_gemm_orders and quad double cannot)
    assert lib.md_gemm_orders(1, 1, 2 ** 24 + 1, 2, fake, fake, fake, None) == md.MD_ERR_K_TOO_LARGE
    assert lib.md_gemm(1, 1, 2 ** 24 + 1, 2, fake, fake, fake, None) == md.MD_ERR_WORKSPACE
    assert lib.md_gemm(1, 1, 2 ** 23 + 1, 4, fake, fake, fake, None) == md.MD_ERR_K_TOO_LARGE
    assert lib.md_gemm(1, 1, 2 ** 24, 2, fake, fake, fake, None) == md.MD_ERR_WORKSPACE  # passes the checks; no workspace
    assert lib.md_split(4, 4, 3, 8, 0, fake, fake, fake, None) == md.MD_ERR_BAD_ARG
    assert lib.md_split(4, 4, 2, 8, 2, fake, fake, fake, None) == md.MD_ERR_BAD_ARG
    assert lib.md_split(4, 4, 2, 73, 0, fake, fake, fake, None) == md.MD_ERR_BAD_ARG  # at most 72 quarters
    assert lib.md_renorm(4, 4, 2, 145, fake, fake, None) == md.MD_ERR_BAD_ARG
    # octo / hexa double (Table 2): k budget 2^27 / 32 and 2^27 / 64; only md_gemm has kernels for them
    assert lib.md_gemm(1, 1, 2 ** 22 + 1, 8, fake, fake, fake, None) == md.MD_ERR_K_TOO_LARGE
    assert lib.md_gemm(1, 1, 2 ** 21 + 1, 16, fake, fake, fake, None) == md.MD_ERR_K_TOO_LARGE
    assert lib.md_gemm(1, 1, 2 ** 21, 16, fake, fake, fake, None) == md.MD_ERR_WORKSPACE
    assert lib.md_renorm(4, 4, 2, 0, fake, fake, None) == md.MD_ERR_BAD_ARG
    # md_qgemm: counts without a plain-layout kernel are repacked into the registered workspace and run on the kernel md_gemm
    # would pick (the generic one if need be); beyond the generic maxima nothing exists
    assert lib.md_qgemm(4, 4, 4, 8, 32, 32, fake, fake, fake, fake, None) == md.MD_ERR_WORKSPACE
    assert lib.md_qgemm(4, 4, 4, 2, 8, 7, fake, fake, fake, fake, None) == md.MD_ERR_WORKSPACE
    assert lib.md_qgemm(4, 4, 4, 2, 12, 12, fake, fake, fake, fake, None) == md.MD_ERR_WORKSPACE
    assert lib.md_qgemm(4, 4, 4, 2, 17, 17, fake, fake, fake, fake, None) == md.MD_ERR_UNSUPPORTED   # dd: at most 16 quarters
    assert lib.md_qgemm(4, 4, 4, 2, 8, 16, fake, fake, fake, fake, None) == md.MD_ERR_UNSUPPORTED    # orders <= 2 quarters - 1
    assert lib.md_qgemm(4, 4, 4, 2, 16, 25, fake, fake, fake, fake, None) == md.MD_ERR_UNSUPPORTED   # dd: at most 24 orders
    assert lib.md_qgemm(4, 4, 4, 4, 25, 25, fake, fake, fake, fake, None) == md.MD_ERR_UNSUPPORTED   # qd: at most 24
    assert lib.md_qgemm(4, 4, 4, 2, 8, 8, fake, fake, None, None, None) == md.MD_ERR_BAD_ARG
    # every quarter count md_plan_quarters may return within the generic maxima has a kernel (R5, R15):
    # dd 1..16, qd 1..24, od 1..40, hd 1..72, and MD_OPT_ORDERS in [Q - 2, Q + 2] (and further: DESIGN.md R22)
    try:
        for limbs, qmax in ((2, 16), (4, 24), (8, 40), (16, 72)):
            for Q in range(3, qmax + 1):
                assert lib.md_set_option(md.MD_OPT_QUARTERS, Q) == md.MD_OK
                for S in (0, Q - 2, Q - 1, Q + 1, Q + 2):
                    assert lib.md_set_option(md.MD_OPT_ORDERS, S) == md.MD_OK
                    assert lib.md_gemm(8, 8, 8, limbs, fake, fake, fake, None) == md.MD_ERR_WORKSPACE, (limbs, Q, S)
                    assert lib.md_workspace_bytes(8, 8, 8, limbs) > 0
            assert lib.md_set_option(md.MD_OPT_ORDERS, 0) == md.MD_OK
            if qmax < 72:  # (72 is also the largest value MD_OPT_QUARTERS takes)
                assert lib.md_set_option(md.MD_OPT_QUARTERS, qmax + 1) == md.MD_OK
                assert lib.md_gemm(8, 8, 8, limbs, fake, fake, fake, None) == md.MD_ERR_UNSUPPORTED
    finally:
        lib.md_set_option(md.MD_OPT_QUARTERS, 0)
        lib.md_set_option(md.MD_OPT_ORDERS, 0)


def test_options_and_workspace_sizes(lib):
    assert lib.md_get_option(md.MD_OPT_QUARTERS) == 0 and lib.md_get_option(99) == -1
    base = lib.md_workspace_bytes(64, 64, 64, 2)
    # a quartered double double matrix has 8 times the size of a matrix of doubles
    # plus the fixed stream-K scratch of the fused GEMM: 256 tiles of 8 orders x 64 x 32 doubles + slab counters
    sk = 1024 + 256 * 8 * 64 * 32 * 8
    assert base >= 2 * 8 * 64 * 64 * 8 + sk and base < 2 * 8 * 64 * 64 * 8 + sk + 4096
    # the packed quarter planes are zero padded to whole CTA tiles (64 rows of A, 32 columns of B) and k-slabs of 8
    assert lib.md_workspace_bytes(65, 33, 9, 2) - lib.md_workspace_bytes(64, 32, 8, 2) == 8 * 8 * (128 * 16 + 64 * 16 - 64 * 8 - 32 * 8) + 256
    assert lib.md_set_option(md.MD_OPT_QUARTERS, 9) == 0
    assert lib.md_workspace_bytes(64, 64, 64, 2) >= 2 * 9 * 64 * 64 * 8
    assert lib.md_set_option(md.MD_OPT_QUARTERS, 0) == 0
    assert lib.md_workspace_bytes(64, 64, 64, 4) >= 2 * 16 * 64 * 64 * 8  # quad double: 16 times
    # octo double 32 times, hexa double 64 times (4 quarters per limb)
    assert lib.md_workspace_bytes(64, 64, 64, 8) >= 2 * 32 * 64 * 64 * 8
    assert lib.md_workspace_bytes(64, 64, 64, 16) >= 2 * 64 * 64 * 64 * 8
    assert lib.md_workspace_bytes(0, 64, 64, 2) == 0 and lib.md_workspace_bytes(64, 64, 64, 3) == 0
    assert lib.md_host_scratch_bytes(64, 64, 64, 2) >= base + 3 * 2 * 64 * 64 * 8
    assert lib.md_set_option(99, 1) == md.MD_ERR_BAD_ARG and lib.md_set_option(md.MD_OPT_QUARTERS, 99) == md.MD_ERR_BAD_ARG
    assert lib.md_set_workspace(None, 16) == md.MD_ERR_BAD_ARG
    assert lib.md_set_workspace(None, 0) == 0


def test_plan_slices_matches_a_brute_force_search(lib):
    """md_plan_slices (host only; R14): fewest slices Q that has a kernel, at the widest W with
    k * Q * 2^(2W) <= 2^53 (eq. 5 generalised), such that W * Q >= 13 * 4 * limbs (the paper's window,
    PAPER.md:47, :73); else the paper's (13, 4 * limbs).  Restated here as a plain search over all (Q, W)."""
    have = {2: (6, 7, 8, 9, 10), 4: (11, 12, 16, 17, 18), 8: (22, 32), 16: (44, 64)}
    for limbs in (2, 4, 8, 16):
        for k in (1, 64, 512, 1024, 2048, 4096, 5461, 5462, 8192, 2 ** 15, 2 ** 18, 2 ** 20):
            best = None
            for Q in have[limbs]:
                if Q >= 4 * limbs:
                    continue
                ok = [W for W in range(4, 25) if k * Q * 2 ** (2 * W) <= 2 ** 53 and W * Q >= 52 * limbs]
                if ok:
                    best = (max(ok), Q)
                    break
            want = best or (13, 4 * limbs)
            assert md.md_plan_slices(k, limbs) == want, (limbs, k)
    assert md.md_plan_slices(4096, 2) == (19, 6) and md.md_plan_slices(2048, 4) == (19, 11)
    assert md.md_plan_slices(1024, 8) == (19, 22) and md.md_plan_slices(512, 16) == (19, 44)
    fake_int = ctypes.c_int(0)
    assert lib.md_plan_slices(0, 2, ctypes.addressof(fake_int), ctypes.addressof(fake_int)) == md.MD_ERR_BAD_ARG
    assert lib.md_plan_slices(8, 3, ctypes.addressof(fake_int), ctypes.addressof(fake_int)) == md.MD_ERR_BAD_ARG


def test_slice_bits_option_and_its_k_budget(lib):
    fake = ctypes.c_void_p(4096)
    assert lib.md_set_option(md.MD_OPT_SLICE_BITS, 3) == md.MD_ERR_BAD_ARG
    assert lib.md_set_option(md.MD_OPT_SLICE_BITS, 25) == md.MD_ERR_BAD_ARG
    try:
        assert lib.md_set_option(md.MD_OPT_SLICE_BITS, 19) == md.MD_OK and lib.md_get_option(md.MD_OPT_SLICE_BITS) == 19
        assert lib.md_set_option(md.MD_OPT_QUARTERS, 6) == md.MD_OK
        # k * 6 * 2^38 <= 2^53  <=>  k <= 5461
        assert lib.md_gemm_orders(1, 1, 5462, 2, fake, fake, fake, None) == md.MD_ERR_K_TOO_LARGE
        assert lib.md_gemm_orders(1, 1, 5461, 2, fake, fake, fake, None) == md.MD_ERR_WORKSPACE
        assert lib.md_gemm(1, 1, 5462, 2, fake, fake, fake, None) == md.MD_ERR_WORKSPACE  # chunked (R16)
        assert lib.md_set_option(md.MD_OPT_QUARTERS, 5) == md.MD_OK    # 5 slices: the chunked kernel for md_gemm, the generic one for the orders
        assert lib.md_gemm(1, 1, 64, 2, fake, fake, fake, None) == md.MD_ERR_WORKSPACE
        assert lib.md_gemm_orders(1, 1, 64, 2, fake, fake, fake, None) == md.MD_ERR_WORKSPACE
        assert lib.md_set_option(md.MD_OPT_QUARTERS, 17) == md.MD_OK   # beyond the generic maximum of double double
        assert lib.md_gemm(1, 1, 64, 2, fake, fake, fake, None) == md.MD_ERR_UNSUPPORTED
    finally:
        lib.md_set_option(md.MD_OPT_SLICE_BITS, 0)
        lib.md_set_option(md.MD_OPT_QUARTERS, 0)


def test_compare_library_exports_its_header(lib):
    """libmdcompare.so (include/mdcompare.h, the paper's own two paths as comparison): every declared symbol exported."""
    from paper_2607_06881_b200 import compare as mdc
    text = open(os.path.join(ROOT, "include", "mdcompare.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = sorted(set(re.findall(r"\b(mdc_[a-z_]+)\s*\(", text)))
    assert declared == sorted(mdc.EXPORTED_SYMBOLS) and len(declared) == 3
    for name in declared:
        assert hasattr(mdc.lib(), name)
    assert mdc.lib().mdc_topdown_workspace_bytes(0, 4, 4, 2, 8) == 0


def test_plan_quarters_argument_errors(lib):
    fake = ctypes.c_void_p(4096)
    q = ctypes.c_int(0)
    assert lib.md_plan_scratch_bytes(0, 4, 4) == 0
    need = lib.md_plan_scratch_bytes(64, 32, 16)
    assert need >= 8 * (64 * 16 + 16 * 32 + 64 * 32) + 4 * (64 + 32)
    args = (fake, fake, fake, need, 0.0, ctypes.addressof(q), None, None)
    assert lib.md_plan_quarters(0, 32, 16, 2, *args) == md.MD_ERR_BAD_ARG
    assert lib.md_plan_quarters(64, 32, 16, 3, *args) == md.MD_ERR_BAD_ARG
    assert lib.md_plan_quarters(64, 32, 16, 2, fake, fake, fake, need - 1, 0.0, ctypes.addressof(q), None, None) == md.MD_ERR_WORKSPACE
    assert lib.md_plan_quarters(64, 32, 16, 2, fake, fake, fake, need, -1.0, ctypes.addressof(q), None, None) == md.MD_ERR_BAD_ARG


def test_chunk_option_and_chunked_plan(lib):
    assert lib.md_set_option(md.MD_OPT_K_CHUNK, 12) == md.MD_ERR_BAD_ARG  # a multiple of the k-slab depth 8
    assert lib.md_set_option(md.MD_OPT_K_CHUNK, 64) == md.MD_OK and lib.md_get_option(md.MD_OPT_K_CHUNK) == 64
    assert lib.md_set_option(md.MD_OPT_K_CHUNK, 0) == md.MD_OK
    # double double, k = 4096, chunks of at least 256: 5 slices of 21 bits (105 >= 104 bits), 2^53 / (5 * 2^42) = 409 -> 408
    assert md.md_plan_slices_chunked(4096, 2, 256) == (21, 5, 408)
    assert md.md_plan_slices_chunked(300, 2, 256) == (21, 5, 0)       # fits one chunk
    assert md.md_plan_slices_chunked(4096, 2, 1024) == (20, 6, 1360)  # no 5-slice chunk that long: 6 slices, one bit wider than unchunked
    assert md.md_plan_slices(4096, 2) == (19, 6)
    assert md.md_plan_slices_chunked(2048, 4, 256) == md.md_plan_slices(2048, 4) + (0,)    # quad double: no chunk that long
    assert md.md_plan_slices_chunked(2048, 4, 128) == (21, 10, 200)   # 10 slices of 21 bits (210 >= 208), 2^11 / 10 = 204 -> 200
    assert md.md_plan_slices_chunked(1024, 8, 64) == md.md_plan_slices(1024, 8) + (0,)     # octo double has no chunked kernel
    for W, Q, c in (md.md_plan_slices_chunked(4096, 2, 256), md.md_plan_slices_chunked(65536, 2, 64)):
        assert c % 8 == 0 and c * Q * 2 ** (2 * W) <= 2 ** 53 and W * Q >= 104

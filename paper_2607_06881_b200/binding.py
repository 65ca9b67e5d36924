"""Thin Python binding of libmdgemm.so (include/mdgemm.h): same names, argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; torch is used for device memory and streams.  There is
no CPU fallback: if the shared library is missing (run `python -m paper_2607_06881_b200.build`) or a call fails, an
exception is raised.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmdgemm.so")

MD_OK = 0
MD_ERR_BAD_ARG, MD_ERR_K_TOO_LARGE, MD_ERR_WORKSPACE, MD_ERR_CUDA, MD_ERR_UNSUPPORTED = -1, -2, -3, -4, -5
MD_ERR_STATIC_LIMIT = -6
MD_OPT_QUARTERS, MD_OPT_ORDERS, MD_OPT_SLICE_BITS, MD_OPT_HOST_BLOCKS, MD_OPT_K_CHUNK, MD_OPT_FUSED_PREP, MD_OPT_TILE, MD_OPT_RASTER_GROUP = 1, 2, 3, 4, 5, 6, 7, 8
MD_OPT_ONE_LAUNCH = 9
MD_OPT_TILE_SCHEDULE = 10

# every symbol include/mdgemm.h declares: name -> (restype, argtypes)
_c = ctypes
_SIGNATURES = {
    "md_set_option": (_c.c_int, [_c.c_int, _c.c_int]),
    "md_get_option": (_c.c_int, [_c.c_int]),
    "md_plan_slices": (_c.c_int, [_c.c_int, _c.c_int, _c.c_void_p, _c.c_void_p]),
    "md_plan_scratch_bytes": (_c.c_size_t, [_c.c_int] * 3),
    "md_plan_quarters": (_c.c_int, [_c.c_int] * 4 + [_c.c_void_p] * 3 + [_c.c_size_t, _c.c_double] + [_c.c_void_p] * 3),
    "md_auto_scratch_bytes": (_c.c_size_t, [_c.c_int] * 5),
    "md_gemm_auto": (_c.c_int, [_c.c_int] * 4 + [_c.c_void_p] * 4 + [_c.c_size_t, _c.c_double, _c.c_void_p, _c.c_void_p]),
    "md_split_literal": (_c.c_int, [_c.c_int] * 5 + [_c.c_void_p] * 4),
    "md_literal_scratch_bytes": (_c.c_size_t, [_c.c_int] * 6),
    "md_gemm_literal": (_c.c_int, [_c.c_int] * 4 + [_c.c_void_p] * 4 + [_c.c_size_t, _c.c_int, _c.c_void_p, _c.c_void_p]),
    "md_qr_scratch_bytes": (_c.c_size_t, [_c.c_int] * 3),
    "md_qr": (_c.c_int, [_c.c_int] * 3 + [_c.c_void_p] * 4 + [_c.c_size_t, _c.c_void_p, _c.c_void_p]),
    "md_plan_slices_chunked": (_c.c_int, [_c.c_int] * 3 + [_c.c_void_p] * 3),
    "md_split": (_c.c_int, [_c.c_int] * 5 + [_c.c_void_p] * 4),
    "md_qgemm": (_c.c_int, [_c.c_int] * 6 + [_c.c_void_p] * 5),
    "md_renorm": (_c.c_int, [_c.c_int] * 4 + [_c.c_void_p] * 3),
    "md_gemm": (_c.c_int, [_c.c_int] * 4 + [_c.c_void_p] * 4),
    "md_gemm_orders": (_c.c_int, [_c.c_int] * 4 + [_c.c_void_p] * 4),
    "md_workspace_bytes": (_c.c_size_t, [_c.c_int] * 4),
    "md_set_workspace": (_c.c_int, [_c.c_void_p, _c.c_size_t]),
    "md_read_flags": (_c.c_int, [_c.c_void_p, _c.c_void_p]),
    "md_host_scratch_bytes": (_c.c_size_t, [_c.c_int] * 4),
    "md_gemm_host": (_c.c_int, [_c.c_int] * 4 + [_c.c_void_p] * 4 + [_c.c_size_t, _c.c_void_p]),
    "md_profile_enable": (_c.c_int, [_c.c_int]),
    "md_profile_read": (_c.c_int, [_c.c_void_p, _c.c_void_p, _c.c_int]),
    "md_probe_dmma": (_c.c_int, [_c.c_int] * 3 + [_c.c_void_p] * 3),
    "md_static_scratch_bytes": (_c.c_size_t, []),
    "md_gemm_static_bytes": (_c.c_size_t, [_c.c_int] * 4),
    "md_gemm_static": (_c.c_int, [_c.c_int] * 4 + [_c.c_void_p] * 4),
    "md_gemm_static_read_flags": (_c.c_int, [_c.c_void_p, _c.c_void_p]),
    "md_launch_count": (_c.c_uint64, []),
    "md_status_string": (_c.c_char_p, [_c.c_int]),
}
EXPORTED_SYMBOLS = tuple(_SIGNATURES)

_lib = None


class MdError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {lib().md_status_string(status).decode()} ({status})")


def lib() -> ctypes.CDLL:
    """Load libmdgemm.so (once).  Raises if it has not been built: there is no fallback path."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2607_06881_b200.build` "
                              "(the CUDA extension is the product; there is no CPU fallback)")
        handle = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(handle, name)
            fn.restype, fn.argtypes = res, args
        _lib = handle
    return _lib


def _check(status: int, where: str):
    if status != MD_OK:
        raise MdError(status, where)


def _dev(t: torch.Tensor, dtype=torch.float64) -> int:
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise ValueError("expected a contiguous CUDA tensor of dtype %s" % dtype)
    return t.data_ptr()


def _stream(stream) -> int:
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream


def md_set_option(key: int, value: int):
    _check(lib().md_set_option(key, value), "md_set_option")


def md_get_option(key: int) -> int:
    return lib().md_get_option(key)


def md_plan_slices(k: int, limbs: int):
    """(slice bits W, slice count Q) of the k-adaptive split for contraction length k (include/mdgemm.h)."""
    bits, quarters = ctypes.c_int(0), ctypes.c_int(0)
    _check(lib().md_plan_slices(k, limbs, ctypes.addressof(bits), ctypes.addressof(quarters)), "md_plan_slices")
    return bits.value, quarters.value


def md_plan_slices_chunked(k: int, limbs: int, min_chunk: int = 256):
    """(W, Q, chunk) with chunked accumulation allowed (include/mdgemm.h, R16); chunk = 0: none needed."""
    bits, quarters, chunk = ctypes.c_int(0), ctypes.c_int(0), ctypes.c_int(0)
    _check(lib().md_plan_slices_chunked(k, limbs, min_chunk, ctypes.addressof(bits), ctypes.addressof(quarters),
                                        ctypes.addressof(chunk)), "md_plan_slices_chunked")
    return bits.value, quarters.value, chunk.value


def md_plan_quarters(A: torch.Tensor, B: torch.Tensor, rel_tol: float = 0.0, stream=None):
    """(Q, D): the quarter count this data needs for rel_tol (0 = the format's tolerance) and the measured spread D
    (include/mdgemm.h).  Synchronises."""
    limbs, m, k = A.shape
    n = B.shape[2]
    scratch = torch.empty(lib().md_plan_scratch_bytes(m, n, k), dtype=torch.uint8, device=A.device)
    q, d = ctypes.c_int(0), ctypes.c_int(0)
    _check(lib().md_plan_quarters(m, n, k, limbs, _dev(A), _dev(B), _dev(scratch, torch.uint8), scratch.numel(),
                                  rel_tol, ctypes.addressof(q), ctypes.addressof(d), _stream(stream)), "md_plan_quarters")
    return q.value, d.value


def md_workspace_bytes(m, n, k, limbs) -> int:
    return lib().md_workspace_bytes(m, n, k, limbs)


def md_set_workspace(ws: torch.Tensor | None):
    """Register a uint8 CUDA tensor (or None) as the library workspace.  The caller keeps it alive."""
    if ws is None:
        _check(lib().md_set_workspace(None, 0), "md_set_workspace")
    else:
        _check(lib().md_set_workspace(_dev(ws, torch.uint8), ws.numel()), "md_set_workspace")


def md_read_flags(stream=None) -> int:
    out = ctypes.c_uint32(0)
    _check(lib().md_read_flags(ctypes.addressof(out), _stream(stream)), "md_read_flags")
    return out.value


def md_split(planes: torch.Tensor, axis: int, quarters: int | None = None, stream=None):
    """planes [limbs, rows, cols] -> (quarter_planes [Q, rows, cols], exps int32[rows or cols])."""
    limbs, rows, cols = planes.shape
    Q = 4 * limbs if quarters is None else quarters
    qp = torch.empty((Q, rows, cols), dtype=torch.float64, device=planes.device)
    exps = torch.empty(rows if axis == 0 else cols, dtype=torch.int32, device=planes.device)
    _check(lib().md_split(rows, cols, limbs, Q, axis, _dev(planes), _dev(qp), _dev(exps, torch.int32),
                          _stream(stream)), "md_split")
    return qp, exps


def md_qgemm(Aq: torch.Tensor, Bq: torch.Tensor, limbs: int, want_orders: bool = False, want_C: bool = True,
             stream=None, orders_kept: int | None = None):
    """Aq [Q, m, k], Bq [Q, k, n] -> (order_planes [S, m, n] or None, C_planes [limbs, m, n] or None); S = orders_kept or Q."""
    Q, m, k = Aq.shape
    n = Bq.shape[2]
    S = Q if orders_kept is None else orders_kept
    assert Bq.shape[0] == Q and Bq.shape[1] == k
    orders = torch.empty((S, m, n), dtype=torch.float64, device=Aq.device) if want_orders else None
    C = torch.empty((limbs, m, n), dtype=torch.float64, device=Aq.device) if want_C else None
    _check(lib().md_qgemm(m, n, k, limbs, Q, S, _dev(Aq), _dev(Bq), None if orders is None else _dev(orders),
                          None if C is None else _dev(C), _stream(stream)), "md_qgemm")
    return orders, C


def md_renorm(order_planes: torch.Tensor, limbs: int, stream=None) -> torch.Tensor:
    S, m, n = order_planes.shape
    C = torch.empty((limbs, m, n), dtype=torch.float64, device=order_planes.device)
    _check(lib().md_renorm(m, n, limbs, S, _dev(order_planes), _dev(C), _stream(stream)), "md_renorm")
    return C


def md_gemm(A: torch.Tensor, B: torch.Tensor, C: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """C = A * B on limb planes: A [limbs, m, k], B [limbs, k, n] -> C [limbs, m, n].  Needs a registered workspace."""
    limbs, m, k = A.shape
    n = B.shape[2]
    assert B.shape[0] == limbs and B.shape[1] == k
    if C is None:
        C = torch.empty((limbs, m, n), dtype=torch.float64, device=A.device)
    _check(lib().md_gemm(m, n, k, limbs, _dev(A), _dev(B), _dev(C), _stream(stream)), "md_gemm")
    return C


def md_static_scratch_bytes() -> int:
    return lib().md_static_scratch_bytes()


def md_gemm_static_bytes(m: int, n: int, k: int, limbs: int) -> int:
    return lib().md_gemm_static_bytes(m, n, k, limbs)


def md_gemm_static(A: torch.Tensor, B: torch.Tensor, C: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """md_gemm with the library's built-in scratch (include/mdgemm.h): no workspace, no allocation inside the call (pass C to
    keep this wrapper from allocating the result either).  MdError(MD_ERR_STATIC_LIMIT) when the problem does not fit."""
    limbs, m, k = A.shape
    n = B.shape[2]
    assert B.shape[0] == limbs and B.shape[1] == k
    if C is None:
        C = torch.empty((limbs, m, n), dtype=torch.float64, device=A.device)
    _check(lib().md_gemm_static(m, n, k, limbs, _dev(A), _dev(B), _dev(C), _stream(stream)), "md_gemm_static")
    return C


def md_gemm_static_read_flags(stream=None) -> int:
    out = ctypes.c_uint32(0)
    _check(lib().md_gemm_static_read_flags(ctypes.addressof(out), _stream(stream)), "md_gemm_static_read_flags")
    return out.value


def md_gemm_auto(A: torch.Tensor, B: torch.Tensor, C: torch.Tensor | None = None, rel_tol: float = 0.0, stream=None):
    """md_plan_quarters + md_gemm in one call (include/mdgemm.h).  Returns (C, quarters used).  Allocates the scratch for the
    paper's count first and again if the plan asks for more.  Synchronises."""
    limbs, m, k = A.shape
    n = B.shape[2]
    if C is None:
        C = torch.empty((limbs, m, n), dtype=torch.float64, device=A.device)
    q = ctypes.c_int(0)
    want = 0
    for _ in range(2):
        scratch = torch.empty(lib().md_auto_scratch_bytes(m, n, k, limbs, want), dtype=torch.uint8, device=A.device)
        st = lib().md_gemm_auto(m, n, k, limbs, _dev(A), _dev(B), _dev(C), _dev(scratch, torch.uint8), scratch.numel(), rel_tol,
                                ctypes.addressof(q), _stream(stream))
        if st != MD_ERR_WORKSPACE or q.value == want or q.value == 0:
            break
        want = q.value
    _check(st, "md_gemm_auto")
    return C, q.value


MD_LITERAL_NO_EQ8, MD_LITERAL_SIGN_GROUPS = 1, 2


def md_split_literal(planes: torch.Tensor, quarters: int | None = None, flags: int = 0, stream=None):
    """Algorithm L (include/mdgemm.h): planes [limbs, rows, cols] -> (parts [Q, rows, cols], per-element exponents int32 [rows, cols])."""
    limbs, rows, cols = planes.shape
    Q = 4 * limbs if quarters is None else quarters
    qp = torch.empty((Q, rows, cols), dtype=torch.float64, device=planes.device)
    exps = torch.empty((rows, cols), dtype=torch.int32, device=planes.device)
    _check(lib().md_split_literal(rows, cols, limbs, Q, flags, _dev(planes), _dev(qp), _dev(exps, torch.int32), _stream(stream)),
           "md_split_literal")
    return qp, exps


def md_gemm_literal(A: torch.Tensor, B: torch.Tensor, C: torch.Tensor | None = None, flags: int = 0, stream=None, scratch=None):
    """The paper's exponent-class product (include/mdgemm.h).  Returns (C, info dict).  Sizes the scratch for no spread first and
    again with the counts the data needs.  Synchronises."""
    limbs, m, k = A.shape
    n = B.shape[2]
    if C is None:
        C = torch.empty((limbs, m, n), dtype=torch.float64, device=A.device)
    info = (ctypes.c_int32 * 8)()
    planes = orders = 0
    st = MD_ERR_WORKSPACE
    for _ in range(2):
        need = lib().md_literal_scratch_bytes(m, n, k, limbs, planes, orders)
        if need == 0:
            raise MdError(MD_ERR_UNSUPPORTED, "md_literal_scratch_bytes")
        if scratch is None or scratch.numel() < need:
            scratch = None
            scratch = torch.empty(need, dtype=torch.uint8, device=A.device)
        st = lib().md_gemm_literal(m, n, k, limbs, _dev(A), _dev(B), _dev(C), _dev(scratch, torch.uint8), scratch.numel(), flags,
                                   ctypes.addressof(info), _stream(stream))
        if st != MD_ERR_WORKSPACE:
            break
        planes, orders = info[4], info[5]
    _check(st, "md_gemm_literal")
    keys = ("zminA", "zmaxA", "zminB", "zmaxB", "planes", "orders", "pairs", "launches")
    return C, dict(zip(keys, (int(v) for v in info)))


def md_qr(A: torch.Tensor, want_times: bool = False, stream=None):
    """Blocked Householder QR on top of md_gemm (include/mdgemm.h): A [limbs, m, n] -> (Q [limbs, m, n], R [limbs, n, n]) with
    diag(R) >= 0; with want_times also (total ms, ms inside the md_gemm path)."""
    limbs, m, n = A.shape
    Q = torch.empty((limbs, m, n), dtype=torch.float64, device=A.device)
    R = torch.empty((limbs, n, n), dtype=torch.float64, device=A.device)
    need = lib().md_qr_scratch_bytes(m, n, limbs)
    if need == 0:
        raise MdError(MD_ERR_UNSUPPORTED, "md_qr_scratch_bytes")
    scratch = torch.empty(need, dtype=torch.uint8, device=A.device)
    times = (ctypes.c_float * 2)()
    _check(lib().md_qr(m, n, limbs, _dev(A), _dev(Q), _dev(R), _dev(scratch, torch.uint8), scratch.numel(),
                       ctypes.addressof(times) if want_times else None, _stream(stream)), "md_qr")
    return (Q, R, (float(times[0]), float(times[1]))) if want_times else (Q, R)


def md_gemm_orders(A: torch.Tensor, B: torch.Tensor, stream=None) -> torch.Tensor:
    limbs, m, k = A.shape
    n = B.shape[2]
    S = md_get_option(MD_OPT_ORDERS) or md_get_option(MD_OPT_QUARTERS) or 4 * limbs
    out = torch.empty((S, m, n), dtype=torch.float64, device=A.device)
    _check(lib().md_gemm_orders(m, n, k, limbs, _dev(A), _dev(B), _dev(out), _stream(stream)), "md_gemm_orders")
    return out


def md_host_scratch_bytes(m, n, k, limbs) -> int:
    return lib().md_host_scratch_bytes(m, n, k, limbs)


def md_gemm_host(A_host: torch.Tensor, B_host: torch.Tensor, C_host: torch.Tensor, scratch: torch.Tensor, stream=None):
    """End-to-end call on HOST tensors (pinned recommended); `scratch` is a uint8 CUDA tensor."""
    limbs, m, k = A_host.shape
    n = B_host.shape[2]
    for t in (A_host, B_host, C_host):
        if t.is_cuda or not t.is_contiguous() or t.dtype != torch.float64:
            raise ValueError("md_gemm_host takes contiguous float64 HOST tensors")
    _check(lib().md_gemm_host(m, n, k, limbs, A_host.data_ptr(), B_host.data_ptr(), C_host.data_ptr(),
                              _dev(scratch, torch.uint8), scratch.numel(), _stream(stream)), "md_gemm_host")
    return C_host


def md_profile_enable(capacity: int):
    _check(lib().md_profile_enable(capacity), "md_profile_enable")


def md_profile_read(capacity: int):
    """Returns (split_ms list, gemm_ms list) for the calls recorded since md_profile_enable."""
    split = (ctypes.c_float * max(capacity, 1))()
    gemm = (ctypes.c_float * max(capacity, 1))()
    count = lib().md_profile_read(split, gemm, capacity)
    if count < 0:
        raise MdError(count, "md_profile_read")
    return list(split[:count]), list(gemm[:count])


def md_probe_dmma(blocks: int, warps_per_block: int, iters: int, sink: torch.Tensor | None = None, stream=None) -> int:
    """Enqueue the register-only DMMA calibration kernel; returns the FP64 flops it issues (time it with CUDA events)."""
    flops = ctypes.c_uint64(0)
    _check(lib().md_probe_dmma(blocks, warps_per_block, iters, None if sink is None else _dev(sink),
                               ctypes.addressof(flops), _stream(stream)), "md_probe_dmma")
    return flops.value


def md_launch_count() -> int:
    return lib().md_launch_count()


class Workspace:
    """Allocates and registers the md_gemm workspace for one problem shape (context manager)."""

    def __init__(self, m, n, k, limbs, quarters: int = 0, device="cuda", bits: int = 0, orders: int = 0):
        md_set_option(MD_OPT_QUARTERS, 0 if quarters == 4 * limbs else quarters)
        md_set_option(MD_OPT_ORDERS, orders)
        md_set_option(MD_OPT_SLICE_BITS, 0 if bits == 13 else bits)
        nbytes = md_workspace_bytes(m, n, k, limbs)
        if nbytes == 0:
            raise ValueError("bad shape for workspace")
        self.buffer = torch.empty(nbytes, dtype=torch.uint8, device=device)
        md_set_workspace(self.buffer)

    def close(self):
        md_set_workspace(None)
        md_set_option(MD_OPT_QUARTERS, 0)
        md_set_option(MD_OPT_ORDERS, 0)
        md_set_option(MD_OPT_SLICE_BITS, 0)
        self.buffer = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

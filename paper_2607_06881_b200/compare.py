"""Thin Python binding of libmdcompare.so (include/mdcompare.h): the PAPER'S OWN two paths on B200 -- the materialised
top-down product through one plain DGEMM (cuBLAS) and the CUDA-core classical multiple-double GEMM -- as comparison
beside the product.  Argument marshalling only; nothing in binding.py / md_gemm uses it.
"""
from __future__ import annotations

import ctypes
import os

import torch

from . import binding as _md

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmdcompare.so")
_c = ctypes
_SIGNATURES = {
    "mdc_topdown_workspace_bytes": (_c.c_size_t, [_c.c_int] * 5),
    "mdc_topdown_gemm": (_c.c_int, [_c.c_int] * 5 + [_c.c_void_p] * 5 + [_c.c_size_t, _c.c_void_p, _c.c_void_p]),
    "mdc_classic_gemm": (_c.c_int, [_c.c_int] * 4 + [_c.c_void_p] * 4),
}
EXPORTED_SYMBOLS = tuple(_SIGNATURES)
_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _md.lib()  # libmdgemm.so first (md_split / md_renorm are called through its C-ABI)
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2607_06881_b200.build`")
        handle = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(handle, name)
            fn.restype, fn.argtypes = res, args
        _lib = handle
    return _lib


def mdc_topdown_workspace_bytes(m, n, k, limbs, quarters) -> int:
    return lib().mdc_topdown_workspace_bytes(m, n, k, limbs, quarters)


def mdc_topdown_gemm(A: torch.Tensor, B: torch.Tensor, quarters: int | None = None, want_orders: bool = False,
                     want_times: bool = False, ws: torch.Tensor | None = None, stream=None):
    """A [limbs, m, k], B [limbs, k, n] -> C [limbs, m, n] (and Cbar as order planes [Q, m, n], stage times in ms:
    split, construction of Atil, DGEMM, recombination)."""
    limbs, m, k = A.shape
    n = B.shape[2]
    Q = 4 * limbs if quarters is None else quarters
    if ws is None:
        ws = torch.empty(mdc_topdown_workspace_bytes(m, n, k, limbs, Q), dtype=torch.uint8, device=A.device)
    C = torch.empty((limbs, m, n), dtype=torch.float64, device=A.device)
    orders = torch.empty((Q, m, n), dtype=torch.float64, device=A.device) if want_orders else None
    times = (ctypes.c_float * 4)() if want_times else None
    st = lib().mdc_topdown_gemm(m, n, k, limbs, Q, _md._dev(A), _md._dev(B), _md._dev(C),
                                None if orders is None else _md._dev(orders), _md._dev(ws, torch.uint8), ws.numel(),
                                _md._stream(stream), None if times is None else ctypes.addressof(times))
    _md._check(st, "mdc_topdown_gemm")
    return C, orders, (list(times) if times is not None else None)


def mdc_classic_gemm(A: torch.Tensor, B: torch.Tensor, stream=None) -> torch.Tensor:
    limbs, m, k = A.shape
    n = B.shape[2]
    C = torch.empty((limbs, m, n), dtype=torch.float64, device=A.device)
    _md._check(lib().mdc_classic_gemm(m, n, k, limbs, _md._dev(A), _md._dev(B), _md._dev(C), _md._stream(stream)),
               "mdc_classic_gemm")
    return C

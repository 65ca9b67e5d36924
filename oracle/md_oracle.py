"""ctypes loader for the CPU oracle (oracle/md_oracle.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from paper_2607_06881_b200 (the CUDA path) and the CUDA path imports nothing from here.
The wrappers only marshal numpy arrays; every arithmetic step is in md_oracle.cpp.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int32)
_lp = ctypes.POINTER(ctypes.c_int64)


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        import importlib.util
        spec = importlib.util.spec_from_file_location("_md_oracle_build", os.path.join(_HERE, "build.py"))
        mod = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mod)
        _lib = ctypes.CDLL(mod.build())
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def split(planes: np.ndarray, axis: int, quarters: int | None = None, want_remainder: bool = False, bits: int = 13):
    """O2.  planes [limbs, rows, cols] -> (quarter_planes [Q, rows, cols], exps int32, remainder or None).
    bits = slice width (13 = the paper's quarter; other widths: DESIGN.md R14)."""
    planes = _f64(planes)
    limbs, rows, cols = planes.shape
    Q = 4 * limbs if quarters is None else quarters
    qp = np.empty((Q, rows, cols), dtype=np.float64)
    exps = np.empty(rows if axis == 0 else cols, dtype=np.int32)
    rem = np.empty_like(planes) if want_remainder else None
    lib().oracle_split_w(rows, cols, limbs, Q, bits, axis, _d(planes), _d(qp), exps.ctypes.data_as(_ip), _d(rem))
    return qp, exps, rem


def orders_int(Aq, expA, Bq, expB, orders: int | None = None, want_raw: bool = False, bits: int = 13):
    """O3, int64 digit route.  Aq [Q, m, k], Bq [Q, k, n] -> order planes [S, m, n] (and raw int64 sums)."""
    Aq, Bq = _f64(Aq), _f64(Bq)
    Q, m, k = Aq.shape
    n = Bq.shape[2]
    S = Q if orders is None else orders
    out = np.empty((S, m, n), dtype=np.float64)
    raw = np.empty((S, m, n), dtype=np.int64) if want_raw else None
    expA = np.ascontiguousarray(expA, dtype=np.int32)
    expB = np.ascontiguousarray(expB, dtype=np.int32)
    lib().oracle_orders_int_w(m, n, k, Q, S, bits, _d(Aq), expA.ctypes.data_as(_ip), _d(Bq), expB.ctypes.data_as(_ip),
                              _d(out), None if raw is None else raw.ctypes.data_as(_lp))
    return (out, raw) if want_raw else out


def orders_int_samples(Aq, expA, Bq, expB, si, sj, orders: int | None = None, bits: int = 13):
    """O3, int64 digit route at sampled positions: returns [nsamples, S]."""
    Aq, Bq = _f64(Aq), _f64(Bq)
    Q, m, k = Aq.shape
    n = Bq.shape[2]
    S = Q if orders is None else orders
    si = np.ascontiguousarray(si, dtype=np.int64)
    sj = np.ascontiguousarray(sj, dtype=np.int64)
    out = np.empty((si.size, S), dtype=np.float64)
    expA = np.ascontiguousarray(expA, dtype=np.int32)
    expB = np.ascontiguousarray(expB, dtype=np.int32)
    lib().oracle_orders_int_samples_w(m, n, k, Q, S, bits, _d(Aq), expA.ctypes.data_as(_ip), _d(Bq),
                                      expB.ctypes.data_as(_ip), ctypes.c_int64(si.size), si.ctypes.data_as(_lp),
                                      sj.ctypes.data_as(_lp), _d(out))
    return out


def orders_fp64(Aq, Bq, orders: int | None = None):
    """O3, plain fp64 route."""
    Aq, Bq = _f64(Aq), _f64(Bq)
    Q, m, k = Aq.shape
    n = Bq.shape[2]
    S = Q if orders is None else orders
    out = np.empty((S, m, n), dtype=np.float64)
    lib().oracle_orders_fp64(m, n, k, Q, S, _d(Aq), _d(Bq), _d(out))
    return out


def renorm(order_planes, limbs: int):
    """O4.  order planes [S, m, n] -> C planes [limbs, m, n] (exact sum, rounded limb by limb)."""
    order_planes = _f64(order_planes)
    S, m, n = order_planes.shape
    C = np.empty((limbs, m, n), dtype=np.float64)
    lib().oracle_renorm(m, n, limbs, S, _d(order_planes), _d(C))
    return C


def exact_samples(A, B, si, sj, C=None, out_limbs: int = 0, want_W: bool = True):
    """O1 at the sampled positions.  Returns dict(err=|C - C_exact|, W=(|A||B|)_ij, exact=[ns, out_limbs])."""
    A, B = _f64(A), _f64(B)
    limbs, m, k = A.shape
    n = B.shape[2]
    si = np.ascontiguousarray(si, dtype=np.int64)
    sj = np.ascontiguousarray(sj, dtype=np.int64)
    ns = si.size
    err = np.empty(ns) if C is not None else None
    W = np.empty(ns) if want_W else None
    ex = np.empty((ns, out_limbs)) if out_limbs else None
    if C is not None:
        C = _f64(C)
        assert C.shape == (limbs, m, n)
    lib().oracle_exact_samples(m, n, k, limbs, _d(A), _d(B), _d(C), ctypes.c_int64(ns), si.ctypes.data_as(_lp),
                               sj.ctypes.data_as(_lp), _d(err), _d(W), _d(ex), out_limbs)
    return {"err": err, "W": W, "exact": ex}


def exact_all(A, B, C=None, out_limbs: int = 0):
    """O1 on every output position (small matrices only).  Arrays come back shaped [m, n] (+[out_limbs])."""
    m, n = A.shape[1], B.shape[2]
    ii, jj = np.meshgrid(np.arange(m), np.arange(n), indexing="ij")
    r = exact_samples(A, B, ii.ravel(), jj.ravel(), C, out_limbs)
    return {key: (None if v is None else v.reshape((m, n) + v.shape[1:])) for key, v in r.items()}


def exact_sum(x, limbs: int):
    x = _f64(x).ravel()
    out = np.empty(limbs)
    lib().oracle_exact_sum(x.size, _d(x), limbs, _d(out))
    return out


def exact_dot(x, y, limbs: int):
    x, y = _f64(x).ravel(), _f64(y).ravel()
    out = np.empty(limbs)
    lib().oracle_exact_dot(x.size, _d(x), _d(y), limbs, _d(out))
    return out


def classic_gemm(A, B):
    """O5.  Classical multiple-double GEMM on the limb planes."""
    A, B = _f64(A), _f64(B)
    limbs, m, k = A.shape
    n = B.shape[2]
    C = np.empty((limbs, m, n))
    lib().oracle_classic_gemm(m, n, k, limbs, _d(A), _d(B), _d(C))
    return C


def md_gemm_rows(A, B, row0: int = 0, row1: int | None = None, quarters: int | None = None,
                 orders: int | None = None, bits: int = 13):
    """The paper's five steps through the oracle: rows [row0,row1) of C = A*B."""
    A, B = _f64(A), _f64(B)
    limbs, m, k = A.shape
    n = B.shape[2]
    row1 = m if row1 is None else row1
    Q = 4 * limbs if quarters is None else quarters
    S = Q if orders is None else orders
    C = np.empty((limbs, row1 - row0, n))
    lib().oracle_md_gemm_rows_w(m, n, k, limbs, Q, S, bits, _d(A), _d(B), row0, row1, _d(C))
    return C


def plan_quarters(A, B, rel_tol: float, bits: int = 13):
    """DESIGN.md R15: the smallest quarter count whose error bound k (Q+3) 2^(E_i+F_j-bits Q-2) stays below
    rel_tol (|A||B|)_ij at every position.  Returns (Q, D), D = max_ij E_i + F_j - ilogb((|A_0||B_0|)_ij)."""
    A, B = _f64(A), _f64(B)
    limbs, m, k = A.shape
    n = B.shape[2]
    D = ctypes.c_int32(0)
    f = lib().oracle_plan_quarters
    f.restype = ctypes.c_int
    Q = f(m, n, k, limbs, bits, _d(A), _d(B), ctypes.c_double(rel_tol), ctypes.byref(D))
    return int(Q), int(D.value)


def md_gemm_rows_chunked(A, B, chunk: int, quarters: int, bits: int, row0: int = 0, row1: int | None = None):
    """DESIGN.md R16: the five steps with the order sums formed exactly per chunk of the contraction."""
    A, B = _f64(A), _f64(B)
    limbs, m, k = A.shape
    n = B.shape[2]
    row1 = m if row1 is None else row1
    C = np.empty((limbs, row1 - row0, n))
    lib().oracle_md_gemm_rows_chunked_w(m, n, k, limbs, quarters, quarters, bits, chunk, _d(A), _d(B), row0, row1, _d(C))
    return C


def quarter_double(x: float):
    """R17: the four 13-bit parts of one double on its own exponent."""
    out = (ctypes.c_double * 4)()
    f = lib().oracle_quarter_double
    f.argtypes = [ctypes.c_double, ctypes.POINTER(ctypes.c_double)]
    f(float(x), out)
    return list(out)


def eq7(limbs_values):
    """R18, eq. (7) on one multiple double: returns (new limbs, carries)."""
    x = _f64(np.array(limbs_values, dtype=np.float64))
    carry = np.zeros_like(x)
    lib().oracle_eq7(x.size, _d(x), _d(carry))
    return x, carry


def eq8(d, e: int):
    """R19, eq. (8) on the quarters of one element of exponent e."""
    d = _f64(np.array(d, dtype=np.float64))
    lib().oracle_eq8(d.size, int(e), _d(d))
    return d


def split_literal(planes, quarters: int | None = None, apply_eq8: bool = True, want_remainder: bool = False):
    """Algorithm L (R17-R19): planes [limbs, rows, cols] -> (quarter planes [Q, rows, cols], per-ELEMENT exponents
    int32 [rows, cols], remainder [2 limbs, rows, cols] or None)."""
    planes = _f64(planes)
    limbs, rows, cols = planes.shape
    Q = 4 * limbs if quarters is None else quarters
    qp = np.empty((Q, rows, cols), dtype=np.float64)
    exps = np.empty((rows, cols), dtype=np.int32)
    rem = np.empty((2 * limbs, rows, cols), dtype=np.float64) if want_remainder else None
    lib().oracle_split_literal(rows, cols, limbs, Q, int(apply_eq8), _d(planes), _d(qp), exps.ctypes.data_as(_ip), _d(rem))
    return qp, exps, rem


def md_gemm_literal(A, B, quarters: int | None = None, apply_eq8: bool = True, sign_groups: bool = False):
    """The paper's literal product (R20-R22): exponent classes A_0..A_12 (x sign groups), exact order sums per class
    pair, exact recombination.  Returns (C [limbs, m, n], info = (zminA, zmaxA, zminB, zmaxB))."""
    A, B = _f64(A), _f64(B)
    limbs, m, k = A.shape
    n = B.shape[2]
    Q = 4 * limbs if quarters is None else quarters
    C = np.empty((limbs, m, n))
    info = np.zeros(4, dtype=np.int32)
    lib().oracle_md_gemm_literal(m, n, k, limbs, Q, int(apply_eq8), int(sign_groups), _d(A), _d(B), _d(C), info.ctypes.data_as(_ip))
    return C, tuple(int(v) for v in info)


def mdx_op(op: str, a, b=None):
    """One scalar multiple-double operation of O7 ('add', 'sub', 'mul', 'div', 'sqrt') on limb vectors."""
    a = _f64(np.array(a, dtype=np.float64))
    b = _f64(np.array(a if b is None else b, dtype=np.float64))
    out = np.empty_like(a)
    lib().oracle_mdx_op(a.size, {"add": 0, "sub": 1, "mul": 2, "div": 3, "sqrt": 4}[op], _d(a), _d(b), _d(out))
    return out


def md_qr(A):
    """O7: unblocked Householder QR in multiple-double arithmetic.  A [limbs, m, n] (m >= n) -> (Q [limbs, m, n], R [limbs, n, n]),
    diag(R) >= 0."""
    A = _f64(A)
    limbs, m, n = A.shape
    assert m >= n
    Q = np.empty((limbs, m, n))
    R = np.empty((limbs, n, n))
    lib().oracle_md_qr(m, n, limbs, _d(A), _d(Q), _d(R))
    return Q, R

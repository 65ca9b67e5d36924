"""Seeded synthetic inputs for the five BASELINE.json configs (plus two wider-format configs, CONFIGS[5:]).

This module is shared by the CPU oracle's tests and by the CUDA path's tests / bench.  It holds
NONE of the method's arithmetic (no splitting, no products, no renormalisation): only a stateless
counter-based random generator and the input recipes of BASELINE.json `configs` (restated in
DESIGN.md "Input recipe").  The paper itself only says "In all experiments, random numbers were
generated" (section 4.1), so these synthetic matrices stand in for its workloads.

Layout of everything returned: float64 ndarray ``[limbs, rows, cols]``, C-contiguous (limb planes,
each row-major) -- the layout `include/mdgemm.h` takes.

Every element is a pure function of (seed, matrix id, stream, global row, global col), so any
sub-block of a matrix can be regenerated without materialising the whole matrix.
"""
from __future__ import annotations

import dataclasses
import numpy as np

_U64 = np.uint64
_MASK = (1 << 64) - 1


@dataclasses.dataclass(frozen=True)
class Config:
    """One BASELINE.json config: C[m,n] = A[m,k] * B[k,n] with `limbs` fp64 limb planes."""
    index: int
    name: str
    m: int
    n: int
    k: int
    limbs: int
    seed: int
    dist: str  # "uniform" | "uniform_exp8" | "normal" | "wide30"
    # Quarters per element (= kept product orders) this config is run with.  The paper's count is 4 per limb
    # (PAPER.md:73, :80); config 3 "stresses balancing/quarter count" (BASELINE.json) and is run with 9, see
    # DESIGN.md reading R5.  This is a parameter handed to md_set_option, not part of the input data.
    quarters: int = 0
    # Slice width in bits: 13 = the paper's quarter.  Other widths are the k-adaptive variant (DESIGN.md
    # R14), again a parameter handed to md_set_option, not part of the input data.
    bits: int = 13
    # Kept product orders S (MD_OPT_ORDERS; the paper's C_1..C_S).  0 = quarters, the paper's set.
    orders: int = 0

    def __post_init__(self):
        if self.quarters == 0:
            object.__setattr__(self, "quarters", 4 * self.limbs)
        if self.orders == 0:
            object.__setattr__(self, "orders", self.quarters)

    @property
    def products(self) -> int:
        """T = number of quarter products issued: pairs (p, q), p, q < quarters, p + q < orders (eq. 4;
        quarters (quarters + 1) / 2 for the paper's set orders = quarters)."""
        Q, S = self.quarters, self.orders
        return sum(min(s + 1, Q, 2 * Q - 1 - s) for s in range(S))

    @property
    def fp64_flops(self) -> int:
        """FP64 flops of all quarter GEMMs issued: T * 2mnk."""
        return self.products * self.md_flops

    @property
    def md_flops(self) -> int:
        """2mnk multiple-double flops (BASELINE.json `metric`)."""
        return 2 * self.m * self.n * self.k

    def with_slices(self, bits: int, quarters: int, orders: int = 0) -> "Config":
        return dataclasses.replace(self, bits=bits, quarters=quarters, orders=orders or quarters)

    def with_shape(self, m=None, n=None, k=None) -> "Config":
        return dataclasses.replace(self, m=m or self.m, n=n or self.n, k=k or self.k)


CONFIGS = (
    Config(0, "dd_64", 64, 64, 64, 2, 0, "uniform"),
    Config(1, "dd_1024_exp8", 1024, 1024, 1024, 2, 1, "uniform_exp8"),
    Config(2, "dd_4096_normal", 4096, 4096, 4096, 2, 2, "normal"),
    Config(3, "dd_8192x8192x2048_wide30", 8192, 8192, 2048, 2, 3, "wide30", quarters=9),
    Config(4, "qd_2048", 2048, 2048, 2048, 4, 4, "uniform"),
    # Beyond BASELINE.json: the two wider formats of the paper's Table 2 (PAPER.md:196-205,
    # octo double = 8 limbs / 32 quarters, hexa double = 16 limbs / 64 quarters), same recipe as configs[4].
    Config(5, "od_1024", 1024, 1024, 1024, 8, 5, "uniform"),
    Config(6, "hd_512", 512, 512, 512, 16, 6, "uniform"),
)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    """The splitmix64 finaliser applied to uint64 counters (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        x = x + _U64(0x9E3779B97F4A7C15)
        x = (x ^ (x >> _U64(30))) * _U64(0xBF58476D1CE4E5B9)
        x = (x ^ (x >> _U64(27))) * _U64(0x94D049BB133111EB)
        return x ^ (x >> _U64(31))


def _bits(seed: int, mat: int, stream: int, rows: np.ndarray, cols: np.ndarray, ncols_total: int) -> np.ndarray:
    """64 random bits per (row, col) of matrix `mat` (0 = A, 1 = B), independent per `stream`."""
    key = (seed * 0x100000001B3 + mat * 0x51ED27 + stream * 0x2545F4914F6CDD1D + 0x1234567) & _MASK
    key = int(_splitmix64(np.array([key], dtype=_U64))[0])
    with np.errstate(over="ignore"):
        idx = rows.astype(_U64)[:, None] * _U64(ncols_total) + cols.astype(_U64)[None, :]
        return _splitmix64(_splitmix64(idx ^ _U64(key)) + _U64(key))


def _u01(bits: np.ndarray) -> np.ndarray:
    """Uniform in [0, 1) with 53 random bits."""
    return (bits >> _U64(11)).astype(np.float64) * 2.0 ** -53


def _sym(bits: np.ndarray) -> np.ndarray:
    """Uniform in [-1, 1)."""
    return 2.0 * _u01(bits) - 1.0


def generate(cfg: Config, which: str, row0: int = 0, row1: int | None = None,
             col0: int = 0, col1: int | None = None) -> np.ndarray:
    """Limb planes ``[limbs, row1-row0, col1-col0]`` of operand `which` ("A": m x k, "B": k x n).

    Recipes (BASELINE.json configs[0..4]):
      uniform       limb0 ~ U[-1,1)
      uniform_exp8  limb0 ~ U[-1,1) * 2^e, e uniform integer in [-8, 8] per element
      normal        limb0 ~ N(0,1) (Box-Muller on two uniform streams)
      wide30        limb0 = U[1,2) * (+-1) * 2^e, e uniform integer in [-30, 30] per element
      lower limbs   limb_i = limb_{i-1} * 2^-53 * U[-1,1)   (i = 1 .. limbs-1)
    """
    mat = {"A": 0, "B": 1}[which]
    nrows, ncols = (cfg.m, cfg.k) if mat == 0 else (cfg.k, cfg.n)
    row1 = nrows if row1 is None else row1
    col1 = ncols if col1 is None else col1
    rows = np.arange(row0, row1, dtype=np.int64)
    cols = np.arange(col0, col1, dtype=np.int64)

    def bits(stream):
        return _bits(cfg.seed, mat, stream, rows, cols, ncols)

    if cfg.dist == "uniform":
        lead = _sym(bits(0))
    elif cfg.dist == "uniform_exp8":
        e = (bits(1) % _U64(17)).astype(np.int64) - 8
        lead = np.ldexp(_sym(bits(0)), e.astype(np.int32))
    elif cfg.dist == "normal":
        u1 = 1.0 - _u01(bits(0))  # (0, 1]
        u2 = _u01(bits(1))
        lead = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
    elif cfg.dist == "wide30":
        b1 = bits(1)
        e = (b1 % _U64(61)).astype(np.int64) - 30
        sign = np.where((b1 >> _U64(63)) == _U64(1), -1.0, 1.0)
        lead = np.ldexp((1.0 + _u01(bits(0))) * sign, e.astype(np.int32))
    else:
        raise ValueError(cfg.dist)

    out = np.empty((cfg.limbs, rows.size, cols.size), dtype=np.float64)
    out[0] = lead
    for l in range(1, cfg.limbs):
        out[l] = out[l - 1] * 2.0 ** -53 * _sym(bits(8 + l))
    return out


def sample_indices(cfg: Config, count: int, salt: int = 0):
    """`count` seeded (i, j) output positions, uniform over the m x n result."""
    h = _splitmix64(np.arange(count, dtype=_U64) + _U64((cfg.seed * 7919 + salt * 104729 + 17) & _MASK))
    i = (h % _U64(cfg.m)).astype(np.int64)
    j = ((h >> _U64(32)) % _U64(cfg.n)).astype(np.int64)
    return i, j

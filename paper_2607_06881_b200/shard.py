"""Host-side sharding logic for N GPUs (one process per GPU).

The path shards by ROWS OF A with no data-path collective: the exponent E_i of row i of A depends on that row only, the
column exponents F_j on B only (replicated), and output rows are independent (SURVEY.md section
8(e)).  So rank r computes C[row0:row1, :] = A[row0:row1, :] * B with the single-GPU path, bit-identical to the rows the
unsharded call would produce.  Only timing is reduced across ranks (max), never data.
"""
from __future__ import annotations


def row_block(m_total: int, world: int, rank: int) -> tuple[int, int]:
    """Rows [row0, row1) of A (and C) owned by `rank`: contiguous blocks, sizes differ by at most one."""
    if world < 1 or not (0 <= rank < world) or m_total < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(m_total, world)
    row0 = rank * base + min(rank, extra)
    return row0, row0 + base + (1 if rank < extra else 0)


def aggregate_throughput(md_flops_per_rank: list[int], seconds_per_rank: list[float]) -> float:
    """Whole-job flop/s: all ranks' flops over the slowest rank's time (bench.py's max-over-ranks rule)."""
    return sum(md_flops_per_rank) / max(seconds_per_rank)

"""CPU tests of the host-side logic: sharding over ranks (world_size-2 gloo processes), workload bookkeeping, paper
constants.  The sharded result is computed with the ORACLE here (tests may use it); the product path shards the same way
with the CUDA kernels (bench.py --gpus N)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_06881_b200 import inputs, shard
from tests.golden import load_paper_constants


def test_row_blocks_partition_the_rows():
    for m in (1, 7, 64, 4096, 4097):
        for world in (1, 2, 3, 8):
            blocks = [shard.row_block(m, world, r) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == m
            assert all(a[1] == b[0] for a, b in zip(blocks, blocks[1:]))
            sizes = [b - a for a, b in blocks]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.row_block(4, 2, 2)
    assert shard.aggregate_throughput([10, 10], [1.0, 2.0]) == 10.0


def test_config_bookkeeping_matches_the_paper():
    paper = load_paper_constants()
    dd, qd = inputs.CONFIGS[2], inputs.CONFIGS[4]
    assert dd.quarters == paper["quarters_double_double"][0] == paper["quarters_per_double"][0] * dd.limbs
    assert qd.quarters == paper["data_growth_qd"][0]
    assert dd.products == 36 and qd.products == 136  # triangular set: S(S+1)/2 (eq. 4 without the zero blocks)
    assert dd.md_flops == 2 * 4096 ** 3 and dd.fp64_flops == 36 * dd.md_flops
    # Table 2: each doubling of the precision halves the md matrix dimensions of the 8192 x 4096 DGEMM
    rows, cols = paper["table2_rows_A"], paper["table2_cols_A"]
    for i, limbs in enumerate((2, 4, 8, 16)):
        assert rows[i + 1] * 4 * limbs == rows[0] and cols[i + 1] * 4 * limbs == cols[0]


def test_generated_inputs_follow_the_recipes():
    for cfg in inputs.CONFIGS:
        small = cfg.with_shape(40, 30, 50)
        A = inputs.generate(small, "A")
        assert A.shape == (cfg.limbs, 40, 50) and np.isfinite(A).all()
        for l in range(1, cfg.limbs):  # limb_l = limb_{l-1} * 2^-53 * U[-1,1)
            assert (np.abs(A[l]) <= np.abs(A[l - 1]) * 2.0 ** -53).all()
        assert (inputs.generate(small, "A", 5, 9, 3, 11) == A[:, 5:9, 3:11]).all()  # sub-blocks regenerate identically
    wide = inputs.generate(inputs.CONFIGS[3].with_shape(64, 64, 64), "A")[0]
    e = np.frexp(np.abs(wide))[1] - 1
    assert e.min() >= -30 and e.max() <= 30 and e.min() < -25 and e.max() > 25
    e8 = inputs.generate(inputs.CONFIGS[1].with_shape(64, 64, 64), "B")[0]
    assert np.abs(e8).max() <= 256.0


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import md_oracle as orc
    cfg = inputs.CONFIGS[3].with_shape(37, 29, 64)  # ragged row count: blocks of 19 and 18 rows
    row0, row1 = shard.row_block(cfg.m, world, rank)
    A_rows = inputs.generate(cfg, "A", row0, row1)  # each rank generates only its own rows
    B = inputs.generate(cfg, "B")
    C_rows = orc.md_gemm_rows(A_rows, B, quarters=cfg.quarters)
    # timing reduction as in bench.py: max over ranks
    t = torch.tensor([1.0 + rank], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    gathered = [None] * world
    dist.all_gather_object(gathered, (row0, row1, C_rows))
    if rank == 0:
        C = np.concatenate([g[2] for g in sorted(gathered, key=lambda g: g[0])], axis=1)
        np.save(os.path.join(out_dir, "C.npy"), C)
        np.save(os.path.join(out_dir, "t.npy"), t.numpy())
    dist.destroy_process_group()


def test_row_sharding_over_two_gloo_ranks_is_bit_identical(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    from oracle import md_oracle as orc
    cfg = inputs.CONFIGS[3].with_shape(37, 29, 64)
    A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    want = orc.md_gemm_rows(A, B, quarters=cfg.quarters)
    got = np.load(os.path.join(str(tmp_path), "C.npy"))
    assert got.shape == want.shape and (got == want).all()
    assert np.load(os.path.join(str(tmp_path), "t.npy"))[0] == 2.0

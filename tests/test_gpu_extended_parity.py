"""Extended full-size parity: collected by pytest with a reduced sample count (`-m gpu`), and runnable by hand on a B200 for
the tables in profiles/:

    python tests/test_gpu_extended_parity.py [--samples 20000] [--risky 1024] [--configs 1,2,3,4,5,6] [--quarters 3:8] > profiles/<name>.md

For every BASELINE.json config at its full size and every slice plan (the paper's quarters, md_plan_slices,
md_plan_slices_chunked) it runs md_gemm through the C-ABI and evaluates |C - C_exact| / (tol * (|A||B|)_ij) with the
oracle's exact product (O1) on many more positions than tests/test_gpu_fullsize.py: `--samples` uniformly random ones
and the `--risky` positions with the smallest (|A_0||B_0|)_ij / 2^(E_i+F_j) (chosen from an fp64 estimate).  It also
checks the order matrices bit-exactly at 2048 of the positions where the plan provides them.  Prints a markdown table."""
import argparse
import os
import sys
import time

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from oracle import md_oracle as orc  # noqa: E402
from paper_2607_06881_b200 import binding as md  # noqa: E402
from paper_2607_06881_b200 import inputs  # noqa: E402

TOL = {2: 1e-28, 4: 1e-58, 8: 1e-120, 16: 1e-245}


def main(argv=None, out=None):
    """Returns the list of (config index, plan name, Q, max uniform ratio, max riskiest ratio, orders bit-exact) rows."""
    import dataclasses
    import functools
    import builtins
    emit = functools.partial(builtins.print, file=out) if out is not None else builtins.print
    ap = argparse.ArgumentParser()
    ap.add_argument("--samples", type=int, default=20000)
    ap.add_argument("--risky", type=int, default=1024)
    ap.add_argument("--configs", default="1,2,3,4,5,6")
    ap.add_argument("--quarters", default="", help="cfg:Q[,cfg:Q] -- run a config with another quarter count (e.g. 3:8 = cfg3 "
                                                   "with the paper's 8 quarters instead of the 9 it is configured with, DESIGN.md R5)")
    ap.add_argument("--paper-only", action="store_true", help="only the plan with the config's 13-bit quarters")
    args = ap.parse_args(argv)
    q_override = {int(a.split(":")[0]): int(a.split(":")[1]) for a in args.quarters.split(",") if a}
    rows = []
    emit("# Extended full-size parity: md_gemm against the exact product at many sampled positions\n")
    emit(f"Command: `python tests/test_gpu_extended_parity.py --samples {args.samples} --risky {args.risky} --configs {args.configs}{' --quarters ' + args.quarters if args.quarters else ''}{' --paper-only' if args.paper_only else ''}` "
          "(one B200).  err = |C - C_exact|_ij evaluated in the oracle's long accumulator, W = (|A||B|)_ij; a ratio <= 1 "
          "meets the north_star tolerance (1e-28 dd, 1e-58 qd; DESIGN.md R13 for od / hd).\n")
    emit("| cfg | workload | plan | Q x W (chunk) | positions | max err/(tol W), uniform | max err/(tol W), riskiest | "
          "median | order matrices bit-exact (positions) | planned Q for this data (D) | seconds (oracle) |")
    emit("|---|---|---|---|---|---|---|---|---|---|---|")
    for ci in [int(x) for x in args.configs.split(",")]:
        cfg = inputs.CONFIGS[ci]
        if ci in q_override:
            cfg = dataclasses.replace(cfg, quarters=q_override[ci])
        L = cfg.limbs
        A, B = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
        dA, dB = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
        si, sj = inputs.sample_indices(cfg, args.samples, salt=99)
        Wt = dA[0].abs() @ dB[0].abs()
        rel = Wt / (dA[0].abs().amax(dim=1)[:, None] * dB[0].abs().amax(dim=0)[None, :])
        flat = torch.topk(rel.flatten(), min(args.risky, rel.numel()), largest=False).indices.cpu().numpy()
        del Wt, rel
        si = np.concatenate([si, flat // cfg.n]).astype(np.int64)
        sj = np.concatenate([sj, flat % cfg.n]).astype(np.int64)
        pq, pd = md.md_plan_quarters(dA, dB)
        plans = [("paper's quarters", cfg.bits, cfg.quarters, 0), ("md_plan_slices",) + md.md_plan_slices(cfg.k, L) + (0,)]
        cw, cq, ck = md.md_plan_slices_chunked(cfg.k, L, 128)
        if (cw, cq) != plans[1][1:3]:
            plans.append(("md_plan_slices_chunked", cw, cq, ck))
        if args.paper_only:
            plans = plans[:1]
        for name, W, Q, chunk in plans:
            with md.Workspace(cfg.m, cfg.n, cfg.k, L, Q, bits=W):
                C = md.md_gemm(dA, dB)
                assert md.md_read_flags() == 0
                Ch = C.cpu().numpy()
                del C
                exact_orders = "n/a (beyond the whole-k budget)"
                if chunk == 0:
                    orders = md.md_gemm_orders(dA, dB)
                    oi, oj = torch.from_numpy(si[:2048]).cuda(), torch.from_numpy(sj[:2048]).cuda()
                    got = orders[:, oi, oj].cpu().numpy().T
                    del orders
                    Aq, eA, _ = orc.split(A, 0, Q, bits=W)
                    Bq, eB, _ = orc.split(B, 1, Q, bits=W)
                    want = orc.orders_int_samples(Aq, eA, Bq, eB, si[:2048], sj[:2048], bits=W)
                    del Aq, Bq
                    exact_orders = f"{bool((got == want).all())} (2048)"
            t0 = time.perf_counter()
            r = orc.exact_samples(A, B, si, sj, Ch)
            dt = time.perf_counter() - t0
            ratio = r["err"] / (TOL[L] * r["W"])
            nu = args.samples
            emit(f"| {ci} | {cfg.name} | {name} | {Q} x {W}{' (%d)' % chunk if chunk else ''} | {si.size} | {ratio[:nu].max():.3g} | "
                  f"{ratio[nu:].max():.3g} | {np.median(ratio):.3g} | {exact_orders} | {pq} ({pd}) | {dt:.0f} |", flush=True)
            rows.append((ci, name, Q, float(ratio[:nu].max()), float(ratio[nu:].max()), exact_orders))
        del dA, dB
        torch.cuda.empty_cache()
    return rows


@pytest.mark.gpu
@pytest.mark.parametrize("ci", [1, 3])
def test_extended_parity_reduced(ci):
    """The extended run with a reduced sample count, so that the driver's `-m gpu` pass covers it: every plan of the config
    meets the north_star tolerance on 1 500 uniform + 256 riskiest positions and the order matrices are bit-exact."""
    import io
    rows = main(["--samples", "1500", "--risky", "256", "--configs", str(ci)], out=io.StringIO())
    assert rows
    for _, name, _, uni, risky, exact_orders in rows:
        assert uni <= 1.0 and risky <= 1.0, (name, uni, risky)
        assert exact_orders.startswith(("True", "n/a")), (name, exact_orders)


if __name__ == "__main__":
    main()

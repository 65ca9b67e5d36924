#!/usr/bin/env python
"""bench.py -- throughput of the multiple-double GEMM hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path (md_gemm: exponent vectors + split of A and B + fused quarter GEMM with the
renormalising epilogue) over one seeded synthetic problem.  The workload at N = 1 is
BASELINE.json configs[2], the config its metric is quoted on: double-double 4096^3, hi ~ N(0,1), lo = hi*2^-53*U[-1,1].
With N > 1 the rows of A are sharded (rank r owns rows [r*4096, (r+1)*4096) of an (N*4096) x 4096 A, B replicated): no
data-path collective is needed because a row's exponent depends on that row only -> weak scaling.

Rank 0 prints ONE JSON line.  value = whole-job double-double GFLOP/s (2mnk per problem) with inputs resident in HBM;
e2e = the same through md_gemm_host with pinned HOST buffers (H2D of A, B and D2H of C inside the timed region);
roofline = the fused quarter-GEMM kernel's issued FP64 flops (T*2mnk, T = 36) / its CUDA-event duration against the FP64
tensor (DMMA) peak; cpu_baseline = the CPU oracle (oracle/, as it stands) on a bounded sample, same run, rank 0, N = 1.
--impl reference times that oracle alone (there is no reference implementation to install: /root/reference holds only
the paper's text).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "effective double-double GFLOP/s at n=4096 on 1 B200; % of FP64 tensor peak"
UNIT = "GFLOP/s (double-double, 2mnk)"
# FP64 tensor (DMMA) peak of B200: 128 flop/clk/SM x 148 SMs x 1.965 GHz (clocks.max.sm) = 37.22 TFLOP/s.
# MEASURED_PEAKS.json holds no FP64 figure, so the denominator is this unit-count x clock figure;
# it is cross-checked LIVE in every run by md_probe_dmma, a register-only mma.sync.m8n8k4.f64 loop (measure_dmma_peak
# below; profiles/r01_dmma_peak.md), and the probe's number is reported beside it.
FP64_TENSOR_PEAK_TFLOPS = 128 * 148 * 1.965e9 / 1e12
# The paper's own figure for this metric and workload (double double, n = 4096, whole pipeline t_TC = 7.93621 s ->
# 2*4096^3 / t = 17.3 GFLOP/s; Table 1; hardware A100 or RTX 4080, the paper does not say): context only.
PAPER_DD_4096_GFLOPS = 2 * 4096 ** 3 / 7.93621 / 1e9
CPU_SAMPLE_ROWS = 16            # cpu_baseline leg of the default run: 16 rows x all columns (~10 s on 16 cores)
REF_ROWS, REF_COLS = 16, 1024   # --impl reference: per step (~2.5 s on 16 cores)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (default 2: the headline)")
    ap.add_argument("--slices", default="paper", choices=["paper", "adaptive", "chunked"],
                    help="paper: 13-bit quarters, 4 per limb (the headline).  adaptive: the (bits, count) md_plan_slices "
                         "picks for this k -- wider, fewer slices (DESIGN.md R14; NOT the paper's quarters).  chunked: "
                         "md_plan_slices_chunked(k, limbs, 128) -- still wider slices, exact per chunk of k (DESIGN.md R16)")
    ap.add_argument("--paper-paths", action="store_true",
                    help="also time the paper's own two paths on this GPU (libmdcompare: materialised top-down product "
                         "through cuBLAS DGEMM, CUDA-core classical GEMM; SURVEY.md 8(f) NEXT-2), outside the timed region")
    ap.add_argument("--shape", default=None, help="m,n,k override of the config's shape (same recipe and seed): for the "
                                                  "small / medium size tables in profiles/")
    ap.add_argument("--quarters", type=int, default=0, help="override the config's quarter count (MD_OPT_QUARTERS)")
    ap.add_argument("--orders", type=int, default=0, help="kept product orders S (MD_OPT_ORDERS); default = quarters")
    ap.add_argument("--raster-group", type=int, default=0, help="MD_OPT_RASTER_GROUP (tile rows per raster group; 0 = default)")
    ap.add_argument("--host-blocks", type=int, default=0, help="MD_OPT_HOST_BLOCKS for the e2e leg (0 = automatic; n = blocks of C; PR * 256 + PC = explicit panels)")
    ap.add_argument("--tile", type=int, default=0, choices=(0, 1, 2),
                    help="MD_OPT_TILE (double double): 0 = automatic, 1 = the 32 x 16 CTA tile wherever it exists, 2 = never")
    ap.add_argument("--tile-schedule", type=int, default=0, choices=(0, 1, 2, 3),
                    help="MD_OPT_TILE_SCHEDULE: 0 = automatic (hybrid from many whole-tile waves on), 1 = hybrid wherever possible, 2 = tile queue only, 3 = static lists")
    ap.add_argument("--one-launch", type=int, default=0, choices=[0, 1, 2],
                    help="MD_OPT_ONE_LAUNCH: 0 = automatic (single-wave problems run a1-a4 in one kernel), 1 = wherever it exists, 2 = never")
    ap.add_argument("--micro", action="store_true",
                    help="instead of the md_gemm step: time the public per-step entry points on this config's shapes -- "
                         "md_split (axis 0 on A, axis 1 on B) and md_renorm -- and print their achieved HBM GB/s against "
                         "MEASURED_PEAKS.json (north_star: 'achieved HBM GB/s for the split and epilogue')")
    ap.add_argument("--balance-table", action="store_true",
                    help="instead of the md_gemm step: the same problem through (a) the row / column grid with the paper's quarter "
                         "count, (b) that with one more ORDER, (c) with one more QUARTER, (d) the paper's own per-element balancing "
                         "with exponent classes (md_gemm_literal) -- time and sampled err / (tol (|A||B|)_ij) of each (DESIGN.md "
                         "R5, R17-R22; the table VERDICT r1 asks for)")
    ap.add_argument("--samples", type=int, default=20000, help="--balance-table: uniformly sampled positions (+ 1024 riskiest)")
    ap.add_argument("--sign-groups", action="store_true", help="--balance-table: also the literal mode with the sign groups of eq. (6)")
    ap.add_argument("--qr", action="store_true",
                    help="instead of the md_gemm step: md_qr (blocked Householder QR on top of md_gemm, PAPER.md:213) of the m x n "
                         "matrix A of this config (--shape m,n,k; k unused): time, share of it inside the md_gemm path, md-GFLOP/s "
                         "counting 2 m n^2 - 2 n^3 / 3 for R plus the same again for Q")
    ap.add_argument("--lean", action="store_true", help="skip the context blocks beside the headline (quarter plan, adaptive slices)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks / throttle reasons of one GPU every 200 ms while running."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        super().__init__(daemon=True)
        self.gpu_index = gpu_index
        self.samples = []
        self.proc = None

    def run(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu_index), f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                parts = [p.strip() for p in line.split(",")]
                if len(parts) == 7:
                    self.samples.append(parts)
        except Exception:
            pass

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()

    def summary(self, t0: float = 0.0):
        sm, reasons, mx, power = [], set(), None, []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in self.samples:
            try:
                sm.append(float(s[0]))
                mx = float(s[1])
                power.append(float(s[2]))
            except ValueError:
                continue
            for name, val in zip(names, s[3:]):
                if val == "Active":
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        busy = [c for c, p in zip(sm, power) if p > 0.5 * max(power)] or sm  # samples under load
        return {"sm_mhz": statistics.median(busy), "sm_max_mhz": mx, "reasons": sorted(reasons),
                "power_w_max": max(power), "samples": len(sm)}


def measure_dmma_peak(md, torch, warps_per_block: int = 8, reps: int = 5):
    """FP64 tensor peak measured now, on this GPU: md_probe_dmma (one CTA per SM, register-only DMMA) timed with CUDA
    events on the launching stream; best of `reps` after one warm-up.  Returns TFLOP/s."""
    sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    stream = torch.cuda.current_stream()
    iters = 100_000
    md.md_probe_dmma(sms, warps_per_block, 1000)
    best = 0.0
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        flops = md.md_probe_dmma(sms, warps_per_block, iters)
        e1.record(stream)
        e1.synchronize()
        best = max(best, flops / (e0.elapsed_time(e1) * 1e-3) / 1e12)
    return best


def cpu_oracle_sample(cfg, rows: int, cols: int | None = None):
    """The oracle's five-step pipeline on the first `rows` rows of A and the first `cols` columns of B (default: all):
    a rows x cols block of C, exactly as the full problem would compute it (a row's / column's exponent depends on
    that row / column only).  Returns (GFLOP/s, seconds, threads)."""
    from oracle import md_oracle as orc
    from paper_2607_06881_b200 import inputs
    cols = cfg.n if cols is None else min(cols, cfg.n)
    rows = min(rows, cfg.m)
    A = inputs.generate(cfg, "A", 0, rows)
    B = np.ascontiguousarray(inputs.generate(cfg, "B", 0, None, 0, cols))
    threads = min(orc.num_threads(), rows)
    t0 = time.perf_counter()
    orc.md_gemm_rows(A, B, quarters=cfg.quarters, bits=cfg.bits)
    dt = time.perf_counter() - t0
    return 2.0 * rows * cols * cfg.k / dt / 1e9, dt, threads


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2607_06881_b200 import inputs
    cfg = inputs.CONFIGS[args.config]
    # one step = a bounded sample: a REF_ROWS x REF_COLS block of C over the full k (a few seconds of CPU work per
    # step, one row per OpenMP thread), so that W + K steps end within minutes
    rows, cols = min(REF_ROWS, cfg.m), min(REF_COLS, cfg.n)
    for _ in range(args.warmup):
        cpu_oracle_sample(cfg, rows, cols)
    steps = args.steps
    secs, threads = [], 1
    for _ in range(steps):
        _, dt, threads = cpu_oracle_sample(cfg, rows, cols)
        secs.append(dt)
    value = 2.0 * rows * cols * cfg.k * steps / sum(secs) / 1e9
    sample = (f"per step: first {rows} rows of A x first {cols} columns of B over the full k ({rows}x{cols} outputs of "
              f"the {cfg.m}x{cfg.n}x{cfg.k} problem); oracle split + {cfg.products} plain fp64 quarter GEMM loops + exact "
              f"renorm, OpenMP over rows; {steps} steps timed")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": value / PAPER_DD_4096_GFLOPS if args.config == 2 else None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{cfg.index}] {cfg.name}: {cfg.m}x{cfg.n}x{cfg.k}, limbs={cfg.limbs}, "
                               f"quarters={cfg.quarters}, seed {cfg.seed}", "kind": "CPU oracle (no GPU work)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def hbm_peak_gbs():
    """Measured HBM copy bandwidth of this pool's B200s (driver-written MEASURED_PEAKS.json), else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:  # noqa: BLE001
        return 6550.0, "fallback of /opt/skills/guides/B200_PROFILING.md (MEASURED_PEAKS.json absent)"


def apply_overrides(args, base):
    import dataclasses
    if args.shape:
        m, n, k = (int(x) for x in args.shape.split(","))
        base = base.with_shape(m, n, k)
    if args.quarters or args.orders:
        q = args.quarters or base.quarters
        base = dataclasses.replace(base, quarters=q, orders=args.orders or q)
    return base


def run_micro(args):
    """--micro: the public per-step entry points (md_split, md_renorm) on this config's shapes, HBM roofline."""
    import torch
    from paper_2607_06881_b200 import binding as md
    from paper_2607_06881_b200 import inputs
    torch.cuda.set_device(0)
    cfg = apply_overrides(args, inputs.CONFIGS[args.config])
    L, Q = cfg.limbs, cfg.quarters
    A = torch.from_numpy(inputs.generate(cfg, "A")).cuda()
    B = torch.from_numpy(inputs.generate(cfg, "B")).cuda()
    peak, src = hbm_peak_gbs()
    stream = torch.cuda.current_stream()

    def timed(fn):
        for _ in range(max(args.warmup, 3)):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps

    out = {"impl": "ours", "mode": "micro", "hbm_peak_gbs": peak, "hbm_peak_source": src, "steps": args.steps,
           "config": {"workload": f"BASELINE.json configs[{cfg.index}] {cfg.name}: m={cfg.m} n={cfg.n} k={cfg.k}, limbs={L}, quarters={Q}"},
           "kernels": {}}
    for name, X, axis in (("md_split_axis0_A", A, 0), ("md_split_axis1_B", B, 1)):
        qp = torch.empty((Q,) + tuple(X.shape[1:]), dtype=torch.float64, device="cuda")
        ex = torch.empty(X.shape[1] if axis == 0 else X.shape[2], dtype=torch.int32, device="cuda")
        rows, cols = X.shape[1], X.shape[2]

        def call():
            st = md.lib().md_split(rows, cols, L, Q, axis, X.data_ptr(), qp.data_ptr(), ex.data_ptr(), stream.cuda_stream)
            assert st == 0
        ms = timed(call)
        # exponent pass reads the leading plane (8 B / element); the split reads 8 L and writes 8 Q bytes per element
        nbytes = X[0].numel() * 8 * (1 + L + Q)
        out["kernels"][name] = {"ms": ms, "algorithmic_bytes": nbytes, "gbs": nbytes / ms / 1e6, "frac_of_hbm_peak": nbytes / ms / 1e6 / peak,
                                "launches": "exponent kernel(s) + split_kernel"}
        del qp
    S = args.orders or Q
    orders = torch.randn((S, cfg.m, cfg.n), dtype=torch.float64, device="cuda") * torch.exp2(-13.0 * torch.arange(S, device="cuda", dtype=torch.float64))[:, None, None]
    C = torch.empty((L, cfg.m, cfg.n), dtype=torch.float64, device="cuda")

    def call_r():
        st = md.lib().md_renorm(cfg.m, cfg.n, L, S, orders.data_ptr(), C.data_ptr(), stream.cuda_stream)
        assert st == 0
    ms = timed(call_r)
    nbytes = cfg.m * cfg.n * 8 * (S + L)
    out["kernels"]["md_renorm"] = {"ms": ms, "algorithmic_bytes": nbytes, "gbs": nbytes / ms / 1e6, "frac_of_hbm_peak": nbytes / ms / 1e6 / peak,
                                   "note": "synthetic order planes of the right magnitudes (timing only)"}
    print(json.dumps(out))


def run_balance_table(args):
    """--balance-table: row / column grid at Q, (Q, Q+1), Q+1 against the paper's literal exponent classes on one workload."""
    import dataclasses
    import torch
    from oracle import md_oracle as orc
    from paper_2607_06881_b200 import binding as md
    from paper_2607_06881_b200 import inputs
    torch.cuda.set_device(0)
    cfg = apply_overrides(args, inputs.CONFIGS[args.config])
    L = cfg.limbs
    Q0 = 4 * L
    tol = {2: 1e-28, 4: 1e-58, 8: 1e-120, 16: 1e-245}[L]
    A_h, B_h = inputs.generate(cfg, "A"), inputs.generate(cfg, "B")
    A, B = torch.from_numpy(A_h).cuda(), torch.from_numpy(B_h).cuda()
    stream = torch.cuda.current_stream()
    si, sj = inputs.sample_indices(cfg, args.samples, salt=7)
    Wt = A[0].abs() @ B[0].abs()
    rel = Wt / (A[0].abs().amax(dim=1)[:, None] * B[0].abs().amax(dim=0)[None, :])
    flat = torch.topk(rel.flatten(), min(1024, rel.numel()), largest=False).indices.cpu().numpy()
    del Wt, rel
    si = np.concatenate([si, flat // cfg.n]).astype(np.int64)
    sj = np.concatenate([sj, flat % cfg.n]).astype(np.int64)

    def timed(fn, steps, warmup):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            out = fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / steps, out

    def accuracy(C):
        r = orc.exact_samples(A_h, B_h, si, sj, C.cpu().numpy())
        ratio = r["err"] / (tol * r["W"])
        return {"max_err_over_tol_W": float(ratio.max()), "median": float(np.median(ratio)), "positions": int(si.size),
                "misses": int((ratio > 1.0).sum())}

    rows = []
    for name, Q, S in (("row/column grid, paper's quarters", Q0, Q0), ("row/column grid, one more ORDER", Q0, Q0 + 1),
                       ("row/column grid, one more QUARTER", Q0 + 1, Q0 + 1)):
        c = dataclasses.replace(cfg, quarters=Q, orders=S)
        with md.Workspace(cfg.m, cfg.n, cfg.k, L, Q, orders=0 if S == Q else S):
            ms, C = timed(lambda: md.md_gemm(A, B), args.steps, args.warmup)
        rows.append({"mode": name, "quarters": Q, "orders": S, "quarter_products": c.products, "ms": ms,
                     "md_gflops": cfg.md_flops / ms / 1e6, **accuracy(C)})
        del C
    variants = [("paper-literal: per-element exponents, eq. 7 + eq. 8, exponent classes A_0..A_12", 0)]
    if args.sign_groups:
        variants.append(("paper-literal with the sign groups of eq. 6", md.MD_LITERAL_SIGN_GROUPS))
    for name, flags in variants:
        box = {}

        def call():
            C, info = md.md_gemm_literal(A, B, flags=flags, scratch=box.get("scratch"))
            box["info"] = info
            return C
        l0 = md.md_launch_count()
        ms, C = timed(call, 1, 0)   # one timed call: it is hundreds of quarter GEMMs
        info = box["info"]
        T = sum(1 for p in range(info["planes"]) for q in range(info["planes"]) if p + q < info["orders"])
        rows.append({"mode": name, "quarters": Q0, "planes_per_class": info["planes"], "orders": info["orders"],
                     "class_pairs": info["pairs"], "quarter_products": info["pairs"] * T, "launches": md.md_launch_count() - l0, "ms": ms,
                     "md_gflops": cfg.md_flops / ms / 1e6, "levels": [info["zminA"], info["zmaxA"], info["zminB"], info["zmaxB"]],
                     **accuracy(C)})
        del C
    print(json.dumps({"impl": "ours", "mode": "balance-table",
                      "config": {"workload": f"BASELINE.json configs[{cfg.index}] {cfg.name}: m={cfg.m} n={cfg.n} k={cfg.k}, limbs={L}, seed {cfg.seed}"},
                      "tolerance": tol, "rows": rows}))


def run_qr(args):
    import torch
    from paper_2607_06881_b200 import binding as md
    from paper_2607_06881_b200 import inputs
    torch.cuda.set_device(0)
    cfg = apply_overrides(args, inputs.CONFIGS[args.config])
    m, n = cfg.m, cfg.n
    cfg = cfg.with_shape(m, 3, n)
    A = torch.from_numpy(inputs.generate(cfg, "A")).cuda()
    l0 = md.md_launch_count()
    rows = []
    for i in range(args.warmup + args.steps):
        Q, R, (total, in_gemm) = md.md_qr(A, want_times=True)
        if i >= args.warmup:
            rows.append((total, in_gemm))
    launches = (md.md_launch_count() - l0) // (args.warmup + args.steps)
    total = sum(r[0] for r in rows) / len(rows)
    in_gemm = sum(r[1] for r in rows) / len(rows)
    flops = 2 * (2.0 * m * n * n - 2.0 * n ** 3 / 3.0)
    print(json.dumps({"impl": "ours", "mode": "qr", "metric": "md_qr: multiple-double GFLOP/s (4 m n^2 - 4 n^3 / 3 for R and Q)",
                      "value": flops / total / 1e6, "unit": "GFLOP/s (multiple double)", "ms": total, "ms_in_md_gemm": in_gemm,
                      "share_in_md_gemm": in_gemm / total, "launches_per_call": launches, "steps": args.steps, "warmup": args.warmup,
                      "config": {"workload": f"{m} x {n} matrix A of BASELINE.json configs[{cfg.index}] ({cfg.name} recipe), limbs={cfg.limbs}, "
                                             f"quarters={cfg.quarters}, panel width 32"}}))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2607_06881_b200 import binding as md
    from paper_2607_06881_b200 import inputs
    from paper_2607_06881_b200 import shard

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; launch with torch.distributed.run")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    md.lib()  # fail loudly now if the extension is missing

    base = apply_overrides(args, inputs.CONFIGS[args.config])
    md.md_set_option(md.MD_OPT_RASTER_GROUP, args.raster_group)
    md.md_set_option(md.MD_OPT_ONE_LAUNCH, args.one_launch)
    md.md_set_option(md.MD_OPT_TILE_SCHEDULE, args.tile_schedule)
    md.md_set_option(md.MD_OPT_TILE, args.tile)
    md.md_set_option(md.MD_OPT_HOST_BLOCKS, args.host_blocks)
    # weak scaling: the global A has world * m rows, rank r owns one block of m rows (no collective on the data path)
    if args.slices == "adaptive":
        base = base.with_slices(*md.md_plan_slices(base.k, base.limbs))
    elif args.slices == "chunked":
        base = base.with_slices(*md.md_plan_slices_chunked(base.k, base.limbs, 128)[:2])
    cfg = base.with_shape(m=base.m * world)
    row0, row1 = shard.row_block(cfg.m, world, rank)
    m, n, k, L, Q, W, S = row1 - row0, cfg.n, cfg.k, cfg.limbs, cfg.quarters, cfg.bits, cfg.orders
    A_host = torch.from_numpy(inputs.generate(cfg, "A", row0, row1)).pin_memory()
    B_host = torch.from_numpy(inputs.generate(cfg, "B")).pin_memory()
    C_host = torch.empty((L, m, n), dtype=torch.float64).pin_memory()
    A, B = A_host.cuda(), B_host.cuda()
    C = torch.empty((L, m, n), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x: float) -> float:
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    sampler = ClockSampler(local_rank)
    with md.Workspace(m, n, k, L, Q, bits=W, orders=0 if S == Q else S):
        for _ in range(args.warmup):
            md.md_gemm(A, B, C)
        barrier()
        sampler.start()
        # CUDA events of the library around the preparation and around the fused kernel of every call (roofline timing).  Inside
        # the timed region, unless a step is so short (< 1 ms, seen in the warm-up) that the three event records per call would
        # distort it: then the timed loop runs bare and the kernel times come from a second loop of the same K steps.
        w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        w0.record(stream)
        md.md_gemm(A, B, C)
        w1.record(stream)
        torch.cuda.synchronize()
        profile_inside = w0.elapsed_time(w1) >= 1.0
        if profile_inside:
            md.md_profile_enable(args.steps)
        launches0 = md.md_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        for _ in range(args.steps):
            md.md_gemm(A, B, C)
        e1.record(stream)
        barrier()
        ms_total = max_over_ranks(e0.elapsed_time(e1))
        launches = md.md_launch_count() - launches0
        if not profile_inside:
            md.md_profile_enable(args.steps)
            for _ in range(args.steps):
                md.md_gemm(A, B, C)
            torch.cuda.synchronize()
        split_ms, gemm_ms = md.md_profile_read(args.steps)
        md.md_profile_enable(0)
        flags = md.md_read_flags()
    clocks_after_device_loop = len(sampler.samples)
    probe_launches0 = md.md_launch_count()
    dmma_probe_tflops = measure_dmma_peak(md, torch)
    probe_launches = md.md_launch_count() - probe_launches0

    # what the data needs (md_plan_quarters, R15): the any-input guarantee for this input, outside the timed region
    # (the blocks from here to the e2e leg are context beside the headline: a failure in one of them is recorded in its
    # place and never costs the JSON line)
    def context_block(fn):
        try:
            return fn()
        except Exception as exc:  # noqa: BLE001
            for key in (md.MD_OPT_SLICE_BITS, md.MD_OPT_QUARTERS):
                md.md_set_option(key, 0)
            md.md_set_workspace(None)
            return {"error": f"{type(exc).__name__}: {exc}"}

    def plan_block():
        md.md_set_option(md.MD_OPT_SLICE_BITS, 0 if W == 13 else W)
        md.md_plan_quarters(A, B)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        pq, pd = md.md_plan_quarters(A, B)
        plan_ms = (time.perf_counter() - t0) * 1e3
        md.md_set_option(md.MD_OPT_SLICE_BITS, 0)
        return {"spread_D": pd, "guaranteed_quarters": pq, "run_with": Q, "slice_bits": W, "ms": plan_ms,
                "note": "smallest Q with k (Q+3) 2^(D - W Q - 2) <= the format's tolerance at every position "
                        "(worst case; measured errors are 2-3 orders of magnitude below the bound)"}

    quarter_plan = context_block(plan_block) if world == 1 and not args.lean else None

    # beside the headline (the paper's quarters): the same problem with the k-adaptive slices, outside the timed region
    adaptive = None

    def time_variant(aW, aQ, note):
        C2 = torch.empty_like(C)
        with md.Workspace(m, n, k, L, aQ, bits=aW):
            md.md_gemm(A, B, C2)
            md.md_profile_enable(3)
            torch.cuda.synchronize()
            v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            v0.record(stream)
            for _ in range(3):
                md.md_gemm(A, B, C2)
            v1.record(stream)
            torch.cuda.synchronize()
            _, a_gemm_ms = md.md_profile_read(3)
            md.md_profile_enable(0)
        a_ms = v0.elapsed_time(v1) / 3
        aT = aQ * (aQ + 1) // 2
        return {"slice_bits": aW, "slices": aQ, "products": aT, "ms_per_step": a_ms,
                "value": base.md_flops / (a_ms * 1e-3) / 1e9, "unit": UNIT,
                "kernel_frac_of_fp64_tensor_peak": aT * base.md_flops / (sum(a_gemm_ms) / 3 * 1e-3) / 1e12 / FP64_TENSOR_PEAK_TFLOPS,
                "max_abs_diff_vs_paper_quarters": float((C2 - C).abs().sum(dim=0).max()), "note": note}

    def adaptive_block():
        cW, cQ, cK = md.md_plan_slices_chunked(k, L, 128)
        aW, aQ = md.md_plan_slices(k, L)
        if (aW, aQ) == (W, Q):
            return None
        out = time_variant(aW, aQ, "md_plan_slices: wider, fewer slices on the same kernels (DESIGN.md R14); not the "
                                   "paper's 13-bit quarters, so not the headline; 3 steps after 1 warm-up, CUDA events")
        if (cW, cQ) != (aW, aQ):
            out["chunked"] = time_variant(cW, cQ, "md_plan_slices_chunked(k, limbs, 128): exactness kept per chunk of %d "
                                                  "contraction indices (DESIGN.md R16)" % cK)
            out["chunked"]["chunk"] = cK
        return out

    if args.slices == "paper" and world == 1 and not args.lean:
        adaptive = context_block(adaptive_block)

    # the paper's own two paths on the same inputs (context; outside the timed region; N = 1, dd / qd only)
    paper_paths = None
    if args.paper_paths and world == 1 and L <= 4:
        from paper_2607_06881_b200 import compare as mdc
        PQ = 4 * L
        ws = torch.empty(mdc.mdc_topdown_workspace_bytes(m, n, k, L, PQ), dtype=torch.uint8, device="cuda")
        C_td, _, _ = mdc.mdc_topdown_gemm(A, B, ws=ws)  # warm-up (cuBLAS handle, heuristics)
        stage = [0.0] * 4
        torch.cuda.synchronize()
        t_e0, t_e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t_e0.record(stream)
        reps = 3
        for _ in range(reps):
            C_td, _, times = mdc.mdc_topdown_gemm(A, B, ws=ws, want_times=True)
            stage = [a + b / reps for a, b in zip(stage, times)]
        t_e1.record(stream)
        torch.cuda.synchronize()
        td_ms = t_e0.elapsed_time(t_e1) / reps
        del ws
        C_cl = mdc.mdc_classic_gemm(A, B)
        torch.cuda.synchronize()
        t_e0.record(stream)
        C_cl = mdc.mdc_classic_gemm(A, B)
        t_e1.record(stream)
        torch.cuda.synchronize()
        cl_ms = t_e0.elapsed_time(t_e1)
        same_as_fused = bool((C_td == C).all()) if (Q, W) == (PQ, 13) else None
        paper_paths = {
            "topdown_materialised_cublas_dgemm": {
                "ms_per_step": td_ms, "value": base.md_flops / (td_ms * 1e-3) / 1e9, "unit": UNIT,
                "stage_ms": {"split": stage[0], "construct_Atil": stage[1], "dgemm": stage[2], "recombine": stage[3]},
                "dgemm_fp64_tflops": 2.0 * (PQ * m) * n * (PQ * k) / (stage[2] * 1e-3) / 1e12,
                "block_products": PQ * PQ, "bit_identical_to_fused_md_gemm": same_as_fused,
                "what": "PAPER.md:73-89 eq. 4, :192-207 Table 2: Atil (A convoluted, %d x %d doubles) * Bstk (B stacked) "
                        "through ONE cublasDgemm, then md_renorm; the paper's t_TC" % (PQ * m, PQ * k)},
            "cuda_core_classical": {
                "ms_per_step": cl_ms, "value": base.md_flops / (cl_ms * 1e-3) / 1e9, "unit": UNIT,
                "max_abs_diff_vs_fused": float((C_cl - C).abs().sum(dim=0).max()),
                "what": "PAPER.md:166: one thread per inner product, TwoSum / TwoProd on the regular FP64 cores; the paper's t_CUDA"},
            "note": "comparison paths (libmdcompare), measured after the timed region: 3 / 1 steps after 1 warm-up, CUDA events",
        }
        del C_td, C_cl

    # end to end: pinned host buffers through md_gemm_host (H2D A, B + the whole path + D2H C, synchronous)
    e2e = None
    if not args.no_e2e:
        try:
            md.md_set_option(md.MD_OPT_QUARTERS, 0 if Q == 4 * L else Q)  # before sizing the scratch: it depends on Q
            md.md_set_option(md.MD_OPT_ORDERS, 0 if S == Q else S)
            md.md_set_option(md.MD_OPT_SLICE_BITS, 0 if W == 13 else W)
            scratch = torch.empty(md.md_host_scratch_bytes(m, n, k, L), dtype=torch.uint8, device="cuda")
            for _ in range(min(args.warmup, 2)):
                md.md_gemm_host(A_host, B_host, C_host, scratch)
            barrier()
            launches_e2e0 = md.md_launch_count()
            t0 = time.perf_counter()
            e0.record(stream)
            for _ in range(args.steps):
                md.md_gemm_host(A_host, B_host, C_host, scratch)
            e1.record(stream)
            barrier()
            e2e_ms = max_over_ranks(e0.elapsed_time(e1))
            wall_ms = max_over_ranks((time.perf_counter() - t0) * 1e3)
            md.md_set_option(md.MD_OPT_QUARTERS, 0)
            md.md_set_option(md.MD_OPT_ORDERS, 0)
            md.md_set_option(md.MD_OPT_SLICE_BITS, 0)
            e2e = {"value": world * base.md_flops * args.steps / (max(e2e_ms, wall_ms) * 1e-3) / 1e9, "unit": UNIT,
                   "h2d_bytes_per_step": A_host.numel() * 8 + B_host.numel() * 8, "d2h_bytes_per_step": C_host.numel() * 8,
                   "ms_per_step": max(e2e_ms, wall_ms) / args.steps, "launches": md.md_launch_count() - launches_e2e0,
                   "matches_device_path": bool((C_host == C.cpu()).all())}
            del scratch
        except Exception as exc:  # noqa: BLE001 -- the device-resident headline must still be reported
            for key in (md.MD_OPT_SLICE_BITS, md.MD_OPT_QUARTERS, md.MD_OPT_ORDERS):
                md.md_set_option(key, 0)
            e2e = {"error": f"{type(exc).__name__}: {exc}"}
    sampler.stop()
    clocks = sampler.summary()
    clocks["samples_in_device_loop"] = clocks_after_device_loop

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms_per_step = ms_total / args.steps
    value = world * base.md_flops / (ms_per_step * 1e-3) / 1e9
    gemm_avg_ms = sum(gemm_ms) / len(gemm_ms)
    issued_flops = base.fp64_flops  # T * 2mnk per launch (per rank)
    achieved = issued_flops / (gemm_avg_ms * 1e-3) / 1e12
    roofline = {
        "bound": "tensor", "kernel": "qgemm_kernel (fused triangular quarter GEMM + renormalising epilogue)",
        "achieved": achieved, "peak": FP64_TENSOR_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP64_TENSOR_PEAK_TFLOPS,
        "peak_source": "FP64 DMMA: 128 flop/clk/SM x 148 SMs x 1.965 GHz (MEASURED_PEAKS.json has no FP64 entry; "
                       "DESIGN.md section 6); cross-checked in this run by md_probe_dmma (peak_probe_measured)",
        "peak_probe_measured": dmma_probe_tflops, "frac_of_probe": achieved / dmma_probe_tflops,
        "probe_launches_outside_timed_region": probe_launches,
        "algorithmic_flops_per_launch": issued_flops, "kernel_ms": gemm_avg_ms, "split_ms": sum(split_ms) / len(split_ms),
        "kernel_share_of_step": gemm_avg_ms / ms_per_step,
        "kernel_timing": ("library CUDA events on the call's stream inside the timed region" if profile_inside else
                          "library CUDA events in a second loop of the same K steps (a step is below 1 ms: three event records per "
                          "call inside the timed loop would distort it)"),
        "traffic": None,
    }
    # DRAM bytes of one launch of this kernel from the committed ncu --set full capture (cfg2 only), else null
    traffic_file = os.path.join(ROOT, "profiles", "qgemm_traffic.txt")
    if os.path.exists(traffic_file) and args.config == 2:
        src = {}
        for ln in open(traffic_file):
            if "=" in ln and not ln.startswith("#"):
                key, val = ln.split("=", 1)
                src[key.strip()] = val.strip()
        if "dram_bytes_per_launch" in src:
            roofline["traffic"] = int(src["dram_bytes_per_launch"])
            roofline["traffic_source"] = ("NOT measured in this run: ncu --set full capture %s taken at commit %s (profiles/qgemm_traffic.txt); "
                                          "stale if the kernel has changed since" % (src.get("capture", "?"), src.get("commit", "?")))

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        try:
            v, dt, threads = cpu_oracle_sample(base, CPU_SAMPLE_ROWS)
        except Exception as exc:  # noqa: BLE001
            v, dt, threads = None, None, 0
            print(f"bench.py: cpu_baseline failed: {exc}", file=sys.stderr)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "seconds": dt,
                        "sample": f"first {CPU_SAMPLE_ROWS} rows of A ({CPU_SAMPLE_ROWS}x{base.n} outputs of the "
                                  f"{base.m}x{base.n}x{base.k} problem), all of B; oracle split + {base.products} plain "
                                  f"fp64 quarter GEMM loops + exact renorm, OpenMP over rows"}
        # the same leg also checks the device result of THIS run against the oracle's exact product (long accumulator) at a few
        # seeded positions: a bench line whose numbers come from a wrong C should say so
        try:
            from oracle import md_oracle as orc
            si, sj = inputs.sample_indices(cfg, 64, salt=4242)
            chk = orc.exact_samples(A_host.numpy(), B_host.numpy(), si, sj, C.cpu().numpy())
            tol = {2: 1e-28, 4: 1e-58, 8: 1e-120, 16: 1e-245}[L]
            ratio = float((chk["err"] / (tol * chk["W"])).max())
            cpu_baseline["sampled_parity"] = {"positions": 64, "max_err_over_tol_W": ratio, "within_tolerance": bool(ratio <= 1.0),
                                              "tolerance": f"{tol:g} (|A||B|)_ij, exact product from the oracle's long accumulator"}
        except Exception as exc:  # noqa: BLE001
            cpu_baseline["sampled_parity"] = {"error": f"{type(exc).__name__}: {exc}"}

    in_mib, qp_mib = (A.numel() + B.numel() + C.numel()) * 8 / 2 ** 20, 8.0 * Q * (m * k + k * n) / 2 ** 20
    if in_mib > 126:
        l2_note = "operands and result (%.0f MiB) and quarter planes (%.0f MiB) exceed the 126 MB L2; no explicit flush" % (in_mib, qp_mib)
    else:
        l2_note = ("operands and result (%.2f MiB) and quarter planes (%.2f MiB) FIT the 126 MB L2 and are not flushed between steps: "
                   "a WARM-L2 number (a small problem called back to back)" % (in_mib, qp_mib))
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": value / PAPER_DD_4096_GFLOPS if args.config == 2 else None,
        "dtype": "f64", "data": "synthetic",
        "config": {
            "workload": f"BASELINE.json configs[{base.index}] {base.name}: m={base.m} n={base.n} k={base.k} per GPU, "
                        f"limbs={L}, quarters={Q} of {W} bits, orders={S} (T={base.products} quarter products), seed {base.seed}",
            "slices": args.slices,
            "parallelism": "single GPU" if world == 1 else f"rows of A sharded over {world} GPUs, B replicated, no collective",
            "l2": l2_note,
            "paper_baseline": "PAPER.md:184 Table 1 t_TC(dd, n=4096) = 7.93621 s = 17.3 GFLOP/s on A100 or RTX 4080 (unstated)",
        },
        "fp64_tflops_issued": world * base.fp64_flops / (ms_per_step * 1e-3) / 1e12,
        "pct_of_fp64_tensor_peak": 100.0 * base.fp64_flops / (ms_per_step * 1e-3) / 1e12 / FP64_TENSOR_PEAK_TFLOPS,
        "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": launches,
        "adaptive_slices": adaptive, "paper_paths": paper_paths, "quarter_plan": quarter_plan,
        "clocks": clocks, "status_flags": flags,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.micro:
        run_micro(args)
    elif args.balance_table:
        run_balance_table(args)
    elif args.qr:
        run_qr(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

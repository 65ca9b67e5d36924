"""Build libmdgemm.so (the CUDA path + its C-ABI) in-tree with nvcc for sm_100a.

    python -m paper_2607_06881_b200.build [--force] [--verbose]

One object per .cu (compiled in parallel), linked with `nvcc -shared`.  No fast-math; -lineinfo so ncu's source page
maps to the kernels; --fmad=false as hygiene (the error-free transformations use explicit _rn intrinsics anyway).
"""
from __future__ import annotations

import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmdgemm.so")
COMPARE_LIB = os.path.join(HERE, "libmdcompare.so")
SOURCES = ["api.cu", "split.cu", "renorm.cu", "qgemm.cu", "qgemm_packed.cu", "qgemm_wide.cu", "probe.cu", "plan.cu", "literal.cu", "qr.cu", "fused_small.cu", "static_gemm.cu"]
HEADERS = [os.path.join(CSRC, "api_internal.h"), os.path.join(CSRC, "md_common.cuh"), os.path.join(CSRC, "md_arith.cuh"), os.path.join(CSRC, "md_kernels.h"), os.path.join(CSRC, "md_packed.cuh"), os.path.join(CSRC, "md_split.cuh"),
           os.path.join(CSRC, "qgemm_common.cuh"), os.path.join(CSRC, "qgemm_pipeline.cuh"),
           os.path.join(os.path.dirname(HERE), "include", "mdgemm.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "--fmad=false",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = _nvcc()
    objs, jobs = [], []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(CSRC, src.replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s] + HEADERS):
            cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
            jobs.append(cmd)
    if jobs:
        with concurrent.futures.ThreadPoolExecutor(max_workers=len(jobs)) as pool:
            for cmd, res in zip(jobs, pool.map(lambda c: subprocess.run(c, capture_output=True, text=True), jobs)):
                if verbose or res.returncode:
                    sys.stderr.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
                if res.returncode:
                    raise RuntimeError("nvcc failed: " + " ".join(cmd))
    if jobs or force or _stale(LIB, objs):
        subprocess.check_call([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs)
    build_compare(nvcc, force, verbose)
    return LIB


def build_compare(nvcc: str, force: bool = False, verbose: bool = False) -> str:
    """libmdcompare.so (include/mdcompare.h): the paper's own two paths as comparison beside the product -- links cuBLAS
    (the plain DGEMM of the top-down path) and libmdgemm.so (md_split / md_renorm through the C-ABI)."""
    src = os.path.join(CSRC, "compare", "compare.cu")
    deps = [src, LIB, os.path.join(os.path.dirname(HERE), "include", "mdcompare.h"),
            os.path.join(os.path.dirname(HERE), "include", "mdgemm.h")]
    if force or _stale(COMPARE_LIB, deps):
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + [
            "-shared", src, "-o", COMPARE_LIB, "-L" + HERE, "-l:libmdgemm.so", "-lcublas",
            "-Xlinker", "-rpath=$ORIGIN"]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode:
            sys.stderr.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
        if res.returncode:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    return COMPARE_LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))

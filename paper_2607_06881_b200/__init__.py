"""B200 (sm_100a) multiple-double matrix multiplication on the FP64 tensor pipe -- the hot path of
arxiv/paper_2607_06881 ("Multiple Double Arithmetic on NVIDIA Tensor Cores").

    from paper_2607_06881_b200 import binding as md     # md.md_gemm, md.md_split, md.md_qgemm, md.md_renorm, ...
    from paper_2607_06881_b200 import inputs            # seeded synthetic workloads (no method arithmetic)

The binding loads libmdgemm.so lazily and raises if it is missing; there is no CPU fallback.
"""

"""Seeded synthetic MSA inputs (layouts + values).

This package is the ONLY code shared by the fp64 oracle (``oracle/``) and the CUDA
path (``paper_2606_02964_b200/``).  It holds no attention arithmetic: it draws
lengths, cuts, residency kinds, block tables and bf16 values, and lays them out
in the physical representation (paged pool + block table, contiguous arena,
segment descriptors) that both sides consume.
"""
from .msa_inputs import (  # noqa: F401
    SEG_PAGED, SEG_CONTIG, SEG_SELF,
    ContextSpec, RunSpec, MsaProblem,
    build_problem, random_problem,
    cfg1_tiny, cfg2_llama8b, cfg3_70b_long, cfg4_mixed, cfg5_short_query, f1_hybrid_pod, f2_fig13,
    CONFIGS, EXTRA_CONFIGS, pick_rows, visible_pairs, to_fp8_pool,
)

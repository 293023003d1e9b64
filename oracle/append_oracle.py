"""KV write-back as its plain definition -- TEST INFRASTRUCTURE ONLY (tests/, bench.py's baseline legs).

include/msa.h, msa_append: arena rows [row_off, row_off + len) go to block block_table[block_off + i // 16], slot i % 16
(PAPER.md:92 step 2: recomputed K/V are written into cache blocks).  One Python loop per token, numpy views, no library call.
Pin (tests/test_kv_append.py): after the write-back, the fp64 attention oracle gives bit-identical results whether the
segment is described as CONTIG rows of the arena or as PAGED blocks of the pool (the cut / residency invariance the MSA
oracle itself is pinned with).
"""
from __future__ import annotations

from typing import Iterable, Tuple

import numpy as np


def kv_append(pool: np.ndarray, arena: np.ndarray, block_table: np.ndarray,
              jobs: Iterable[Tuple[int, int, int]]) -> np.ndarray:
    """pool [num_blocks][16][...], arena [rows][...] (same trailing shape); returns the updated copy of pool."""
    out = pool.copy()
    for row_off, n, block_off in jobs:
        for i in range(n):
            out[int(block_table[block_off + i // 16]), i % 16] = arena[row_off + i]
    return out

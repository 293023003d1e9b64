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


def quantize_e4m3(values: np.ndarray, scale: float, decode) -> np.ndarray:
    """fp8 pool (include/msa.h, msa_kv_append on an MSA_POOL_FP8_E4M3 handle): the E4M3 code nearest to value / scale,
    ties to the even code, |value / scale| beyond 448 saturates to +-448, NaN gives the NaN code 0x7f.  Written as the
    definition: a search over the 127 non-negative finite codes, whose values come from `decode` (the oracle's own E4M3
    decoder, oracle.e4m3_to_double).  Pin (tests/test_kv8.py): torch's float8_e4m3fn conversion inside +-448, closed forms
    outside it and at the ties."""
    grid = np.array([decode(c) for c in range(0x7f)], np.float64)          # ascending: code order is value order
    v = np.asarray(values, np.float64) / float(scale)
    out = np.zeros(v.shape, np.uint8)
    flat_v, flat_o = v.reshape(-1), out.reshape(-1)
    for i, x in enumerate(flat_v):
        if np.isnan(x):
            flat_o[i] = 0x7f
            continue
        a = abs(x)
        if a >= grid[-1]:
            c = 0x7e
        else:
            hi = int(np.searchsorted(grid, a, side="left"))                 # grid[hi-1] < a <= grid[hi]
            lo = max(hi - 1, 0)
            d_lo, d_hi = a - grid[lo], grid[hi] - a
            c = lo if d_lo < d_hi else hi if d_hi < d_lo else (lo if lo % 2 == 0 else hi)
        flat_o[i] = c | (0x80 if np.signbit(x) else 0)
    return out

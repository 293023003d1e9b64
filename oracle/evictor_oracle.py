"""Plain O(n) statement of the paper's eviction rule -- TEST INFRASTRUCTURE ONLY (tests/, bench.py's baseline legs).

Follows the paper line by line, no ordered sets, no log-domain keys:
  Eq. (7)       dT_B   = 2*k5*pos_B + c0            (pos_B = tokens in front of block B)
  Eq. (9)       f_B(t) = min(exp(-tau/alpha), exp(-(tau - tau0)/beta)),  tau = t - last_access(B)
  Eq. (3)   evict argmin_B f_B(t) * dT_B
  Algorithm 1 line 8 generalises the argmin with lambda: argmin{ min_B w1, lambda * min_B w2 };
  Eq. (10) says which lambda moves the turning point to a lifespan tau:
  lambda = exp((tau - tau0)/beta - tau/alpha), i.e. w1 == lambda*w2 for a block of exactly that age.
Shares no code with paper_2606_02964_b200/csrc/msa_evictor.cpp (which never forms these exponentials).

Pins (tests/test_evictor.py): constant dT degenerates to LRU; equal recency evicts the cheapest-to-
recompute block; the two branches of Eq. (9) cross at tau* = tau0*alpha/(alpha-beta); each branch obeys
the order-preserving rule Eq. (8); the lambda branch: with Eq. (10)'s lambda the two branch weights of a
block of age tau are equal, and the victim flips from the w1-minimum to the w2-minimum as lambda crosses that value.
"""
from __future__ import annotations

import math
from typing import Dict, Tuple


def delta_t(pos: int, k5: float, c0: float) -> float:
    """Eq. (7)."""
    return 2.0 * k5 * pos + c0


def branches(tau: float, alpha: float, beta: float, tau0: float) -> Tuple[float, float]:
    """The two exponentials of Eq. (9)."""
    return math.exp(-tau / alpha), math.exp(-(tau - tau0) / beta)


def frequency(tau: float, alpha: float, beta: float, tau0: float) -> float:
    """Eq. (9)."""
    return min(branches(tau, alpha, beta, tau0))


class LinearEvictor:
    """Algorithm 1 with the ordered sets replaced by a scan over every block (the O(n) strategy of PAPER.md:235)."""

    def __init__(self, alpha: float, beta: float, tau0: float, k5: float, c0: float, lambda_: float = 1.0):
        self.alpha, self.beta, self.tau0, self.k5, self.c0, self.lambda_ = alpha, beta, tau0, k5, c0, lambda_
        self.blocks: Dict[int, Tuple[int, float]] = {}          # id -> (pos, last access)

    def add(self, block_id: int, position: int, last_access: float) -> None:
        assert block_id not in self.blocks and delta_t(position, self.k5, self.c0) > 0.0
        self.blocks[block_id] = (position, last_access)

    def remove(self, block_id: int) -> None:
        del self.blocks[block_id]

    def weights(self, block_id: int, t: float) -> Tuple[float, float]:
        pos, last = self.blocks[block_id]
        e1, e2 = branches(t - last, self.alpha, self.beta, self.tau0)
        d = delta_t(pos, self.k5, self.c0)
        return e1 * d, e2 * d

    def weight(self, block_id: int, t: float) -> float:
        w1, w2 = self.weights(block_id, t)
        return min(w1, self.lambda_ * w2)

    def evict(self, t: float) -> int:
        b1 = min(self.blocks, key=lambda b: (self.weights(b, t)[0], b))
        b2 = min(self.blocks, key=lambda b: (self.weights(b, t)[1], b))
        victim = b1 if self.weights(b1, t)[0] <= self.lambda_ * self.weights(b2, t)[1] else b2
        del self.blocks[victim]
        return victim

    def __len__(self) -> int:
        return len(self.blocks)

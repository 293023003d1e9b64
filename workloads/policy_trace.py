"""Residency patterns decided by the paper's own eviction policy.

The five BASELINE.json configs draw which blocks are cached and which are recomputed at random.  Here the split comes
from Algorithm 1 (include/msa_evictor.h, the C++ evictor): a cache holds the KV blocks of many sessions, it is put under
pressure, the evictor chooses the victims, and the surviving blocks of every session become its PAGED segments while the
evicted runs become recomputed CONTIG segments.  Observation 2 of the paper then shows up by
itself: shared prefixes (recently touched by every session) and suffixes (expensive to recompute) survive, the middle goes.

No attention arithmetic here: the function only produces segment lists for ``workloads.build_problem``.
"""
from __future__ import annotations

import math
from typing import Dict, List, Tuple

import numpy as np

from . import msa_inputs as W

BLOCK = 16


def policy_residency(n_sessions: int = 48, keep_fraction: float = 0.6, seed: int = 1007,
                     k5: float = 1.2e-11, c0: float = 9.6e-8, alpha: float = 600.0, beta: float = 15.0,
                     tau0: float = 540.0, prefix_tokens: int = 512) -> Tuple[List[Dict], Dict]:
    """Returns per session {L, T, resident: bool per block} and a summary.  k5 / c0 default to the values refitted from
    measured msa_forward latencies on B200 (bench.py --workload costmodel, Eq. (6)/(7) of the paper)."""
    # the product's C++ evictor decides the victims (imported here, not at module level: the generator package
    # itself never depends on the product library)
    from paper_2606_02964_b200.binding import MsaEvictor
    rng = np.random.default_rng(seed)
    ev = MsaEvictor(alpha=alpha, beta=beta, tau0=tau0, k5=k5, c0=c0)
    t_now = 3000.0
    sessions = []
    next_id = 0
    owner: Dict[int, Tuple[int, int]] = {}
    for s in range(n_sessions):
        L = int(min(math.floor(math.exp(math.log(4096.0) + 0.8 * rng.standard_normal())), 16384))
        L = max(1024, L // BLOCK * BLOCK)
        T = int(rng.choice([256, 512, 1024]))
        # when the session's previous turn finished: three of four sessions are still inside the lifespan
        # (tau < tau0: the slow branch of Eq. (9), where the recomputation cost decides), the rest are stale
        last = float(t_now - rng.uniform(0.0, 0.9 * tau0)) if rng.random() < 0.75 else float(rng.uniform(0.0, t_now - tau0))
        nblk = L // BLOCK
        for b in range(nblk):
            # the shared system prompt is touched by every session, i.e. just now; the rest when the session last ran
            touched = t_now - 1.0 if b * BLOCK < prefix_tokens else last
            ev.add(next_id, b * BLOCK, touched)
            owner[next_id] = (s, b)
            next_id += 1
        sessions.append(dict(L=L, T=T, last=last, resident=np.ones(nblk, bool)))
    total = next_id
    n_evict = total - int(keep_fraction * total)
    for _ in range(n_evict):
        s, b = owner[ev.evict(t_now)]
        sessions[s]["resident"][b] = False
    ev.close()
    kept = np.concatenate([x["resident"] for x in sessions])
    summary = dict(blocks=total, evicted=int(n_evict), kept_fraction=float(kept.mean()),
                   sessions_fully_resident=int(sum(bool(x["resident"].all()) for x in sessions)),
                   sessions_fully_evicted=int(sum(not x["resident"].any() for x in sessions)))
    return sessions, summary


def f3_policy_trace(device="cpu", layout_only: bool = False, **kw):
    """The batch in which every session comes back with a new chunk of T tokens, Llama-3-8B heads."""
    sessions, summary = policy_residency(**kw)
    ctxs, runs = [], []
    cached_blocks = 0
    n_segments = []
    for s, x in enumerate(sessions):
        res = x["resident"]
        segs = []
        b = 0
        while b < len(res):
            e = b
            while e < len(res) and res[e] == res[b]:
                e += 1
            kind = W.SEG_PAGED if res[b] else W.SEG_CONTIG
            segs.append((kind, b * BLOCK, (e - b) * BLOCK))
            if res[b]:
                cached_blocks += e - b
            b = e
        n_segments.append(len(segs))
        segs.append((W.SEG_SELF, x["L"], x["T"]))
        ctxs.append(W.ContextSpec(segs))
        runs.append(W.RunSpec(s, x["L"], x["T"]))
    p = W.build_problem("f3_policy_trace", 32, 8, 128, ctxs, runs, seed=kw.get("seed", 1007), device=device,
                        pool_blocks=int(1.1 * cached_blocks) + 1, layout_only=layout_only)
    summary["segments_per_request_mean"] = float(np.mean(n_segments))
    summary["segments_per_request_max"] = int(np.max(n_segments))
    p.policy_summary = summary
    return p

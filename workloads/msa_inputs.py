"""Seeded generator of Multi-Segment-Attention (MSA) problems.

What it produces (and nothing else): the *physical* inputs of one MSA call, as
BASELINE.json's ``north_star`` words them -- a chunk of query tokens per
request, and a logically contiguous KV context that is physically split into
segments of three kinds:

* ``SEG_PAGED``   cached 16-token blocks in a shared pool, reached through a
                  (shuffled) block table
* ``SEG_CONTIG``  a run that was evicted and has just been recomputed into a
                  contiguous scratch arena
* ``SEG_SELF``    the current chunk's own K/V, also in the arena

Which segments are resident and which are recomputed stands in for the paper's
eviction policy / chunk scheduler; the recipes follow
SURVEY.md section 8(d) and are restated in DESIGN.md.  No dataset item is used:
the kernel only ever sees lengths and residency structure (PAPER.md:291 gives
the length scale).

No attention arithmetic lives here.  ``visible_pairs`` is integer bookkeeping
used to count algorithmic FLOPs / bytes for reporting.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np
import torch

SEG_PAGED, SEG_CONTIG, SEG_SELF = 0, 1, 2
BLOCK = 16  # tokens per paged block (BASELINE.json; PAPER.md:268-273 sizes are multiples of 16)


# --------------------------------------------------------------------------- specs
@dataclass
class ContextSpec:
    """Logical KV context shared by one or more query runs: [(kind, abs_start, len)]."""
    segs: List[Tuple[int, int, int]]


@dataclass
class RunSpec:
    """One query run: attends to context ``ctx``; its first token sits at ``q_abs_start``."""
    ctx: int
    q_abs_start: int
    q_len: int


@dataclass
class MsaProblem:
    name: str
    Hq: int
    Hkv: int
    D: int
    scale: float                      # the fp32 softmax scale, as a python float
    seed: int
    # descriptors (host, numpy)
    req: np.ndarray                   # int32 [n_req,5]: q_row_start,q_len,q_abs_start,seg_begin,seg_count
    seg_kind: np.ndarray              # int32 [n_seg]
    seg_abs_start: np.ndarray         # int32 [n_seg]
    seg_len: np.ndarray               # int32 [n_seg]
    seg_block_off: np.ndarray         # int32 [n_seg]  (PAGED: offset into block_table)
    seg_row_off: np.ndarray           # int64 [n_seg]  (CONTIG/SELF: first arena row)
    block_table_np: np.ndarray        # int32 [n_tbl]  physical block ids, logical order
    num_blocks: int
    contig_rows: int
    total_q: int
    q_to_kv: Optional[np.ndarray] = None   # int32 [Hq] or None (=> h // (Hq//Hkv))
    # values (torch, on `device`); None when layout_only
    q: Optional[torch.Tensor] = None           # bf16 [total_q,Hq,D]
    pool_k: Optional[torch.Tensor] = None      # bf16 [num_blocks,16,Hkv,D]
    pool_v: Optional[torch.Tensor] = None
    contig_k: Optional[torch.Tensor] = None    # bf16 [contig_rows,Hkv,D]
    contig_v: Optional[torch.Tensor] = None
    block_table: Optional[torch.Tensor] = None  # int32 [n_tbl] on device
    # dense, un-segmented copy per context (small problems only; CPU):
    # list of dict(pos=int64[n], k=bf16[n,Hkv,D], v=bf16[n,Hkv,D]) in ascending position
    dense: Optional[List[Dict[str, torch.Tensor]]] = None
    run_ctx: Optional[np.ndarray] = None       # int32 [n_req] context index of each run
    # fp8 paged pool: pool_k / pool_v are uint8 [num_blocks,16,Hkv,D] holding OCP E4M3 codes and
    # k_scale / v_scale float32 [Hkv] (powers of two) -- see to_fp8_pool(); None for a bf16 pool
    k_scale: Optional[np.ndarray] = None
    v_scale: Optional[np.ndarray] = None
    notes: Dict[str, object] = field(default_factory=dict)

    # ---- convenience -----------------------------------------------------
    @property
    def n_req(self) -> int:
        return int(self.req.shape[0])

    @property
    def n_seg(self) -> int:
        return int(self.seg_kind.shape[0])

    @property
    def G(self) -> int:
        return self.Hq // self.Hkv

    def head_map(self) -> np.ndarray:
        if self.q_to_kv is not None:
            return self.q_to_kv.astype(np.int32)
        return (np.arange(self.Hq, dtype=np.int32) // self.G).astype(np.int32)

    def kv_tokens(self, kind: Optional[int] = None) -> int:
        """Tokens of K/V a launch must read at least once per KV head (sum over runs); `kind`: only segments of that kind."""
        tot = 0
        for r in range(self.n_req):
            _, q_len, q_abs, sb, sc = (int(x) for x in self.req[r])
            p_last = q_abs + q_len - 1
            for s in range(sb, sb + sc):
                if kind is not None and int(self.seg_kind[s]) != kind:
                    continue
                a, n = int(self.seg_abs_start[s]), int(self.seg_len[s])
                tot += max(0, min(n, p_last - a + 1))
        return tot

    def algorithmic(self) -> Dict[str, float]:
        """Algorithmic work of one msa_forward: FLOPs = 4*D*Hq*pairs;
        bytes = visible K and V once per KV head + Q + O + LSE + block ids."""
        pairs = visible_pairs(self)
        kv_tok = self.kv_tokens()
        kv_bytes = kv_tok * self.Hkv * self.D * 2 * 2
        if self.k_scale is not None:       # fp8 pool: one byte per cached element
            kv_bytes -= self.kv_tokens(SEG_PAGED) * self.Hkv * self.D * 2
        qo_bytes = self.total_q * self.Hq * self.D * 2 * 2 + self.total_q * self.Hq * 4
        id_bytes = int(self.block_table_np.size) * 4
        return dict(pairs_per_head=pairs, flops=4.0 * self.D * self.Hq * pairs,
                    kv_bytes=kv_bytes, qo_bytes=qo_bytes, id_bytes=id_bytes,
                    bytes=kv_bytes + qo_bytes + id_bytes)

    def host_arrays(self, reqs: Optional[Sequence[int]] = None) -> Dict[str, np.ndarray]:
        """Raw host (numpy) views for the oracle.  bf16 tensors become uint16 arrays.

        For multi-GB pools only the blocks / arena rows referenced by ``reqs`` are copied
        from the device; the rest of the host array is left uninitialised (it is never
        read by a correct gather)."""
        assert self.q is not None, "layout_only problem has no values"
        big = (self.pool_k.numel() + self.contig_k.numel()) * 2 > (1 << 30)
        kv8 = self.k_scale is not None

        def u16(t: torch.Tensor) -> np.ndarray:
            if t.dtype == torch.uint8:      # fp8 pool: the E4M3 codes as they are
                return t.detach().cpu().contiguous().numpy()
            return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)

        out: Dict[str, np.ndarray] = dict(
            q=u16(self.q), block_table=self.block_table_np,
            req=self.req, seg_kind=self.seg_kind, seg_abs_start=self.seg_abs_start,
            seg_len=self.seg_len, seg_block_off=self.seg_block_off, seg_row_off=self.seg_row_off,
            q_to_kv=self.head_map())
        if kv8:
            out.update(k_scale=np.asarray(self.k_scale, np.float32), v_scale=np.asarray(self.v_scale, np.float32))
        if not big or reqs is None:
            out.update(pool_k=u16(self.pool_k), pool_v=u16(self.pool_v),
                       contig_k=u16(self.contig_k), contig_v=u16(self.contig_v))
            return out
        pk = np.empty(tuple(self.pool_k.shape), np.uint8 if kv8 else np.uint16)
        pv = np.empty(tuple(self.pool_v.shape), np.uint8 if kv8 else np.uint16)
        ck = np.empty(tuple(self.contig_k.shape), np.uint16)
        cv = np.empty(tuple(self.contig_v.shape), np.uint16)
        blk_ids: List[np.ndarray] = []
        for r in sorted(set(int(x) for x in reqs)):
            sb, sc = int(self.req[r, 3]), int(self.req[r, 4])
            for s in range(sb, sb + sc):
                n = int(self.seg_len[s])
                if int(self.seg_kind[s]) == SEG_PAGED:
                    o = int(self.seg_block_off[s])
                    blk_ids.append(self.block_table_np[o:o + (n + BLOCK - 1) // BLOCK])
                else:
                    r0 = int(self.seg_row_off[s])
                    ck[r0:r0 + n] = u16(self.contig_k[r0:r0 + n])
                    cv[r0:r0 + n] = u16(self.contig_v[r0:r0 + n])
        if blk_ids:
            ids = np.unique(np.concatenate(blk_ids)).astype(np.int64)
            idt = torch.from_numpy(ids).to(self.pool_k.device)
            pk[ids] = u16(self.pool_k.index_select(0, idt))
            pv[ids] = u16(self.pool_v.index_select(0, idt))
        out.update(pool_k=pk, pool_v=pv, contig_k=ck, contig_v=cv)
        return out


# --------------------------------------------------------------------------- helpers
def _randn_bf16(shape: Tuple[int, ...], gen: torch.Generator, device: torch.device) -> torch.Tensor:
    """N(0,1) rounded to bf16, generated in bounded fp32 chunks along dim 0."""
    out = torch.empty(shape, dtype=torch.bfloat16, device=device)
    if out.numel() == 0:
        return out
    per_row = max(1, out[0].numel())
    rows = max(1, (1 << 27) // per_row)
    for r0 in range(0, shape[0], rows):
        r1 = min(shape[0], r0 + rows)
        out[r0:r1] = torch.randn((r1 - r0,) + tuple(shape[1:]), generator=gen, device=device,
                                 dtype=torch.float32).to(torch.bfloat16)
    return out


def visible_pairs(p: MsaProblem) -> int:
    """Number of (query row, visible key) pairs per q head: key visible iff abs_j <= p_i."""
    tot = 0
    for r in range(p.n_req):
        _, q_len, q_abs, sb, sc = (int(x) for x in p.req[r])
        for s in range(sb, sb + sc):
            a, n = int(p.seg_abs_start[s]), int(p.seg_len[s])
            # row i (position q_abs+i) sees clamp(q_abs+i-a+1, 0, n) keys of this segment
            c = np.arange(q_abs - a + 1, q_abs - a + 1 + q_len, dtype=np.int64)
            tot += int(np.clip(c, 0, n).sum())
    return tot


def pick_rows(p: MsaProblem, n_random: int, seed: int,
              reqs: Optional[Sequence[int]] = None) -> Tuple[np.ndarray, np.ndarray]:
    """Seeded row subset (request index, row-in-run) that always holds the first and last
    row of every chosen run and the rows whose position touches a segment boundary."""
    rng = np.random.default_rng(seed)
    rr: List[int] = []
    ii: List[int] = []
    chosen = range(p.n_req) if reqs is None else reqs
    for r in chosen:
        _, q_len, q_abs, sb, sc = (int(x) for x in p.req[r])
        rows = {0, q_len - 1}
        for s in range(sb, sb + sc):
            a, n = int(p.seg_abs_start[s]), int(p.seg_len[s])
            for pos in (a - 1, a, a + n - 1, a + n):
                i = pos - q_abs
                if 0 <= i < q_len:
                    rows.add(i)
        if n_random > 0:
            rows.update(int(x) for x in rng.integers(0, q_len, size=n_random))
        for i in sorted(rows):
            rr.append(int(r))
            ii.append(i)
    return np.asarray(rr, np.int32), np.asarray(ii, np.int32)


# --------------------------------------------------------------------------- builder
def build_problem(name: str, Hq: int, Hkv: int, D: int,
                  contexts: Sequence[ContextSpec], runs: Sequence[RunSpec], seed: int,
                  device: str | torch.device = "cpu", pool_blocks: Optional[int] = None,
                  fill: str = "random", keep_dense: bool = False, layout_only: bool = False,
                  q_to_kv: Optional[Sequence[int]] = None, scale: Optional[float] = None,
                  arena_gap: int = 0, shuffle_segments: bool = False,
                  table_seed: Optional[int] = None,
                  values: Optional[Dict[str, object]] = None) -> MsaProblem:
    """Lay out ``contexts``/``runs`` physically and (unless layout_only) draw bf16 values.

    fill: 'random' -> unused pool blocks / block tails / arena gaps hold finite N(0,1) data;
          'nan'    -> they hold NaN (poison test: a correct path never lets them reach O).
    keep_dense: also keep an un-segmented per-context copy (brute-force pin; CPU, small only).
    shuffle_segments: store each context's segment list in a seeded random order (the
          oracle accepts any order; the library requires ascending abs_start).
    table_seed: seed of the physical placement (block-table permutation) alone, so the same
          values can be re-laid-out differently; defaults to ``seed``.
    values: explicit values instead of random ones (implies keep_dense):
          {'q': bf16 [total_q,Hq,D], 'kv': [(k_by_pos, v_by_pos) per context]} where
          k_by_pos[a] is the key at absolute position a.
    """
    device = torch.device(device)
    rng = np.random.default_rng(seed)
    trng = rng if table_seed is None else np.random.default_rng(table_seed)
    if values is not None:
        keep_dense = True
    assert Hq % Hkv == 0
    # ---- descriptors ---------------------------------------------------------
    seg_kind: List[int] = []
    seg_abs: List[int] = []
    seg_len: List[int] = []
    seg_boff: List[int] = []
    seg_roff: List[int] = []
    ctx_range: List[Tuple[int, int]] = []
    n_tbl = 0
    n_rows = 0
    for c in contexts:
        order = list(range(len(c.segs)))
        if shuffle_segments:
            order = [int(x) for x in rng.permutation(len(c.segs))]
        b0 = len(seg_kind)
        for j in order:
            kind, a, n = c.segs[j]
            assert n >= 1 and a >= 0
            seg_kind.append(kind)
            seg_abs.append(a)
            seg_len.append(n)
            if kind == SEG_PAGED:
                seg_boff.append(n_tbl)
                seg_roff.append(0)
                n_tbl += (n + BLOCK - 1) // BLOCK
            else:
                n_rows += arena_gap
                seg_boff.append(0)
                seg_roff.append(n_rows)
                n_rows += n
        ctx_range.append((b0, len(seg_kind) - b0))
    n_rows += arena_gap
    num_blocks = max(int(pool_blocks or 0), n_tbl, 1)
    block_table_np = trng.permutation(num_blocks)[:n_tbl].astype(np.int32)
    req = np.zeros((len(runs), 5), np.int32)
    row = 0
    for i, r in enumerate(runs):
        b0, cnt = ctx_range[r.ctx]
        req[i] = (row, r.q_len, r.q_abs_start, b0, cnt)
        row += r.q_len
    total_q = row
    if scale is None:
        scale = float(np.float32(1.0) / np.sqrt(np.float32(D)))
    else:
        scale = float(np.float32(scale))
    p = MsaProblem(
        name=name, Hq=Hq, Hkv=Hkv, D=D, scale=scale, seed=seed, req=req,
        seg_kind=np.asarray(seg_kind, np.int32), seg_abs_start=np.asarray(seg_abs, np.int32),
        seg_len=np.asarray(seg_len, np.int32), seg_block_off=np.asarray(seg_boff, np.int32),
        seg_row_off=np.asarray(seg_roff, np.int64), block_table_np=block_table_np,
        num_blocks=num_blocks, contig_rows=max(n_rows, 1), total_q=total_q,
        q_to_kv=None if q_to_kv is None else np.asarray(q_to_kv, np.int32),
        run_ctx=np.asarray([r.ctx for r in runs], np.int32))
    if layout_only:
        return p
    # ---- values --------------------------------------------------------------
    gen = torch.Generator(device=device)
    gen.manual_seed(seed)
    if values is not None:
        p.q = values["q"].to(torch.bfloat16).reshape(total_q, Hq, D).to(device)
    else:
        p.q = _randn_bf16((total_q, Hq, D), gen, device)
    p.block_table = torch.from_numpy(block_table_np).to(device)
    if not keep_dense:
        assert fill == "random", "NaN poison needs keep_dense=True (small problems)"
        p.pool_k = _randn_bf16((num_blocks, BLOCK, Hkv, D), gen, device)
        p.pool_v = _randn_bf16((num_blocks, BLOCK, Hkv, D), gen, device)
        p.contig_k = _randn_bf16((p.contig_rows, Hkv, D), gen, device)
        p.contig_v = _randn_bf16((p.contig_rows, Hkv, D), gen, device)
        return p
    # dense first (un-segmented, ascending position), then scatter into the physical layout
    cpu_gen = torch.Generator(device="cpu")
    cpu_gen.manual_seed(seed + 7919)
    if fill == "nan":
        mk = lambda shape: torch.full(shape, float("nan"), dtype=torch.bfloat16)
    else:
        mk = lambda shape: _randn_bf16(shape, cpu_gen, torch.device("cpu"))
    pool_k = mk((num_blocks, BLOCK, Hkv, D))
    pool_v = mk((num_blocks, BLOCK, Hkv, D))
    ck = mk((p.contig_rows, Hkv, D))
    cv = mk((p.contig_rows, Hkv, D))
    dense: List[Dict[str, torch.Tensor]] = []
    for ci, (b0, cnt) in enumerate(ctx_range):
        order = sorted(range(b0, b0 + cnt), key=lambda s: seg_abs[s])
        pos_l, k_l, v_l = [], [], []
        for s in order:
            n = seg_len[s]
            if values is not None:
                kb, vb = values["kv"][ci]
                k = kb[seg_abs[s]:seg_abs[s] + n].to(torch.bfloat16).reshape(n, Hkv, D)
                v = vb[seg_abs[s]:seg_abs[s] + n].to(torch.bfloat16).reshape(n, Hkv, D)
            else:
                k = _randn_bf16((n, Hkv, D), cpu_gen, torch.device("cpu"))
                v = _randn_bf16((n, Hkv, D), cpu_gen, torch.device("cpu"))
            pos_l.append(torch.arange(seg_abs[s], seg_abs[s] + n, dtype=torch.int64))
            k_l.append(k)
            v_l.append(v)
            if seg_kind[s] == SEG_PAGED:
                ids = torch.from_numpy(block_table_np[seg_boff[s]:seg_boff[s] + (n + BLOCK - 1) // BLOCK]
                                       .astype(np.int64))
                flat_rows = (ids[:, None] * BLOCK + torch.arange(BLOCK)[None, :]).reshape(-1)[:n]
                pool_k.view(-1, Hkv, D)[flat_rows] = k
                pool_v.view(-1, Hkv, D)[flat_rows] = v
            else:
                ck[seg_roff[s]:seg_roff[s] + n] = k
                cv[seg_roff[s]:seg_roff[s] + n] = v
        dense.append(dict(pos=torch.cat(pos_l), k=torch.cat(k_l), v=torch.cat(v_l)))
    p.dense = dense
    p.pool_k, p.pool_v = pool_k.to(device), pool_v.to(device)
    p.contig_k, p.contig_v = ck.to(device), cv.to(device)
    return p


# --------------------------------------------------------------------------- fp8 paged pool
def to_fp8_pool(p: MsaProblem, k_exp: Optional[Sequence[int]] = None, v_exp: Optional[Sequence[int]] = None) -> MsaProblem:
    """The same problem with its paged pool stored as OCP FP8 E4M3 codes (KV footprint).

    k_exp / v_exp: per KV head, the power of two of the scale (k_scale[h] = 2**k_exp[h]); default: the smallest power of two
    that brings the head's largest |value| within E4M3's 448, so every head uses the format's full range.  The codes are
    produced with torch's float8_e4m3fn conversion (round to nearest even) of value / scale: this is input generation --
    both the oracle and the CUDA path start from the bytes.  Descriptors, q and the arena are shared with ``p``."""
    import copy
    assert p.pool_k is not None and p.pool_k.dtype == torch.bfloat16
    out = copy.copy(p)
    out.name = p.name + "_kv8"
    out.dense = None                         # the un-segmented bf16 copy no longer describes the pool

    def quant(pool: torch.Tensor, exps: Optional[Sequence[int]]):
        codes = torch.empty(pool.shape, dtype=torch.uint8, device=pool.device)
        scales = np.zeros(p.Hkv, np.float32)
        for h in range(p.Hkv):
            x = pool[:, :, h, :].float()
            fin = torch.where(torch.isfinite(x), x.abs(), torch.zeros_like(x))
            if exps is None:
                amax = float(fin.max()) if fin.numel() else 1.0
                e = int(math.ceil(math.log2(max(amax, 2.0 ** -20) / 448.0)))
            else:
                e = int(exps[h])
            scales[h] = np.float32(2.0 ** e)
            y = (x * (2.0 ** -e)).clamp(-448.0, 448.0)          # NaN stays NaN (poisoned slack in the tests)
            codes[:, :, h, :] = y.to(torch.float8_e4m3fn).view(torch.uint8)
        return codes, scales

    out.pool_k, out.k_scale = quant(p.pool_k, k_exp)
    out.pool_v, out.v_scale = quant(p.pool_v, v_exp)
    return out


# --------------------------------------------------------------------------- random problems
def random_problem(seed: int, n_req: int = 3, Hq: int = 4, Hkv: int = 2, D: int = 64,
                   max_ctx: int = 400, max_q: int = 96, max_segs: int = 5,
                   ragged: bool = True, gaps: bool = False, hybrid: bool = False,
                   device: str | torch.device = "cpu", fill: str = "random",
                   keep_dense: bool = True, pool_slack: float = 1.5, arena_gap: int = 0,
                   shuffle_segments: bool = False, min_ctx: int = 1,
                   q_to_kv: Optional[Sequence[int]] = None) -> MsaProblem:
    """Small random multi-request problem for property / parity tests.

    ragged: segment boundaries need not be multiples of 16 (partly filled blocks).
    gaps:   leave holes in absolute position between segments (attention over the union).
    hybrid: split the chunk into two query runs separated by a cached run, sharing one
            segment list (compute -> cached -> compute, PAPER.md:92 step 5, :247).
    """
    rng = np.random.default_rng(seed)
    contexts: List[ContextSpec] = []
    runs: List[RunSpec] = []
    blocks = 0
    for _ in range(n_req):
        L = int(rng.integers(min_ctx, max_ctx + 1))
        T = int(rng.integers(1, max_q + 1))
        if not ragged:
            L = max(BLOCK, L // BLOCK * BLOCK)
        k = int(rng.integers(1, max_segs + 1))
        k = max(1, min(k, L // (1 if ragged else BLOCK)))
        if ragged:
            cuts = sorted(set(int(x) for x in rng.integers(1, max(2, L), size=k - 1))) if L > 1 else []
        else:
            cuts = sorted(set(int(x) * BLOCK for x in rng.integers(1, max(2, L // BLOCK), size=k - 1)))
        cuts = [c for c in cuts if 0 < c < L]
        bounds = [0] + cuts + [L]
        segs: List[Tuple[int, int, int]] = []
        shift = 0
        for j in range(len(bounds) - 1):
            n = bounds[j + 1] - bounds[j]
            kind = SEG_PAGED if rng.random() < 0.6 else SEG_CONTIG
            if gaps and j > 0 and rng.random() < 0.5:
                shift += int(rng.integers(1, 40))
            segs.append((kind, bounds[j] + shift, n))
            if kind == SEG_PAGED:
                blocks += (n + BLOCK - 1) // BLOCK
        q0 = L + shift
        if gaps and rng.random() < 0.5:
            q0 += int(rng.integers(1, 20))
        ci = len(contexts)
        if hybrid and T >= 3:
            t1 = int(rng.integers(1, T - 1))
            mid = int(rng.integers(1, 3 * BLOCK))
            t2 = T - t1
            segs.append((SEG_SELF, q0, t1))
            kind = SEG_PAGED
            segs.append((kind, q0 + t1, mid))
            blocks += (mid + BLOCK - 1) // BLOCK
            segs.append((SEG_SELF, q0 + t1 + mid, t2))
            contexts.append(ContextSpec(segs))
            runs.append(RunSpec(ci, q0, t1))
            runs.append(RunSpec(ci, q0 + t1 + mid, t2))
        else:
            segs.append((SEG_SELF, q0, T))
            contexts.append(ContextSpec(segs))
            runs.append(RunSpec(ci, q0, T))
    return build_problem(f"random{seed}", Hq, Hkv, D, contexts, runs, seed, device=device,
                         pool_blocks=int(math.ceil(blocks * pool_slack)) + 1, fill=fill,
                         keep_dense=keep_dense, arena_gap=arena_gap,
                         shuffle_segments=shuffle_segments, q_to_kv=q_to_kv)


# --------------------------------------------------------------------------- the five configs
def cfg1_tiny(device="cpu", keep_dense=True, layout_only=False, fill="random") -> MsaProblem:
    """BASELINE.json configs[0]: 1 request, 64-token chunk, 4/4 heads, D=64, three segments."""
    ctx = ContextSpec([(SEG_PAGED, 0, 128), (SEG_CONTIG, 128, 64), (SEG_SELF, 192, 64)])
    return build_problem("cfg1_tiny", 4, 4, 64, [ctx], [RunSpec(0, 192, 64)], seed=1001,
                         device=device, pool_blocks=32, keep_dense=keep_dense,
                         layout_only=layout_only, fill=fill, scale=0.125)


def cfg2_llama8b(device="cpu", layout_only=False, n_req: int = 8) -> MsaProblem:
    """configs[1]: Llama-3-8B-shaped layer, 8 x (chunk 512 after 8192 prior in 4x2048
    alternating PAGED/CONTIG), block tables drawn from a 16384-block pool."""
    ctxs, runs = [], []
    for r in range(n_req):
        segs = [(SEG_PAGED, 0, 2048), (SEG_CONTIG, 2048, 2048), (SEG_PAGED, 4096, 2048),
                (SEG_CONTIG, 6144, 2048), (SEG_SELF, 8192, 512)]
        ctxs.append(ContextSpec(segs))
        runs.append(RunSpec(r, 8192, 512))
    return build_problem("cfg2_llama8b", 32, 8, 128, ctxs, runs, seed=1002, device=device,
                         pool_blocks=16384, layout_only=layout_only)


def cfg3_70b_long(device="cpu", layout_only=False) -> MsaProblem:
    """configs[2]: 70B-shaped long session, 64/8 heads, 32768 prior tokens cut at seeded
    block-aligned boundaries into 8 segments (~60% cached), chunk 2048."""
    rng = np.random.default_rng(1003)
    L, T = 32768, 2048
    while True:
        cuts = np.sort(rng.choice(np.arange(1, L // BLOCK), size=7, replace=False)) * BLOCK
        bounds = np.concatenate([[0], cuts, [L]])
        lens = np.diff(bounds)
        if lens.min() < 256:
            continue
        cached = lens[0::2].sum() / L
        if 0.55 <= cached <= 0.65:
            break
    segs = [((SEG_PAGED if j % 2 == 0 else SEG_CONTIG), int(bounds[j]), int(lens[j])) for j in range(8)]
    segs.append((SEG_SELF, L, T))
    return build_problem("cfg3_70b_long", 64, 8, 128, [ContextSpec(segs)], [RunSpec(0, L, T)],
                         seed=1003, device=device, pool_blocks=4096, layout_only=layout_only)


def cfg4_mixed(device="cpu", layout_only=False, n_req: int = 64) -> MsaProblem:
    """configs[3]: multi-turn mixed batch; lognormal prior lengths (median 4096, sigma 1.0,
    cap 32768, floor 64), chunk in {256,512,1024,2048}, 1-16 segments, evicted fraction
    U[0,0.8] marked middle-out (prefix and suffix stay cached)."""
    rng = np.random.default_rng(1004)
    ctxs, runs = [], []
    cached_blocks = 0
    for r in range(n_req):
        L = int(min(math.floor(math.exp(math.log(4096.0) + 1.0 * rng.standard_normal())), 32768))
        L = max(L, 64)
        T = int(rng.choice([256, 512, 1024, 2048]))
        k = int(rng.integers(1, 17))
        k = max(1, min(k, L // BLOCK))
        cuts = np.sort(rng.choice(np.arange(1, max(2, L // BLOCK)), size=min(k - 1, max(0, L // BLOCK - 1)),
                                  replace=False)) * BLOCK if k > 1 else np.zeros(0, np.int64)
        bounds = np.concatenate([[0], cuts, [L]]).astype(np.int64)
        lens = np.diff(bounds)
        f = float(rng.uniform(0.0, 0.8))
        kinds = [SEG_PAGED] * len(lens)
        mid = len(lens) // 2
        order = [mid]
        for d in range(1, len(lens)):
            if mid - d >= 0:
                order.append(mid - d)
            if mid + d < len(lens):
                order.append(mid + d)
        share = 0.0
        for j in order:
            new = share + lens[j] / L
            if abs(new - f) < abs(share - f):
                kinds[j] = SEG_CONTIG
                share = new
            else:
                break
        segs = [(kinds[j], int(bounds[j]), int(lens[j])) for j in range(len(lens))]
        cached_blocks += sum((int(lens[j]) + BLOCK - 1) // BLOCK for j in range(len(lens)) if kinds[j] == SEG_PAGED)
        segs.append((SEG_SELF, L, T))
        ctxs.append(ContextSpec(segs))
        runs.append(RunSpec(r, L, T))
    return build_problem("cfg4_mixed", 32, 8, 128, ctxs, runs, seed=1004, device=device,
                         pool_blocks=int(1.25 * cached_blocks) + 1, layout_only=layout_only)


def cfg5_short_query(device="cpu", layout_only=False, n_req: int = 256) -> MsaProblem:
    """configs[4]: short-query (decode/TPOT-like) batch; q_len U{1..8}, prior U[2048,16384]
    (ragged), up to 8 segments, at most 2 recomputed-contiguous (each <= 25% of L)."""
    rng = np.random.default_rng(1005)
    ctxs, runs = [], []
    cached_blocks = 0
    for r in range(n_req):
        T = int(rng.integers(1, 9))
        L = int(rng.integers(2048, 16385))
        k = int(rng.integers(1, 9))
        cuts = np.sort(rng.choice(np.arange(1, L // BLOCK), size=k - 1, replace=False)) * BLOCK if k > 1 \
            else np.zeros(0, np.int64)
        bounds = np.concatenate([[0], cuts, [L]]).astype(np.int64)
        lens = np.diff(bounds)
        kinds = [SEG_PAGED] * len(lens)
        n_contig = int(rng.integers(0, 3))
        cand = [j for j in range(len(lens)) if lens[j] <= 0.25 * L]
        if cand and n_contig:
            for j in rng.choice(cand, size=min(n_contig, len(cand)), replace=False):
                kinds[int(j)] = SEG_CONTIG
        segs = [(kinds[j], int(bounds[j]), int(lens[j])) for j in range(len(lens))]
        cached_blocks += sum((int(lens[j]) + BLOCK - 1) // BLOCK for j in range(len(lens)) if kinds[j] == SEG_PAGED)
        segs.append((SEG_SELF, L, T))
        ctxs.append(ContextSpec(segs))
        runs.append(RunSpec(r, L, T))
    return build_problem("cfg5_short_query", 32, 8, 128, ctxs, runs, seed=1005, device=device,
                         pool_blocks=int(1.02 * cached_blocks) + 1, layout_only=layout_only)


def f1_hybrid_pod(device="cpu", layout_only=False, n_prefill: int = 16, n_decode: int = 128) -> MsaProblem:
    """hybrid chunks and decode rows in ONE launch (PAPER.md:92 step 5, :247;
    the POD-Attention setting of PAPER.md:310).  Llama-3-8B shape.  Each prefill request: prior context
    L = 16 * U{256..512} tokens in 4 segments alternating cached-paged / recomputed-contiguous, then a
    chunk of 512 positions of which the middle 128 are already cached: compute run A (256 tokens),
    cached run (128, paged), compute run B (128 tokens); both runs share one segment list.  Each decode
    request: one query token behind U[1024, 8192] cached tokens (paged, one contiguous tail <= 64)."""
    rng = np.random.default_rng(1006)
    ctxs, runs = [], []
    cached_blocks = 0
    for r in range(n_prefill):
        L = BLOCK * int(rng.integers(256, 513))
        cuts = np.sort(rng.choice(np.arange(1, L // BLOCK), size=3, replace=False)) * BLOCK
        bounds = np.concatenate([[0], cuts, [L]]).astype(np.int64)
        segs = []
        for j in range(4):
            kind = SEG_PAGED if j % 2 == 0 else SEG_CONTIG
            n = int(bounds[j + 1] - bounds[j])
            segs.append((kind, int(bounds[j]), n))
            if kind == SEG_PAGED:
                cached_blocks += (n + BLOCK - 1) // BLOCK
        segs += [(SEG_SELF, L, 256), (SEG_PAGED, L + 256, 128), (SEG_SELF, L + 384, 128)]
        cached_blocks += 128 // BLOCK
        ci = len(ctxs)
        ctxs.append(ContextSpec(segs))
        runs.append(RunSpec(ci, L, 256))
        runs.append(RunSpec(ci, L + 384, 128))
    for r in range(n_decode):
        L = int(rng.integers(1024, 8193))
        tail = int(rng.integers(0, 65))
        segs = [(SEG_PAGED, 0, L - tail)]
        cached_blocks += (L - tail + BLOCK - 1) // BLOCK
        if tail:
            segs.append((SEG_CONTIG, L - tail, tail))
        segs.append((SEG_SELF, L, 1))
        ci = len(ctxs)
        ctxs.append(ContextSpec(segs))
        runs.append(RunSpec(ci, L, 1))
    return build_problem("f1_hybrid_pod", 32, 8, 128, ctxs, runs, seed=1006, device=device,
                         pool_blocks=int(1.1 * cached_blocks) + 1, layout_only=layout_only)


def f2_fig13(cached_tokens: int, layout: str, device="cpu", new_tokens: int = 128, keep_dense: bool = False,
             recompute_tokens: Optional[int] = None) -> MsaProblem:
    """the request shape of the paper's Fig. 13, Llama-3-8B heads:
    "a variable number of cached tokens [N] and ends with 128 new (uncached) tokens".  The figure itself is missing
    from PAPER.md, so how long the uncached history is stays a reading (DESIGN.md c18): R = N recomputed tokens.

      'prefix_new'  [cached N][new 128]                   one run of 128 (what remains when nothing was evicted)
      'prefix'      [cached N][recompute R + new 128]     caching from the prefix: ONE run of R+128 tokens behind N cached
      'suffix'      [recompute R][cached N][new 128]      caching from the suffix: TWO runs (R tokens at position 0, the
                                                          128 new ones at R+N) sharing one segment list -- the
                                                          two-segment instance of Eq. (2)
    """
    N, T = int(cached_tokens), int(new_tokens)
    R = N if recompute_tokens is None else int(recompute_tokens)
    if layout == "prefix_new":
        ctx = ContextSpec([(SEG_PAGED, 0, N), (SEG_SELF, N, T)])
        runs = [RunSpec(0, N, T)]
    elif layout == "prefix":
        ctx = ContextSpec([(SEG_PAGED, 0, N), (SEG_SELF, N, R + T)])
        runs = [RunSpec(0, N, R + T)]
    elif layout == "suffix":
        ctx = ContextSpec([(SEG_SELF, 0, R), (SEG_PAGED, R, N), (SEG_SELF, R + N, T)])
        runs = [RunSpec(0, 0, R), RunSpec(0, R + N, T)]
    else:
        raise ValueError(layout)
    return build_problem(f"f2_fig13_{layout}_{N}", 32, 8, 128, [ctx], runs, seed=1300 + N, device=device,
                         keep_dense=keep_dense)


CONFIGS = dict(cfg1_tiny=cfg1_tiny, cfg2_llama8b=cfg2_llama8b, cfg3_70b_long=cfg3_70b_long,
               cfg4_mixed=cfg4_mixed, cfg5_short_query=cfg5_short_query)
# workloads beyond BASELINE.json's five (SURVEY.md section 8 (f) "next" rows)
EXTRA_CONFIGS = dict(f1_hybrid_pod=f1_hybrid_pod)

"""Pins for the fp64 oracle (oracle/msa_oracle.c) -- CPU only, no product code.

The paper prints no worked numeric example for MSA, so the oracle is
pinned to what the paper and the mathematics fix:

P1  brute force over the generator's UN-segmented dense copy (never touches descriptors)
P2  library routine: torch SDPA / logsumexp in float64 with an explicit mask, including
    the Eq. (2) two-call decomposition and plain causal self-attention
P3  segment-cut invariance ("any number of non-contiguous cache segments")
P4  block-table permutation invariance (lossless claim) -- bit identical
P5  LSE-merge identity over a split context, incl. an empty side
P6  closed forms (uniform scores, V==1, V[0]=position, query at position 0)
P7  future independence (causality by absolute position)
P8  key-shift invariance of softmax
P9  visible-pair counts: sum_i (p_i+1), bounded by Eq. (4)'s rectangles
"""
import math

import numpy as np
import pytest
import torch

import oracle
import workloads as W
from workloads import SEG_CONTIG, SEG_PAGED, SEG_SELF, ContextSpec, RunSpec, build_problem

TOL = 1e-12


def _dense_ref_sdpa(p):
    """Per run: torch SDPA (float64, explicit boolean mask) over the un-segmented copy."""
    O = np.zeros((p.total_q, p.Hq, p.D))
    LSE = np.zeros((p.total_q, p.Hq))
    hm = torch.from_numpy(p.head_map().astype(np.int64))
    for r in range(p.n_req):
        r0, T, qa, _, _ = (int(x) for x in p.req[r])
        d = p.dense[int(p.run_ctx[r])]
        q = p.q[r0:r0 + T].cpu().double().permute(1, 0, 2)                   # [Hq,T,D]
        k = d["k"].double().permute(1, 0, 2)[hm]                              # [Hq,n,D]
        v = d["v"].double().permute(1, 0, 2)[hm]
        mask = d["pos"][None, :] <= (qa + torch.arange(T))[:, None]          # [T,n]
        any_vis = mask.any(dim=1)
        safe = mask.clone()
        safe[~any_vis, 0] = True                                              # avoid NaN rows in SDPA
        scale = float(np.float32(p.scale))
        o = torch.nn.functional.scaled_dot_product_attention(q, k, v, attn_mask=safe[None], scale=scale)
        o[:, ~any_vis] = 0.0
        s = torch.einsum("htd,hnd->htn", q, k) * scale
        s = s.masked_fill(~mask[None], float("-inf"))
        lse = torch.logsumexp(s, dim=-1)
        O[r0:r0 + T] = o.permute(1, 0, 2).numpy()
        LSE[r0:r0 + T] = lse.permute(1, 0).numpy()
    return O, LSE


def _brute_force(p):
    """Plain loops over the dense copy; scores via numpy dot in float64."""
    O = np.zeros((p.total_q, p.Hq, p.D))
    LSE = np.full((p.total_q, p.Hq), -np.inf)
    hm = p.head_map()
    sc = float(np.float32(p.scale))
    for r in range(p.n_req):
        r0, T, qa, _, _ = (int(x) for x in p.req[r])
        d = p.dense[int(p.run_ctx[r])]
        pos = d["pos"].numpy()
        K = d["k"].double().numpy()
        V = d["v"].double().numpy()
        Q = p.q[r0:r0 + T].cpu().double().numpy()
        for i in range(T):
            vis = np.nonzero(pos <= qa + i)[0]
            if vis.size == 0:
                continue
            for h in range(p.Hq):
                s = sc * (K[vis, hm[h]] @ Q[i, h])
                m = s.max()
                w = np.exp(s - m)
                LSE[r0 + i, h] = m + math.log(w.sum())
                O[r0 + i, h] = (w[:, None] * V[vis, hm[h]]).sum(0) / w.sum()
    return O, LSE


def _close(a, b, tol=TOL):
    fin = np.isfinite(b)
    assert np.array_equal(np.isfinite(a), fin)
    assert np.array_equal(a[~fin], b[~fin])
    if fin.any():
        assert np.max(np.abs(a[fin] - b[fin])) <= tol, np.max(np.abs(a[fin] - b[fin]))


# ------------------------------------------------------------------------------ P1 / P2
@pytest.mark.parametrize("seed,kw", [
    (11, dict()),
    (12, dict(Hq=8, Hkv=2, D=8, max_ctx=300, ragged=True)),
    (13, dict(gaps=True)),
    (14, dict(hybrid=True)),
    (15, dict(Hq=4, Hkv=4, D=64, shuffle_segments=True, gaps=True, hybrid=True)),
    (16, dict(Hq=4, Hkv=2, D=16, q_to_kv=[1, 0, 0, 1])),
])
def test_p2_sdpa_library_routine(seed, kw):
    p = W.random_problem(seed, **kw)
    O, LSE = oracle.forward_problem(p)
    O2, LSE2 = _dense_ref_sdpa(p)
    _close(O, O2)
    _close(LSE, LSE2)


@pytest.mark.parametrize("seed", [21, 22])
def test_p1_brute_force_unsegmented(seed):
    p = W.random_problem(seed, n_req=2, max_ctx=300, max_q=40, D=8 if seed == 21 else 64, gaps=(seed == 22))
    O, LSE = oracle.forward_problem(p)
    O2, LSE2 = _brute_force(p)
    _close(O, O2)
    _close(LSE, LSE2)


def test_p1_cfg1_tiny_matches_brute_force():
    p = W.cfg1_tiny()
    O, LSE = oracle.forward_problem(p)
    O2, LSE2 = _brute_force(p)
    _close(O, O2)
    _close(LSE, LSE2)


def test_p2_eq2_two_run_decomposition():
    """Eq. (2), PAPER.md:104-112 (reading c1): O1 = Attn(Q1,K1,V1), O2 = Attn(Q2,K,V),
    O = Concat(O1,O2) -- and, the two runs being adjacent, equal to plain causal
    self-attention over H = Concat(h1,h2) (torch SDPA is_causal=True)."""
    Hq = Hkv = 2
    D, n1, n2 = 16, 37, 29
    g = torch.Generator().manual_seed(5)
    q = torch.randn(n1 + n2, Hq, D, generator=g).bfloat16()
    k = torch.randn(n1 + n2, Hkv, D, generator=g).bfloat16()
    v = torch.randn(n1 + n2, Hkv, D, generator=g).bfloat16()
    ctx = ContextSpec([(SEG_SELF, 0, n1), (SEG_SELF, n1, n2)])
    p = build_problem("eq2", Hq, Hkv, D, [ctx], [RunSpec(0, 0, n1), RunSpec(0, n1, n2)], seed=1,
                      values=dict(q=q, kv=[(k, v)]))
    O, _ = oracle.forward_problem(p)
    sc = float(np.float32(p.scale))
    f = torch.nn.functional.scaled_dot_product_attention
    qd, kd, vd = (t.double().permute(1, 0, 2) for t in (q, k, v))
    o1 = f(qd[:, :n1], kd[:, :n1], vd[:, :n1], is_causal=True, scale=sc)
    m2 = (torch.arange(n1 + n2)[None, :] <= (n1 + torch.arange(n2))[:, None])
    o2 = f(qd[:, n1:], kd, vd, attn_mask=m2[None], scale=sc)
    _close(O, torch.cat([o1, o2], dim=1).permute(1, 0, 2).numpy())
    o_full = f(qd, kd, vd, is_causal=True, scale=sc)
    _close(O, o_full.permute(1, 0, 2).numpy())


# ------------------------------------------------------------------------------ P3 / P4
def _values(Hq, Hkv, D, n_pos, T, seed):
    g = torch.Generator().manual_seed(seed)
    return dict(q=torch.randn(T, Hq, D, generator=g).bfloat16(),
                kv=[(torch.randn(n_pos, Hkv, D, generator=g).bfloat16(),
                     torch.randn(n_pos, Hkv, D, generator=g).bfloat16())])


def _cut(L, T, cuts, kinds):
    b = [0] + list(cuts) + [L]
    segs = [(kinds[j % len(kinds)], b[j], b[j + 1] - b[j]) for j in range(len(b) - 1)]
    segs.append((SEG_SELF, L, T))
    return ContextSpec(segs)


def test_p3_segment_cut_invariance():
    Hq, Hkv, D, L, T = 4, 2, 32, 333, 21
    vals = _values(Hq, Hkv, D, L + T, T, 3)
    base = None
    rng = np.random.default_rng(0)
    for n_seg in [1, 2, 3, 5, 8, 16]:
        cuts = sorted(int(x) for x in rng.choice(np.arange(1, L), size=n_seg - 1, replace=False))
        for kinds in ([SEG_PAGED], [SEG_CONTIG], [SEG_PAGED, SEG_CONTIG], [SEG_CONTIG, SEG_PAGED, SEG_PAGED]):
            p = build_problem("cut", Hq, Hkv, D, [_cut(L, T, cuts, kinds)], [RunSpec(0, L, T)], seed=n_seg,
                              values=vals, shuffle_segments=True)
            O, LSE = oracle.forward_problem(p)
            if base is None:
                base = (O, LSE)
            _close(O, base[0], 1e-13)
            _close(LSE, base[1], 1e-13)


def test_p4_block_table_permutation_invariance_bit_identical():
    Hq, Hkv, D, L, T = 4, 2, 32, 200, 9
    vals = _values(Hq, Hkv, D, L + T, T, 4)
    outs = []
    for ts in [1, 2, 3]:
        p = build_problem("perm", Hq, Hkv, D, [_cut(L, T, [48, 130], [SEG_PAGED, SEG_CONTIG])],
                          [RunSpec(0, L, T)], seed=9, values=vals, table_seed=ts, pool_blocks=64)
        outs.append((p.block_table_np.copy(),) + oracle.forward_problem(p))
    assert not np.array_equal(outs[0][0], outs[1][0])
    for t, O, LSE in outs[1:]:
        assert np.array_equal(O, outs[0][1]) and np.array_equal(LSE, outs[0][2])


# ------------------------------------------------------------------------------ P5
def test_p5_lse_merge_identity():
    Hq, Hkv, D, L, T = 4, 2, 32, 160, 12
    vals = _values(Hq, Hkv, D, L + T, T, 6)
    whole = _cut(L, T, [40, 96], [SEG_PAGED, SEG_CONTIG])
    O, LSE = oracle.forward_problem(build_problem("w", Hq, Hkv, D, [whole], [RunSpec(0, L, T)], 1, values=vals))
    for split in (1, 2, 3, 4):          # 4: side B is empty for every row (only the SELF tail ... nothing)
        A = ContextSpec(whole.segs[:split])
        B = ContextSpec(whole.segs[split:]) if split < 4 else ContextSpec([(SEG_CONTIG, L + T + 5, 3)])
        OA, LA = oracle.forward_problem(build_problem("a", Hq, Hkv, D, [A], [RunSpec(0, L, T)], 1, values=dict(
            q=vals["q"], kv=[(torch.cat([vals["kv"][0][0], torch.zeros(16, Hkv, D).bfloat16()]),
                              torch.cat([vals["kv"][0][1], torch.zeros(16, Hkv, D).bfloat16()]))])))
        OB, LB = oracle.forward_problem(build_problem("b", Hq, Hkv, D, [B], [RunSpec(0, L, T)], 1, values=dict(
            q=vals["q"], kv=[(torch.cat([vals["kv"][0][0], torch.zeros(16, Hkv, D).bfloat16()]),
                              torch.cat([vals["kv"][0][1], torch.zeros(16, Hkv, D).bfloat16()]))])))
        if split == 4:
            assert np.all(np.isneginf(LB)) and np.all(OB == 0.0)     # empty side: O=0, LSE=-inf
        with np.errstate(divide="ignore"):
            Lm = np.logaddexp(LA, LB)
        Om = np.exp(LA - Lm)[..., None] * OA + np.exp(LB - Lm)[..., None] * OB
        _close(Lm, LSE)
        _close(Om, O)


# ------------------------------------------------------------------------------ P6
def _const_problem(q, k_by_pos, v_by_pos, segs, runs, Hq, Hkv, D, **kw):
    return build_problem("cf", Hq, Hkv, D, [ContextSpec(segs)], runs, seed=2,
                         values=dict(q=q, kv=[(k_by_pos, v_by_pos)]), **kw)


def test_p6_uniform_scores_mean_of_v_and_log_n():
    Hq, Hkv, D = 2, 1, 8
    g = torch.Generator().manual_seed(8)
    # context with a gap: positions 0..49 and 70..99; chunk at 100..109
    P = 110
    k = torch.randn(P, Hkv, D, generator=g).bfloat16()
    v = torch.randn(P, Hkv, D, generator=g).bfloat16()
    segs = [(SEG_PAGED, 0, 50), (SEG_CONTIG, 70, 30), (SEG_SELF, 100, 10)]
    q = torch.zeros(10, Hq, D).bfloat16()                      # q = 0 -> all scores equal
    p = _const_problem(q, k, v, segs, [RunSpec(0, 100, 10)], Hq, Hkv, D)
    O, LSE = oracle.forward_problem(p)
    vd = v.double().numpy()
    for i in range(10):
        vis = list(range(0, 50)) + list(range(70, 100 + i + 1))
        _close(O[i, 0], vd[vis, 0].mean(0))
        _close(LSE[i], np.full(Hq, math.log(len(vis))))
    # identical keys, non-zero q: LSE = scale*q.k + ln n
    k1 = torch.randn(1, Hkv, D, generator=g).bfloat16().expand(P, Hkv, D).contiguous()
    q1 = torch.randn(10, Hq, D, generator=g).bfloat16()
    p = _const_problem(q1, k1, v, segs, [RunSpec(0, 100, 10)], Hq, Hkv, D)
    O, LSE = oracle.forward_problem(p)
    s = float(np.float32(p.scale)) * (q1.double().numpy() @ k1[0, 0].double().numpy())   # [10,Hq]
    for i in range(10):
        n = 50 + 30 + i + 1
        _close(LSE[i], s[i] + math.log(n), 1e-11)
        vis = list(range(0, 50)) + list(range(70, 100 + i + 1))
        _close(O[i, 1], vd[vis, 0].mean(0), 1e-12)


def test_p6_v_ones_and_position_ramp():
    Hq, Hkv, D, L, T = 4, 2, 16, 180, 40
    g = torch.Generator().manual_seed(9)
    q = torch.randn(T, Hq, D, generator=g).bfloat16()
    k = torch.randn(L + T, Hkv, D, generator=g).bfloat16()
    segs = [(SEG_PAGED, 0, 50), (SEG_CONTIG, 50, 77), (SEG_PAGED, 127, 53), (SEG_SELF, L, T)]
    # (ii) V == 1  =>  O == 1
    p = _const_problem(q, k, torch.ones(L + T, Hkv, D).bfloat16(), segs, [RunSpec(0, L, T)], Hq, Hkv, D)
    O, _ = oracle.forward_problem(p)
    _close(O, np.ones_like(O), 1e-13)
    # (iii) V[...,0] = absolute position (exact in bf16 up to 256), uniform scores => O[0] = p_i/2
    v = torch.zeros(L + T, Hkv, D)
    v[:, :, 0] = torch.arange(L + T, dtype=torch.float32)[:, None]
    assert torch.equal(v.bfloat16().float(), v)
    p = _const_problem(torch.zeros(T, Hq, D).bfloat16(), k, v.bfloat16(), segs, [RunSpec(0, L, T)], Hq, Hkv, D)
    O, LSE = oracle.forward_problem(p)
    pi = L + np.arange(T)
    _close(O[:, :, 0], np.repeat((pi / 2.0)[:, None], Hq, 1), 1e-11)
    _close(LSE, np.repeat(np.log(pi + 1.0)[:, None], Hq, 1))


def test_p6_query_at_position_zero_and_empty_row():
    Hq, Hkv, D = 2, 2, 8
    g = torch.Generator().manual_seed(10)
    q = torch.randn(3, Hq, D, generator=g).bfloat16()
    k = torch.randn(8, Hkv, D, generator=g).bfloat16()
    v = torch.randn(8, Hkv, D, generator=g).bfloat16()
    # run A starts at position 0 (row 0 sees only key 0); run B sits before every key -> empty rows
    segs = [(SEG_SELF, 0, 2), (SEG_PAGED, 5, 3)]
    p = _const_problem(q[:2], k, v, segs, [RunSpec(0, 0, 2)], Hq, Hkv, D)
    O, LSE = oracle.forward_problem(p)
    _close(O[0], v[0].double().numpy())
    s = float(np.float32(p.scale)) * (q[0].double().numpy() * k[0].double().numpy()).sum(-1)
    _close(LSE[0], s)
    segs = [(SEG_PAGED, 5, 3)]
    p = _const_problem(q, k, v, segs, [RunSpec(0, 2, 3)], Hq, Hkv, D)     # positions 2,3,4 < 5
    O, LSE = oracle.forward_problem(p)
    assert np.all(O == 0.0) and np.all(np.isneginf(LSE))


# ------------------------------------------------------------------------------ P7 / P8
def test_p7_future_independence():
    Hq, Hkv, D, L, T = 4, 2, 16, 96, 24
    vals = _values(Hq, Hkv, D, L + T, T, 12)
    ctx = _cut(L, T, [32, 70], [SEG_PAGED, SEG_CONTIG])
    O, LSE = oracle.forward_problem(build_problem("f", Hq, Hkv, D, [ctx], [RunSpec(0, L, T)], 1, values=vals))
    cut = L + 10                                     # change everything after position `cut`
    k2, v2 = vals["kv"][0][0].clone(), vals["kv"][0][1].clone()
    k2[cut + 1:] = 7.0
    v2[cut + 1:] = -3.0
    O2, LSE2 = oracle.forward_problem(build_problem("f", Hq, Hkv, D, [ctx], [RunSpec(0, L, T)], 1,
                                                    values=dict(q=vals["q"], kv=[(k2, v2)])))
    assert np.array_equal(O[:11], O2[:11]) and np.array_equal(LSE[:11], LSE2[:11])
    assert not np.array_equal(O[11:], O2[11:])


def test_p8_key_shift_invariance():
    Hq, Hkv, D, L, T = 4, 2, 16, 120, 16
    g = torch.Generator().manual_seed(13)
    quant = lambda t: (torch.round(t * 4) / 4).clamp(-3, 3)         # multiples of 1/4: k+u exact in bf16
    q = quant(torch.randn(T, Hq, D, generator=g)).bfloat16()
    k = quant(torch.randn(L + T, Hkv, D, generator=g))
    u = quant(torch.randn(1, Hkv, D, generator=g))
    v = torch.randn(L + T, Hkv, D, generator=g).bfloat16()
    assert torch.equal((k + u).bfloat16().float(), k + u)
    ctx = _cut(L, T, [33, 64, 100], [SEG_CONTIG, SEG_PAGED])
    mk = lambda kk: build_problem("s", Hq, Hkv, D, [ctx], [RunSpec(0, L, T)], 1, values=dict(q=q, kv=[(kk.bfloat16(), v)]))
    p = mk(k)
    O, LSE = oracle.forward_problem(p)
    O2, LSE2 = oracle.forward_problem(mk(k + u))
    _close(O2, O, 1e-10)
    hm = p.head_map()
    shift = float(np.float32(p.scale)) * np.einsum("thd,hd->th", q.double().numpy(), u[0].double().numpy()[hm])
    _close(LSE2 - LSE, shift, 1e-10)


# ------------------------------------------------------------------------------ P9
def test_p9_pair_counts_closed_forms_and_eq4_bound():
    # gap-free single-run contexts: pairs = sum_i (p_i + 1) = T*L + T(T+1)/2
    assert W.visible_pairs(W.cfg1_tiny(layout_only=True)) == 64 * 192 + 64 * 65 // 2 == 14368
    assert W.visible_pairs(W.cfg2_llama8b(layout_only=True)) == 8 * (512 * 8192 + 512 * 513 // 2) == 34605056
    assert W.visible_pairs(W.cfg3_70b_long(layout_only=True)) == 2048 * 32768 + 2048 * 2049 // 2 == 69207040
    # two-run hybrid layout l1,q1,l2,q2 of Eq. (4): causal triangles <= rectangles
    l1, q1, l2, q2 = 40, 24, 56, 31
    ctx = ContextSpec([(SEG_PAGED, 0, l1), (SEG_SELF, l1, q1), (SEG_CONTIG, l1 + q1, l2), (SEG_SELF, l1 + q1 + l2, q2)])
    p = build_problem("eq4", 2, 1, 8, [ctx], [RunSpec(0, l1, q1), RunSpec(0, l1 + q1 + l2, q2)], seed=1,
                      values=dict(q=torch.zeros(q1 + q2, 2, 8), kv=[(torch.zeros(200, 1, 8), torch.ones(200, 1, 8))]))
    exact = q1 * l1 + q1 * (q1 + 1) // 2 + q2 * (l1 + q1 + l2) + q2 * (q2 + 1) // 2
    assert W.visible_pairs(p) == exact <= q1 * (l1 + q1) + q2 * (l1 + q1 + l2 + q2)
    # and the oracle's own mask agrees: with q = 0, exp(LSE) = number of visible keys
    _, LSE = oracle.forward_problem(p)
    assert int(round(float(np.exp(LSE[:, 0]).sum()))) == exact


def test_generator_recipes_are_deterministic_and_well_formed():
    for name, fn in W.CONFIGS.items():
        a, b = fn(layout_only=True), fn(layout_only=True)
        assert np.array_equal(a.req, b.req) and np.array_equal(a.block_table_np, b.block_table_np)
        assert np.array_equal(a.seg_len, b.seg_len) and np.array_equal(a.seg_kind, b.seg_kind)
        assert len(np.unique(a.block_table_np)) == a.block_table_np.size      # distinct physical blocks
        for r in range(a.n_req):
            _, T, qa, sb, sc = (int(x) for x in a.req[r])
            ab, ln = a.seg_abs_start[sb:sb + sc], a.seg_len[sb:sb + sc]
            assert np.all(ab[1:] == ab[:-1] + ln[:-1]) and ab[0] == 0           # gap-free, sorted
            assert a.seg_kind[sb + sc - 1] == SEG_SELF and ab[-1] == qa and ln[-1] == T
    c3 = W.cfg3_70b_long(layout_only=True)
    cached = c3.seg_len[:8][c3.seg_kind[:8] == SEG_PAGED].sum() / 32768
    assert 0.55 <= cached <= 0.65 and c3.n_seg == 9
    c5 = W.cfg5_short_query(layout_only=True)
    assert c5.n_req == 256 and c5.req[:, 1].min() >= 1 and c5.req[:, 1].max() <= 8


# ---------------------------------------------------------------- P10: fp8 (E4M3) paged pool (reading c20)
def test_p10_e4m3_decoder_against_torch_and_the_formats_closed_forms():
    """The oracle's own E4M3 decoder: every one of the 256 codes against torch's float8_e4m3fn -> float32 conversion
    (a library routine that shares nothing with the oracle) and against what the OCP format fixes."""
    codes = torch.arange(256, dtype=torch.int32).to(torch.uint8)
    ref = codes.view(torch.float8_e4m3fn).float().numpy().astype(np.float64)
    mine = np.array([oracle.e4m3_to_double(c) for c in range(256)])
    nan = np.isnan(ref)
    assert nan.sum() == 2 and np.isnan(mine[0x7f]) and np.isnan(mine[0xff])        # S.1111.111, no infinities
    assert np.array_equal(np.isnan(mine), nan)
    assert np.array_equal(mine[~nan], ref[~nan])
    assert np.array_equal(np.signbit(mine[~nan]), np.signbit(ref[~nan]))            # -0 keeps its sign
    # closed forms: largest finite 448 = 2^8 * 1.75, smallest subnormal 2^-9, smallest normal 2^-6, one
    assert mine[0x7e] == 448.0 and mine[0xfe] == -448.0
    assert mine[0x01] == 2.0 ** -9 and mine[0x07] == 7 * 2.0 ** -9 and mine[0x08] == 2.0 ** -6
    assert mine[0x38] == 1.0 and mine[0x3c] == 1.5 and mine[0x40] == 2.0
    # monotone over the positive codes
    assert np.all(np.diff(mine[:0x7f]) > 0)


def _dequantised_twin(p8):
    """bf16 problem whose pool holds code * scale (exact in bf16 for power-of-two scales), made with torch's decoder."""
    import copy
    p = copy.copy(p8)
    for name, sc in (("pool_k", p8.k_scale), ("pool_v", p8.v_scale)):
        codes = getattr(p8, name)
        val = codes.view(torch.float8_e4m3fn).float() * torch.from_numpy(np.asarray(sc, np.float32))[None, None, :, None]
        assert torch.equal(val.to(torch.bfloat16).float()[torch.isfinite(val)], val[torch.isfinite(val)])
        setattr(p, name, val.to(torch.bfloat16))
    p.k_scale = p.v_scale = None
    return p


@pytest.mark.parametrize("seed", [5, 6, 7])
def test_p10_kv8_forward_equals_the_bf16_oracle_on_the_dequantised_pool(seed):
    """msa_oracle_forward_kv8 = msa_oracle_forward (pinned by P1-P9) on a pool that holds the dequantised values:
    a wrong scale index, K / V scale swapped, a wrong byte offset or a decoder slip changes the result."""
    p = W.random_problem(seed, n_req=3, Hq=8, Hkv=4, D=64, max_ctx=300, max_q=40, keep_dense=False)
    p8 = W.to_fp8_pool(p, k_exp=[-6, -5, -7, -4], v_exp=[-5, -6, -3, -7])          # different scale per head, K != V
    O8, L8 = oracle.forward_problem(p8)
    O, L = oracle.forward_problem(_dequantised_twin(p8))
    assert np.array_equal(O8, O) and np.array_equal(L8, L)
    # and it is not the bf16 problem's result (quantisation moved the values) nor scale-blind
    O0, _ = oracle.forward_problem(p)
    assert np.abs(O8 - O0).max() > 1e-3
    p8b = W.to_fp8_pool(p, k_exp=[-6, -5, -7, -4], v_exp=[-5, -6, -3, -7])
    p8b.v_scale = p8b.v_scale * 2
    Ob, Lb = oracle.forward_problem(p8b)
    assert np.abs(Ob - O8).max() > 1e-3 and np.array_equal(Lb, L8)                  # V's scale moves O, never LSE


def test_p10_kv8_scale_closed_form():
    """Only paged segments: doubling v_scale doubles O exactly; multiplying k_scale by 2 equals doubling the softmax scale."""
    ctx = ContextSpec([(SEG_PAGED, 0, 75)])
    p = build_problem("kv8_only_paged", 4, 2, 64, [ctx], [RunSpec(0, 70, 5)], seed=77)
    p8 = W.to_fp8_pool(p, k_exp=[-6, -6], v_exp=[-6, -6])
    O, L = oracle.forward_problem(p8)
    p8.v_scale = p8.v_scale * 2
    O2, L2 = oracle.forward_problem(p8)
    assert np.array_equal(O2, 2 * O) and np.array_equal(L2, L)
    p8.v_scale = p8.v_scale / 2
    p8.k_scale = p8.k_scale * 2
    O3, L3 = oracle.forward_problem(p8)
    p8.k_scale = p8.k_scale / 2
    p8.scale = float(np.float32(p8.scale * 2))
    O4, L4 = oracle.forward_problem(p8)
    assert np.allclose(O3, O4, atol=1e-13) and np.allclose(L3, L4, atol=1e-12)

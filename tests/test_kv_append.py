"""KV write-back (include/msa.h msa_kv_append): oracle pin, host validation, GPU parity (bit-exact)."""
import numpy as np
import pytest
import torch

import oracle
import workloads as W
from oracle.append_oracle import kv_append
from paper_2606_02964_b200 import (MsaError, MSA_ERR_INVALID_ARG, MSA_ERR_OUT_OF_RANGE, MSA_ERR_OVERLAP, MSA_ERR_UNSUPPORTED,
                                   MsaSession, make_descriptors, msa_append_plan_create, msa_append_plan_destroy, msa_create,
                                   msa_destroy, msa_forward, msa_forward_writeback, msa_kv_append, msa_plan_create,
                                   msa_plan_create_writeback, msa_plan_destroy, msa_plan_export, msa_workspace_bytes)
from workloads import SEG_PAGED

NAN16 = np.uint16(0x7FC0)          # bf16 NaN: whatever is not written must stay exactly this


def _jobs_and_redescription(p):
    """Every CONTIG / SELF segment gets fresh blocks behind the existing block table; returns
    (jobs, extended block table, extra blocks, seg_kind', seg_block_off')."""
    bt = p.block_table_np
    n_pool = int(p.pool_k.shape[0])
    jobs, kind2, boff2 = [], p.seg_kind.copy(), p.seg_block_off.copy()
    cursor = len(bt)
    for s in range(len(p.seg_kind)):
        if int(p.seg_kind[s]) != SEG_PAGED:
            n = int(p.seg_len[s])
            jobs.append((int(p.seg_row_off[s]), n, cursor))
            kind2[s], boff2[s] = SEG_PAGED, cursor
            cursor += (n + 15) // 16
    extra = cursor - len(bt)
    rng = np.random.default_rng(5)
    new_ids = n_pool + rng.permutation(extra)                        # shuffled fresh blocks
    return jobs, np.concatenate([bt, new_ids.astype(np.int32)]), extra, kind2, boff2


def test_oracle_append_then_paged_description_equals_contig_description():
    p = W.random_problem(301, n_req=3, Hq=4, Hkv=2, D=64, max_ctx=300, max_q=40, hybrid=True)
    a = p.host_arrays()
    jobs, bt2, extra, kind2, boff2 = _jobs_and_redescription(p)
    assert jobs
    a2 = dict(a)
    for name, arena in (("pool_k", a["contig_k"]), ("pool_v", a["contig_v"])):
        ext = np.concatenate([a[name], np.full((extra,) + a[name].shape[1:], NAN16, np.uint16)])
        a2[name] = kv_append(ext, arena, bt2, jobs)
    a2.update(block_table=bt2, seg_kind=kind2, seg_block_off=boff2)
    rr = np.concatenate([np.full(int(p.req[r, 1]), r, np.int32) for r in range(p.n_req)])
    ii = np.concatenate([np.arange(int(p.req[r, 1]), dtype=np.int32) for r in range(p.n_req)])
    O1, L1 = oracle.forward(a, p.Hq, p.Hkv, p.D, p.scale, rr, ii)
    O2, L2 = oracle.forward(a2, p.Hq, p.Hkv, p.D, p.scale, rr, ii)
    assert np.array_equal(O1, O2) and np.array_equal(L1, L2)
    # a ragged job leaves the tail of its last block alone
    n_tail = sum(1 for (_, n, _) in jobs if n % 16)
    assert n_tail > 0 and (a2["pool_k"] == NAN16).any()


def test_append_plan_validation():
    h = msa_create(4, 2, 64, device=-1)
    msa_append_plan_destroy(msa_append_plan_create(h, [(0, 40, 0), (40, 16, 3)]))
    msa_append_plan_destroy(msa_append_plan_create(h, []))
    for jobs, code in [([(0, 40, 0), (40, 16, 2)], MSA_ERR_OVERLAP),          # 40 tokens take blocks 0..2
                       ([(0, 0, 0)], MSA_ERR_INVALID_ARG), ([(-1, 4, 0)], MSA_ERR_INVALID_ARG),
                       ([(0, 4, -1)], MSA_ERR_INVALID_ARG)]:
        with pytest.raises(MsaError) as e:
            msa_append_plan_create(h, jobs)
        assert e.value.status == code, jobs
    msa_destroy(h)


@pytest.mark.gpu
@pytest.mark.parametrize("seed,kw", [(311, dict(Hq=8, Hkv=2, D=128, max_ctx=900, max_q=150)),
                                     (312, dict(Hq=4, Hkv=4, D=64, max_ctx=300, max_q=33, hybrid=True, n_req=5)),
                                     # an arena row of 4 KB: wider than the bulk-copy kernel's row limit, the plain copy kernel
                                     (313, dict(Hq=16, Hkv=16, D=128, max_ctx=260, max_q=40, n_req=2))])
def test_kv_append_matches_the_oracle_bit_for_bit_and_forward_sees_the_same_values(seed, kw):
    dev = "cuda:0"
    p = W.random_problem(seed, device=dev, fill="nan", **kw)
    jobs, bt2, extra, kind2, boff2 = _jobs_and_redescription(p)
    a = p.host_arrays()

    def ext(t):
        pad = torch.full((extra,) + tuple(t.shape[1:]), float("nan"), dtype=torch.bfloat16, device=dev)
        return torch.cat([t, pad]).contiguous()

    pool_k, pool_v = ext(p.pool_k), ext(p.pool_v)
    bt_dev = torch.from_numpy(bt2).to(dev)
    u16 = lambda t: t.cpu().view(torch.int16).numpy().view(np.uint16)
    want_k = kv_append(u16(pool_k), a["contig_k"], bt2, jobs)
    want_v = kv_append(u16(pool_v), a["contig_v"], bt2, jobs)
    h = msa_create(p.Hq, p.Hkv, p.D, p.q_to_kv)
    ap = msa_append_plan_create(h, jobs)
    msa_kv_append(h, ap, p.contig_k, p.contig_v, pool_k, pool_v, bt_dev, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert np.array_equal(u16(pool_k), want_k) and np.array_equal(u16(pool_v), want_v)
    with pytest.raises(MsaError) as e:
        msa_kv_append(h, ap, p.contig_k[:3], p.contig_v, pool_k, pool_v, bt_dev)
    assert e.value.status == MSA_ERR_OUT_OF_RANGE
    # the forward pass over the written blocks (PAGED description) equals the one over the arena rows
    with MsaSession(p) as s:
        o1, l1 = s.forward()
        o1, l1 = o1.clone(), l1.clone()
    R, n, S, m = make_descriptors(p.req, kind2, p.seg_abs_start, p.seg_len, boff2, p.seg_row_off)
    plan = msa_plan_create(h, R, n, S, m)
    nb = msa_workspace_bytes(plan)
    ws = torch.empty(max(nb, 16), dtype=torch.uint8, device=dev) if nb else None
    o2 = torch.zeros_like(p.q)
    l2 = torch.zeros(p.total_q, p.Hq, dtype=torch.float32, device=dev)
    msa_forward(h, plan, p.q, pool_k, pool_v, bt_dev, p.contig_k, p.contig_v, p.scale, o2, l2, ws)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2) and torch.equal(l1, l2)
    msa_plan_destroy(plan)
    msa_append_plan_destroy(ap)
    msa_destroy(h)


# ------------------------------------------------------------------ write-back fused into the forward launch
def test_writeback_plan_validation_and_writer_units():
    """Host side of msa_plan_create_writeback: every destination block is written by exactly one flagged unit per kv
    head; jobs that do not coincide with 16-token blocks of a segment, or that nobody attends to, are refused."""
    p = W.random_problem(321, n_req=4, Hq=8, Hkv=2, D=128, max_ctx=700, max_q=90, hybrid=True)
    jobs, bt2, extra, kind2, boff2 = _jobs_and_redescription(p)
    h = msa_create(p.Hq, p.Hkv, p.D, device=-1)
    R, n, S, m = make_descriptors(p.req, p.seg_kind, p.seg_abs_start, p.seg_len, p.seg_block_off, p.seg_row_off)
    plan = msa_plan_create_writeback(h, R, n, S, m, jobs)
    units = msa_plan_export(plan, 1)
    vbl = msa_plan_export(plan, 0)
    vb_dst, tile_writer = msa_plan_export(plan, 5), msa_plan_export(plan, 6)
    assert len(vb_dst) == len(vbl) and (vb_dst >= 0).sum() == sum((ln + 15) // 16 for _, ln, _ in jobs) > 0
    assert np.all(vbl["paged"][vb_dst >= 0] == 0)
    n_written = 0
    for ctx_vb, ctx_ti in sorted(set(zip(units["vb_begin"].tolist(), units["tile_info_begin"].tolist()))):
        mine = units[units["vb_begin"] == ctx_vb]
        n_tiles = (int(mine["vb_count"].max()) + 7) // 8
        for t in range(n_tiles):
            has_dst = bool((vb_dst[ctx_vb + 8 * t: ctx_vb + 8 * t + 8] >= 0).any())
            w = int(tile_writer[ctx_ti + t])
            assert (w >= 0) == has_dst
            if not has_dst:
                continue
            # the tile is stored by exactly one unit per kv head: a flagged unit of item w whose tile range holds t
            for kvh in range(p.Hkv):
                hit = mine[(mine["q_row0"] == w) & (mine["kvh"] == kvh) & (mine["tile_begin"] <= t) & (mine["tile_end"] > t)]
                assert len(hit) == 1 and int(hit["writeback"][0]) == 1 and int(hit["vb_count"][0]) > max(
                    b for b in range(8 * t, 8 * t + 8) if b < len(vb_dst) - ctx_vb and vb_dst[ctx_vb + b] >= 0)
            n_written += 1
    assert n_written > 0
    msa_plan_destroy(plan)
    # an ordinary plan through the same entry
    msa_plan_destroy(msa_plan_create_writeback(h, R, n, S, m, []))
    # a job shifted by 3 rows cuts the arena differently from the segment
    ro, ln, bo = jobs[0]
    bad = [(ro + 3, max(1, ln - 3), bo)] + jobs[1:]
    with pytest.raises(MsaError) as e:
        msa_plan_create_writeback(h, R, n, S, m, bad)
    assert e.value.status == MSA_ERR_UNSUPPORTED
    # rows that no segment of the batch holds
    with pytest.raises(MsaError) as e:
        msa_plan_create_writeback(h, R, n, S, m, jobs + [(int(p.contig_rows) + 64, 16, int(len(bt2)) + 8)])
    assert e.value.status == MSA_ERR_UNSUPPORTED
    # two jobs into the same block-table entries
    with pytest.raises(MsaError) as e:
        msa_plan_create_writeback(h, R, n, S, m, jobs + [(jobs[0][0], jobs[0][1], jobs[0][2])])
    assert e.value.status == MSA_ERR_OVERLAP
    msa_destroy(h)


@pytest.mark.gpu
@pytest.mark.parametrize("seed,kw", [(331, dict(Hq=8, Hkv=2, D=128, max_ctx=900, max_q=150)),
                                     (332, dict(Hq=4, Hkv=4, D=64, max_ctx=300, max_q=33, hybrid=True, n_req=5)),
                                     (333, dict(Hq=8, Hkv=2, D=128, max_ctx=5000, max_q=300, min_ctx=2500, n_req=6, arena_gap=5))])
def test_forward_writeback_is_forward_plus_kv_append_bit_for_bit(seed, kw):
    """One launch: O / LSE bit-identical to msa_forward on the same plan, and the pool bit-identical to the append
    oracle (every block, including the ones nobody writes and the tails of partly filled blocks: NaN canaries)."""
    dev = "cuda:0"
    p = W.random_problem(seed, device=dev, fill="nan", **kw)
    jobs, bt2, extra, kind2, boff2 = _jobs_and_redescription(p)
    a = p.host_arrays()

    def ext(t):
        pad = torch.full((extra,) + tuple(t.shape[1:]), float("nan"), dtype=torch.bfloat16, device=dev)
        return torch.cat([t, pad]).contiguous()

    pool_k, pool_v = ext(p.pool_k), ext(p.pool_v)
    bt_dev = torch.from_numpy(bt2).to(dev)
    u16 = lambda t: t.cpu().view(torch.int16).numpy().view(np.uint16)
    want_k = kv_append(u16(pool_k), a["contig_k"], bt2, jobs)
    want_v = kv_append(u16(pool_v), a["contig_v"], bt2, jobs)
    h = msa_create(p.Hq, p.Hkv, p.D, p.q_to_kv)
    R, n, S, m = make_descriptors(p.req, p.seg_kind, p.seg_abs_start, p.seg_len, p.seg_block_off, p.seg_row_off)
    plan = msa_plan_create_writeback(h, R, n, S, m, jobs)
    nb = msa_workspace_bytes(plan)
    ws = torch.empty(max(nb, 16), dtype=torch.uint8, device=dev) if nb else None
    o1, o2 = torch.zeros_like(p.q), torch.zeros_like(p.q)
    l1 = torch.zeros(p.total_q, p.Hq, dtype=torch.float32, device=dev)
    l2 = torch.zeros_like(l1)
    before_k = u16(pool_k).copy()
    msa_forward(h, plan, p.q, pool_k, pool_v, bt_dev, p.contig_k, p.contig_v, p.scale, o1, l1, ws)       # O / LSE only
    torch.cuda.synchronize()
    assert np.array_equal(u16(pool_k), before_k)
    msa_forward_writeback(h, plan, p.q, pool_k, pool_v, bt_dev, p.contig_k, p.contig_v, p.scale, o2, l2, ws)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2) and torch.equal(l1, l2)
    assert np.array_equal(u16(pool_k), want_k) and np.array_equal(u16(pool_v), want_v)
    # error paths
    plain = msa_plan_create(h, R, n, S, m)
    with pytest.raises(MsaError) as e:
        msa_forward_writeback(h, plain, p.q, pool_k, pool_v, bt_dev, p.contig_k, p.contig_v, p.scale, o2, l2, ws)
    assert e.value.status == MSA_ERR_INVALID_ARG
    with pytest.raises(MsaError) as e:
        msa_forward_writeback(h, plan, p.q, pool_k, pool_v, bt_dev[:len(p.block_table_np)], p.contig_k, p.contig_v, p.scale, o2, l2, ws)
    assert e.value.status == MSA_ERR_OUT_OF_RANGE
    msa_plan_destroy(plain)
    msa_plan_destroy(plan)
    msa_destroy(h)


# ------------------------------------------------------------------ debug check of the block ids
@pytest.mark.gpu
def test_check_block_ids_flags_the_smallest_bad_entry_a_plan_refers_to():
    """msa_check_block_ids (SURVEY.md 8(b) debug mode): -1 on a good table; the smallest offending block-table index when ids the
    plan refers to are negative or >= num_blocks; entries the plan does not use are ignored; forward and append plans alike."""
    from paper_2606_02964_b200 import msa_check_block_ids
    dev = "cuda:0"
    p = W.random_problem(321, n_req=3, Hq=8, Hkv=2, D=128, max_ctx=700, max_q=60, device=dev)
    h = msa_create(p.Hq, p.Hkv, p.D, p.q_to_kv)
    R, n, S, m = make_descriptors(p.req, p.seg_kind, p.seg_abs_start, p.seg_len, p.seg_block_off, p.seg_row_off)
    plan = msa_plan_create(h, R, n, S, m)
    vb = msa_plan_export(plan, 0)
    used = np.unique(vb["src"][(vb["paged"] != 0) & (vb["nvalid"] > 0)])
    assert len(used) >= 4
    nb = int(p.pool_k.shape[0])
    pad = 5                                                         # entries beyond the plan's: never looked at
    bt = torch.cat([p.block_table, torch.full((pad,), 10 ** 9, dtype=torch.int32, device=dev)])
    flag = torch.zeros(1, dtype=torch.int32, device=dev)
    st = torch.cuda.current_stream().cuda_stream

    def check(table, plan_=plan, ap_=None):
        msa_check_block_ids(h, plan_, ap_, table, nb, flag, st)
        torch.cuda.synchronize()
        return int(flag.item())

    assert check(bt) == -1
    lo, hi = int(used[1]), int(used[-2])
    bad = bt.clone()
    bad[hi] = nb                                                    # one past the pool
    assert check(bad) == hi
    bad[lo] = -3
    assert check(bad) == lo                                         # the smallest offending index
    unused = sorted(set(range(int(p.block_table.numel()))) - set(int(x) for x in used))
    if unused:
        only_unused = bt.clone()
        only_unused[unused[0]] = -1
        assert check(only_unused) == -1
    with pytest.raises(MsaError) as e:
        msa_check_block_ids(h, plan, None, bt[: int(used[-1])], nb, flag, st)
    assert e.value.status == MSA_ERR_OUT_OF_RANGE
    # an append plan: jobs into entries [2, 5) of a table of their own
    ap = msa_append_plan_create(h, [(0, 40, 2)])
    tbl = torch.tensor([10 ** 9, -7, 3, 1, 0, 10 ** 9], dtype=torch.int32, device=dev)
    assert check(tbl, None, ap) == -1
    tbl[4] = nb
    assert check(tbl, None, ap) == 4
    assert check(bt, plan, None) == -1
    msa_append_plan_destroy(ap)
    msa_plan_destroy(plan)
    msa_destroy(h)
    # write-back plans: the destinations count as well -- fused store (bf16 pool) and the fp8 pool's append plan
    from paper_2606_02964_b200 import MSA_POOL_FP8_E4M3
    p = W.random_problem(331, device=dev, Hq=8, Hkv=2, D=128, max_ctx=900, max_q=150)
    jobs, bt2, extra, _, _ = _jobs_and_redescription(p)
    nb2 = int(p.pool_k.shape[0]) + extra
    R, n, S, m = make_descriptors(p.req, p.seg_kind, p.seg_abs_start, p.seg_len, p.seg_block_off, p.seg_row_off)
    first_dst = int(jobs[0][2])
    for fmt in (0, MSA_POOL_FP8_E4M3):
        h = msa_create(p.Hq, p.Hkv, p.D, p.q_to_kv, pool_format=fmt)
        plan = msa_plan_create_writeback(h, R, n, S, m, jobs)
        tbl = torch.from_numpy(bt2).to(dev)
        msa_check_block_ids(h, plan, None, tbl, nb2, flag, st)
        torch.cuda.synchronize()
        assert int(flag.item()) == -1
        tbl[first_dst + 1] = nb2 + 4                                # a destination block beyond the pool
        msa_check_block_ids(h, plan, None, tbl, nb2, flag, st)
        torch.cuda.synchronize()
        assert int(flag.item()) == first_dst + 1, fmt
        msa_plan_destroy(plan)
        msa_destroy(h)

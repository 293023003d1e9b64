"""CPU tests of the C-ABI library's host side: it loads, exports what include/msa.h declares,
validates descriptors with the documented status codes, and its planner (virtual blocks,
causal horizons, persistent split-KV schedule) is arithmetically right.  No GPU compute."""
import ctypes
import os
import re

import numpy as np
import pytest

import workloads as W
from paper_2606_02964_b200 import (MsaError, MSA_ERR_INVALID_ARG, MSA_ERR_NO_DEVICE, MSA_ERR_OUT_OF_RANGE,
                                   MSA_ERR_OVERLAP, MSA_ERR_UNSORTED, MSA_ERR_UNSUPPORTED, LIB_PATH, binding,
                                   make_descriptors, msa_create, msa_destroy, msa_plan_create, msa_plan_destroy,
                                   msa_plan_export, msa_plan_get_info, msa_workspace_bytes)
from workloads import SEG_CONTIG, SEG_PAGED, SEG_SELF

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "msa.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(msa_[a-z_]+)\s*\(", hdr))
    assert {"msa_create", "msa_plan_create", "msa_forward", "msa_forward_host", "msa_workspace_bytes"} <= declared
    lib = ctypes.CDLL(LIB_PATH)
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in msa.h but not exported"
    assert set(binding.EXPORTS) == declared
    hdr2 = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "msa_evictor.h")).read(), flags=re.S)
    declared2 = set(re.findall(r"\b(msa_evictor_[a-z_]+)\s*\(", hdr2))
    for name in sorted(declared2):
        assert hasattr(lib, name), f"{name} declared in msa_evictor.h but not exported"
    assert set(binding.EVICTOR_EXPORTS) == declared2


def test_binding_constants_equal_the_headers():
    """Status codes, segment kinds, pool formats and MSA_STATIC_WS_BYTES of binding.py against include/msa.h, and every status
    code has a text of its own."""
    hdr = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "msa.h")).read(), flags=re.S)
    enums = {k: int(v) for k, v in re.findall(r"\b(MSA_[A-Z0-9_]+)\s*=\s*(-?\d+)", hdr)}
    assert len([k for k in enums if k.startswith("MSA_ERR_")]) == 10 and enums["MSA_OK"] == 0
    for name, value in enums.items():
        assert getattr(binding, name) == value, name
    m = re.search(r"#define\s+MSA_STATIC_WS_BYTES\s+\((\d+)u\s*<<\s*(\d+)\)", hdr)
    assert m and binding.MSA_STATIC_WS_BYTES == int(m.group(1)) << int(m.group(2))
    lib = binding._lib()
    texts = [lib.msa_strerror(v).decode() for k, v in enums.items() if k.startswith("MSA_ERR_") or k == "MSA_OK"]
    assert len(set(texts)) == len(texts) and "unknown status" not in texts
    assert lib.msa_strerror(-99).decode() == "unknown status"


def test_create_rejects_unsupported_shapes_and_reports_no_device():
    for args in [(32, 8, 96), (30, 8, 128), (64, 2, 128)]:          # head_dim, divisibility, G > 16
        with pytest.raises(MsaError) as e:
            msa_create(*args, device=-1)
        assert e.value.status == MSA_ERR_UNSUPPORTED
    with pytest.raises(MsaError) as e:
        msa_create(4, 2, 64, q_to_kv_head=[0, 0, 0, 1], device=-1)   # kv head 0 gets 3 q heads
    assert e.value.status == MSA_ERR_UNSUPPORTED
    with pytest.raises(MsaError) as e:
        msa_create(4, 2, 64, device=-1, block_size=32)
    assert e.value.status == MSA_ERR_UNSUPPORTED
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(MsaError) as e:                            # no silent CPU fallback
            msa_create(4, 2, 64, device=0)
        assert e.value.status == MSA_ERR_NO_DEVICE


def _plan(h, req, segs):
    kind, a, n, bo, ro = (list(x) for x in zip(*segs)) if segs else ([], [], [], [], [])
    R, nr, S, ns = make_descriptors(np.asarray(req, np.int32).reshape(-1, 5), kind, a, n, bo, ro)
    return msa_plan_create(h, R, nr, S, ns)


def test_descriptor_validation_status_codes():
    h = msa_create(4, 2, 64, device=-1)
    ok = [(SEG_PAGED, 0, 40, 0, 0), (SEG_CONTIG, 40, 10, 0, 0), (SEG_SELF, 50, 4, 0, 10)]
    msa_plan_destroy(_plan(h, [[0, 4, 50, 0, 3]], ok))
    cases = [
        ([[0, 4, 50, 0, 3]], [ok[1], ok[0], ok[2]], MSA_ERR_UNSORTED),
        ([[0, 4, 50, 0, 3]], [ok[0], (SEG_CONTIG, 39, 10, 0, 0), ok[2]], MSA_ERR_OVERLAP),
        ([[0, 4, 50, 0, 3]], [ok[0], (SEG_CONTIG, 0, 10, 0, 0), ok[2]], MSA_ERR_OVERLAP),
        ([[0, 4, 50, 0, 4]], ok, MSA_ERR_OUT_OF_RANGE),               # seg slice past the array
        ([[0, 4, 50, 0, 3]], [ok[0], (SEG_CONTIG, 40, 0, 0, 0), ok[2]], MSA_ERR_INVALID_ARG),   # len 0
        ([[0, 4, 50, 0, 3]], [(7, 0, 40, 0, 0), ok[1], ok[2]], MSA_ERR_INVALID_ARG),           # bad kind
        ([[0, 4, 50, 0, 3]], [(SEG_PAGED, 0, 40, -1, 0), ok[1], ok[2]], MSA_ERR_OUT_OF_RANGE),
        ([[0, 4, 50, 0, 3]], [ok[0], (SEG_CONTIG, 40, 10, 0, -5), ok[2]], MSA_ERR_OUT_OF_RANGE),
        ([[0, 4, 50, 0, 3], [2, 4, 50, 0, 3]], ok, MSA_ERR_OVERLAP),   # two runs write the same q rows
        ([[0, -1, 50, 0, 3]], ok, MSA_ERR_INVALID_ARG),
    ]
    for req, segs, code in cases:
        with pytest.raises(MsaError) as e:
            _plan(h, req, segs)
        assert e.value.status == code, (req, segs, e.value.status, code)
    msa_destroy(h)


def _check_plan(p):
    h = msa_create(p.Hq, p.Hkv, p.D, p.q_to_kv, device=-1)
    R, nr, S, ns = make_descriptors(p.req, p.seg_kind, p.seg_abs_start, p.seg_len, p.seg_block_off, p.seg_row_off)
    plan = msa_plan_create(h, R, nr, S, ns)
    info = msa_plan_get_info(plan)
    vb, units, cta, merge = (msa_plan_export(plan, k) for k in range(4))
    G = p.Hq // p.Hkv
    Rtok = info["rows_per_tile"] // G
    # P9: planner pair arithmetic == generator bookkeeping (closed form sum_i (p_i+1) on gap-free contexts)
    assert info["visible_pairs"] == W.visible_pairs(p)
    assert len(cta) == info["num_ctas"] + 1 and cta[0] == 0 and cta[-1] == len(units) and np.all(np.diff(cta) >= 0)
    # virtual blocks: every token of every referenced segment exactly once, positions ascending
    seen_ctx = {}
    for r in range(p.n_req):
        key = (int(p.req[r, 3]), int(p.req[r, 4]))
        seen_ctx.setdefault(key, None)
    # units of one item: contiguous tile ranges covering [0, n_tiles) exactly once
    items = {}
    for u in units:
        items.setdefault((int(u["q_row0"]), int(u["kvh"])), []).append(u)
    n_split = 0
    for (q_row0, kvh), us in items.items():
        us = sorted(us, key=lambda u: int(u["tile_begin"]))
        r = next(i for i in range(p.n_req) if p.req[i, 0] <= q_row0 < p.req[i, 0] + max(1, p.req[i, 1]))
        t0 = q_row0 - int(p.req[r, 0])
        left = int(p.req[r, 1]) - t0
        # groups of 2R tokens run as "pair" units; a remainder of <= R tokens as a "split" unit
        assert t0 % (2 * Rtok) == 0
        assert us[0]["n_tok"] == (min(2 * Rtok, left) if left > Rtok else left)
        assert all(int(u["mode"]) == (0 if left > Rtok else 1) for u in us)
        assert us[0]["q_abs0"] == int(p.req[r, 2]) + t0
        p_max = int(us[0]["q_abs0"]) + int(us[0]["n_tok"]) - 1
        blocks = vb[int(us[0]["vb_begin"]):]
        # horizon: exactly the virtual blocks of this context that start at or before p_max
        sb, sc = int(p.req[r, 3]), int(p.req[r, 4])
        n_ctx_vb = int(sum((int(p.seg_len[s]) + 15) // 16 for s in range(sb, sb + sc)))
        ctx_blocks = blocks[:n_ctx_vb]
        assert np.all(np.diff(ctx_blocks["abs_start"]) > 0)
        assert int(us[0]["vb_count"]) == int((ctx_blocks["abs_start"] <= p_max).sum())
        n_tiles = (int(us[0]["vb_count"]) + 7) // 8
        assert int(us[0]["tile_begin"]) == 0 and int(us[-1]["tile_end"]) == n_tiles
        for a, b in zip(us[:-1], us[1:]):
            assert int(a["tile_end"]) == int(b["tile_begin"]) and int(a["tile_end"]) > int(a["tile_begin"])
        if len(us) > 1:
            n_split += 1
            assert all(int(u["partial_off"]) >= 0 for u in us)
        else:
            assert int(us[0]["partial_off"]) == -1
    assert n_split == info["num_split_items"] == len(merge)
    assert len(items) == info["num_items"]
    # partial slots: disjoint, inside the workspace, 16-byte aligned
    spans = []
    for mi in merge:
        rows = int(mi["n_tok"]) * G
        assert int(mi["stride"]) >= rows * (p.D + 1) and int(mi["stride"]) % 4 == 0 and int(mi["first_off"]) % 4 == 0
        spans.append((int(mi["first_off"]), int(mi["first_off"]) + int(mi["stride"]) * int(mi["n_partials"])))
    spans.sort()
    for a, b in zip(spans[:-1], spans[1:]):
        assert a[1] <= b[0]
    assert msa_workspace_bytes(plan) == (spans[-1][1] * 4 if spans else 0)
    # virtual block contents against the raw descriptors
    for r in range(p.n_req):
        sb, sc = int(p.req[r, 3]), int(p.req[r, 4])
        key = (sb, sc)
        if seen_ctx[key] is not None or p.req[r, 1] == 0:
            continue
        seen_ctx[key] = True
        u0 = next(u for u in units if p.req[r, 0] <= u["q_row0"] < p.req[r, 0] + p.req[r, 1])
        i = int(u0["vb_begin"])
        for s in range(sb, sb + sc):
            n = int(p.seg_len[s])
            for b in range((n + 15) // 16):
                e = vb[i]
                assert e["abs_start"] == p.seg_abs_start[s] + 16 * b and e["nvalid"] == min(16, n - 16 * b)
                if p.seg_kind[s] == SEG_PAGED:
                    assert e["paged"] == 1 and e["src"] == p.seg_block_off[s] + b
                else:
                    assert e["paged"] == 0 and e["src"] == p.seg_row_off[s] + 16 * b
                i += 1
    # balance of the persistent schedule (whole items first, leftovers cut into the room that is left):
    # shares differ by a few snap windows at most
    per_cta = np.array([sum(max(1, int(u["tile_end"]) - int(u["tile_begin"])) * (2 if u["mode"] == 0 else 1)
                            for u in units[cta[c]:cta[c + 1]]) for c in range(info["num_ctas"])])
    if info["num_ctas"] > 1 and per_cta.sum() >= 148 * 16:
        assert per_cta.max() - per_cta.min() <= max(24, 0.01 * per_cta.mean()), (per_cta.min(), per_cta.max())
    # no sliver pieces: a split item is never cut within two tiles of its ends
    for (q_row0, kvh), us in items.items():
        if len(us) > 1:
            assert all(int(u["tile_end"]) - int(u["tile_begin"]) > 2 for u in us), (q_row0, kvh)
    # per-tile mask summaries agree with the (padded) virtual block list
    ti = msa_plan_export(plan, 4)
    assert len(vb) % 8 == 0 and len(ti) == len(vb) // 8
    for k in range(len(ti)):
        blk = vb[8 * k:8 * k + 8]
        valid = blk[blk["nvalid"] > 0]
        assert ti[k]["ragged"] == int((blk["nvalid"] < 16).any())
        assert ti[k]["max_abs"] == (int((valid["abs_start"] + valid["nvalid"] - 1).max()) if len(valid) else -1)
    msa_plan_destroy(plan)
    msa_destroy(h)
    return info


@pytest.mark.parametrize("name", list(W.CONFIGS))
def test_planner_on_the_five_configs(name):
    p = W.CONFIGS[name](layout_only=True)
    info = _check_plan(p)
    assert info["num_ctas"] <= 148
    if name != "cfg1_tiny":
        assert info["num_ctas"] == 148 and info["num_split_items"] <= 148


def test_planner_on_the_hybrid_prefill_plus_decode_workload():
    """several runs share one segment list, decode rows ride in the same launch."""
    info = _check_plan(W.f1_hybrid_pod(layout_only=True))
    assert info["num_ctas"] == 148 and info["num_split_items"] <= 148


@pytest.mark.parametrize("seed,kw", [(1, dict()), (2, dict(gaps=True, hybrid=True)), (3, dict(Hq=6, Hkv=2, max_ctx=3000)),
                                     (4, dict(n_req=9, max_q=5, max_ctx=50)), (5, dict(Hq=16, Hkv=1, D=128))])
def test_planner_on_random_problems(seed, kw):
    _check_plan(W.random_problem(seed, **kw))

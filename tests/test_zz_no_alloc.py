"""msa_forward_static_ws: the forward call for callers that cannot allocate its workspace.

Some users of libmsa have no way to get scratch memory at step time: a serving engine that gave every free byte of
HBM to its paged KV pool at start-up has nothing left for cudaMalloc to return, and code that runs next to in-flight
steps (or inside another framework's memory manager) must not call cudaMalloc / cudaFree at all, because both
synchronise the device.  For them the library carries a fixed 32 MiB array in its own device image and
msa_forward_static_ws uses that array as the split-KV workspace (include/msa.h has the contract).

What is checked here: the call gives the same O and LSE as msa_forward with a caller-allocated workspace -- the same
kernels run, so "the same" means bit for bit, the bar this suite uses wherever two CUDA launches of one kernel are
compared (test_split_kv_merge_path_and_determinism) -- on calls issued one after the other, so that each call after
the first finds the previous call's partials still lying in the shared array, under a different split layout.  The
reference path is also held against the fp64 oracle at the stated tolerances, so "equal to msa_forward" is anchored.
A plan that needs more than the array holds must be refused with MSA_ERR_STATIC_WS before anything is launched.

This file sorts last on purpose (pytest -x stops at the first failure, and a failure here should not hide the parity
tests); it passes on its own in a fresh process, where its first call is the one that does the per-device set-up.
"""
import numpy as np
import pytest
import torch

import oracle
import workloads as W
from paper_2606_02964_b200 import (MSA_ERR_NO_DEVICE, MSA_ERR_STATIC_WS, MSA_POOL_FP8_E4M3, MSA_STATIC_WS_BYTES, MsaError,
                                   MsaSession, make_descriptors, msa_create, msa_destroy, msa_forward_static_ws,
                                   msa_last_launch_count, msa_plan_create, msa_plan_destroy, msa_workspace_bytes)
from workloads import SEG_CONTIG, SEG_PAGED, SEG_SELF, ContextSpec, RunSpec, build_problem

DEV = "cuda:0"
TOL_O_MAX, TOL_O_MEAN, TOL_LSE = 2e-2, 2e-3, 1e-3          # BASELINE.json north_star, as in test_msa_gpu.py


def _long_stream(seed):
    """One request, 40 query rows on 6277 tokens of context: the schedule cuts it along KV, all 148 CTAs write partials."""
    ctx = ContextSpec([(SEG_PAGED, 0, 3000), (SEG_CONTIG, 3000, 1777), (SEG_PAGED, 4777, 1500), (SEG_SELF, 6277, 40)])
    return build_problem("static_ws_a", 8, 2, 128, [ctx], [RunSpec(0, 6277, 40)], seed=seed, device=DEV)


def _short_queries(seed):
    """Six decode-like requests of another head shape (D = 64): other partial sizes, offsets and strides in the array."""
    ctxs, runs, pos = [], [], [2100, 3333, 1234, 4000, 2777, 1900]
    for r, L in enumerate(pos):
        n = 1 + r % 5
        ctxs.append(ContextSpec([(SEG_PAGED, 0, L - 300), (SEG_CONTIG, L - 300, 300), (SEG_SELF, L, n)]))
        runs.append(RunSpec(r, L, n))
    return build_problem("static_ws_b", 8, 4, 64, ctxs, runs, seed=seed, device=DEV)


def _existing_path(s):
    """msa_forward with a workspace the caller allocated (MsaSession owns a torch buffer), checked against the oracle."""
    p = s.problem
    o, lse = s.forward()
    torch.cuda.synchronize()
    o, lse = o.clone(), lse.clone()
    O, LSE = oracle.forward_problem(p)
    d_o = np.abs(o.float().cpu().numpy().astype(np.float64) - O)
    d_l = np.abs(lse.cpu().numpy().astype(np.float64) - LSE)
    assert d_o.max() <= TOL_O_MAX and d_o.mean() <= TOL_O_MEAN and d_l.max() <= TOL_LSE
    return o, lse


def _static_path(s):
    """The same plan and tensors through msa_forward_static_ws, into output buffers that start as NaN."""
    p = s.problem
    o = torch.full_like(s.o, float("nan"))
    lse = torch.full_like(s.lse, float("nan"))
    msa_forward_static_ws(s.h, s.plan, p.q, p.pool_k, p.pool_v, p.block_table, p.contig_k, p.contig_v, p.scale, o, lse,
                          torch.cuda.current_stream().cuda_stream)
    launches = msa_last_launch_count(s.h)
    torch.cuda.synchronize()
    return o, lse, launches


@pytest.mark.gpu
def test_static_workspace_calls_in_a_row_match_msa_forward():
    with MsaSession(_long_stream(31)) as a, MsaSession(_short_queries(32)) as b:
        for s in (a, b):
            assert s.info["num_split_items"] > 0 and 0 < msa_workspace_bytes(s.plan) <= MSA_STATIC_WS_BYTES
        ref_a, ref_b = _existing_path(a), _existing_path(b)
        # a, b, a, a: every call but the first starts on the leftovers of the one before it -- of another layout (a -> b,
        # b -> a) and of its own (a -> a)
        for s, (ro, rl) in ((a, ref_a), (b, ref_b), (a, ref_a), (a, ref_a)):
            o, lse, launches = _static_path(s)
            assert launches == 2, "forward kernel + LSE-merge kernel"
            assert torch.equal(o, ro), f"O differs from msa_forward: max|d| = {(o.float() - ro.float()).abs().max().item()}"
            assert torch.equal(lse, rl), f"LSE differs from msa_forward: max|d| = {(lse - rl).abs().max().item()}"


@pytest.mark.gpu
def test_static_workspace_on_an_fp8_handle_and_a_side_stream():
    """An fp8 prefill plan keeps, besides the partials, the bf16 copy of its cached blocks and the copy's block table in the
    workspace (written by the dequantising pre-pass of the same call): through the built-in array, on a stream that is not
    the default one, twice in a row -- bit-identical to msa_forward with a caller workspace."""
    ctx = ContextSpec([(SEG_PAGED, 0, 500), (SEG_CONTIG, 500, 100), (SEG_SELF, 600, 300)])
    p = build_problem("static_ws_fp8", 8, 2, 128, [ctx], [RunSpec(0, 600, 300)], seed=34, device=DEV)
    p8 = W.to_fp8_pool(p, k_exp=[-6, -4], v_exp=[-5, -7])
    side = torch.cuda.Stream()
    with MsaSession(p8) as s:
        need = msa_workspace_bytes(s.plan)
        assert 2 * 32 * 16 * p8.Hkv * p8.D * 2 <= need <= MSA_STATIC_WS_BYTES          # the copy of 32 cached blocks is in there
        ro, rl = _existing_path(s)
        for _ in range(2):
            o = torch.full_like(s.o, float("nan"))
            lse = torch.full_like(s.lse, float("nan"))
            side.wait_stream(torch.cuda.current_stream())
            msa_forward_static_ws(s.h, s.plan, p8.q, p8.pool_k, p8.pool_v, p8.block_table, p8.contig_k, p8.contig_v, p8.scale,
                                  o, lse, side.cuda_stream)
            assert msa_last_launch_count(s.h) >= 2                                  # pre-pass + forward kernel (+ merge)
            side.synchronize()
            assert torch.equal(o, ro) and torch.equal(lse, rl)


@pytest.mark.gpu
def test_static_workspace_refuses_a_plan_beyond_its_size():
    """An fp8 prefill plan dequantises the cached blocks it refers to into the workspace: 640 blocks x 64 KiB > 32 MiB."""
    Hq, Hkv, D, L, T = 32, 8, 128, 640 * 16, 512
    ctx = ContextSpec([(SEG_PAGED, 0, L), (SEG_SELF, L, T)])
    p = build_problem("static_ws_big", Hq, Hkv, D, [ctx], [RunSpec(0, L, T)], seed=33, device="cpu", layout_only=True)
    h = msa_create(Hq, Hkv, D, None, device=0, pool_format=MSA_POOL_FP8_E4M3)
    R, n_req, S, n_seg = make_descriptors(p.req, p.seg_kind, p.seg_abs_start, p.seg_len, p.seg_block_off, p.seg_row_off)
    plan = msa_plan_create(h, R, n_req, S, n_seg)
    try:
        assert msa_workspace_bytes(plan) > MSA_STATIC_WS_BYTES
        q = torch.zeros((p.total_q, Hq, D), dtype=torch.bfloat16, device=DEV)
        o = torch.full_like(q, 7.0)
        lse = torch.full((p.total_q, Hq), 7.0, dtype=torch.float32, device=DEV)
        pool = torch.zeros((L // 16, 16, Hkv, D), dtype=torch.uint8, device=DEV)
        arena = torch.zeros((T, Hkv, D), dtype=torch.bfloat16, device=DEV)
        bt = torch.arange(L // 16, dtype=torch.int32, device=DEV)
        with pytest.raises(MsaError) as e:
            msa_forward_static_ws(h, plan, q, pool, pool, bt, arena, arena, 0.088, o, lse)
        assert e.value.status == MSA_ERR_STATIC_WS and "32 MiB" in str(e.value)
        torch.cuda.synchronize()
        assert bool((o == 7.0).all()) and bool((lse == 7.0).all())
    finally:
        msa_plan_destroy(plan)
        msa_destroy(h)


def test_static_workspace_on_a_planning_only_handle_reports_no_device():
    """CPU: the symbol is exported and a handle without a device is turned away before any CUDA call."""
    p = W.cfg1_tiny(device="cpu", layout_only=True)
    h = msa_create(p.Hq, p.Hkv, p.D, p.q_to_kv, device=-1)
    R, n_req, S, n_seg = make_descriptors(p.req, p.seg_kind, p.seg_abs_start, p.seg_len, p.seg_block_off, p.seg_row_off)
    plan = msa_plan_create(h, R, n_req, S, n_seg)
    try:
        with pytest.raises(MsaError) as e:
            msa_forward_static_ws(h, plan, np.zeros((p.total_q, p.Hq, p.D), np.uint16), None, None, None, None, None, 0.125,
                                  np.zeros(1, np.uint16), np.zeros(1, np.float32))
        assert e.value.status == MSA_ERR_NO_DEVICE
    finally:
        msa_plan_destroy(plan)
        msa_destroy(h)

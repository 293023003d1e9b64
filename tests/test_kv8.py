"""fp8 (E4M3) paged pool (include/msa.h MSA_POOL_FP8_E4M3; reading c20).

CPU part: host validation of the scales, the quantiser oracle's pins.  GPU part (-m gpu): the CUDA path against the fp64
oracle, which dequantises the same bytes itself -- same tolerances as the bf16 path (BASELINE.json north_star), because
code * 2^k is exactly a bf16 -- plus bit-identity with the bf16 kernel on the dequantised pool, and the quantising
msa_kv_append byte for byte.
"""
import numpy as np
import pytest
import torch

import oracle
import workloads as W
from oracle.append_oracle import kv_append, quantize_e4m3
from paper_2606_02964_b200 import (MSA_ERR_INVALID_ARG, MSA_ERR_UNSUPPORTED, MSA_POOL_FP8_E4M3, MsaError, MsaSession,
                                   make_descriptors, msa_append_plan_create, msa_append_plan_destroy, msa_create, msa_destroy,
                                   msa_kv_append, msa_plan_create_writeback, msa_plan_export)
from workloads import SEG_CONTIG, SEG_PAGED, SEG_SELF, ContextSpec, RunSpec, build_problem

DEV = "cuda:0"
TOL_O_MAX, TOL_O_MEAN, TOL_LSE = 2e-2, 2e-3, 1e-3


# ------------------------------------------------------------------ CPU: host logic and the quantiser oracle
def test_scales_must_be_powers_of_two_within_range():
    ok = msa_create(8, 2, 128, device=-1, pool_format=MSA_POOL_FP8_E4M3, k_scale=[0.25, 2.0 ** -14], v_scale=[2.0 ** 7, 1.0])
    msa_destroy(ok)
    msa_destroy(msa_create(8, 2, 128, device=-1, pool_format=MSA_POOL_FP8_E4M3))            # NULL scales: all 1.0
    for bad in ([0.3, 1.0], [2.0 ** -15, 1.0], [2.0 ** 8, 1.0]):
        with pytest.raises(MsaError) as e:
            msa_create(8, 2, 128, device=-1, pool_format=MSA_POOL_FP8_E4M3, k_scale=bad)
        assert e.value.status == MSA_ERR_UNSUPPORTED
    for bad in ([0.0, 1.0], [-1.0, 1.0], [float("nan"), 1.0], [float("inf"), 1.0]):
        with pytest.raises(MsaError) as e:
            msa_create(8, 2, 128, device=-1, pool_format=MSA_POOL_FP8_E4M3, v_scale=bad)
        assert e.value.status == MSA_ERR_INVALID_ARG
    with pytest.raises(MsaError) as e:
        msa_create(8, 2, 128, device=-1, pool_format=7)
    assert e.value.status == MSA_ERR_INVALID_ARG


def test_writeback_plan_on_an_fp8_pool_validates_like_an_append_plan():
    """An fp8 handle accepts write-back plans (forward kernel + quantising append kernel in one call); bad jobs are refused."""
    from paper_2606_02964_b200 import MSA_ERR_OVERLAP, msa_plan_destroy
    h = msa_create(4, 2, 64, device=-1, pool_format=MSA_POOL_FP8_E4M3)
    R, n_req, S, n_seg = make_descriptors(np.array([[0, 16, 16, 0, 2]], np.int32), [SEG_PAGED, SEG_SELF], [0, 16], [16, 16],
                                          [0, 0], [0, 0])
    msa_plan_destroy(msa_plan_create_writeback(h, R, n_req, S, n_seg, [(0, 16, 1)]))
    for jobs, code in (([(0, 16, 1), (0, 16, 1)], MSA_ERR_OVERLAP), ([(0, 0, 1)], MSA_ERR_INVALID_ARG)):
        with pytest.raises(MsaError) as e:
            msa_plan_create_writeback(h, R, n_req, S, n_seg, jobs)
        assert e.value.status == code
    msa_destroy(h)


def _kv8_path(p, device=-1):
    """Which way an fp8 handle would serve this batch: 'prepass' (cached blocks dequantised once, bf16 kernel), 'kernel_pair'
    or 'kernel_split' (codes converted inside the forward kernel, layout with two / one Q tiles)."""
    from paper_2606_02964_b200 import msa_plan_create, msa_plan_destroy, msa_workspace_bytes
    h = msa_create(p.Hq, p.Hkv, p.D, p.q_to_kv, device=device, pool_format=MSA_POOL_FP8_E4M3)
    R, n_req, S, n_seg = make_descriptors(p.req, p.seg_kind, p.seg_abs_start, p.seg_len, p.seg_block_off, p.seg_row_off)
    pl = msa_plan_create(h, R, n_req, S, n_seg)
    deq = msa_plan_export(pl, 7)
    units = msa_plan_export(pl, 1)
    ws = msa_workspace_bytes(pl)
    msa_plan_destroy(pl)
    msa_destroy(h)
    pair = bool(((units["mode"] == 0) & (units["tile_end"] > units["tile_begin"])).any())
    return ("prepass" if len(deq) else "kernel_pair" if pair else "kernel_split"), deq, ws


def _three_paths(device="cpu"):
    mk = lambda name, ctx, q0, T: build_problem(name, 8, 2, 128, [ContextSpec(ctx + [(SEG_SELF, q0, T)])], [RunSpec(0, q0, T)], seed=21,
                                                device=device)
    return dict(prepass=mk("reuse5", [(SEG_PAGED, 0, 500), (SEG_CONTIG, 500, 100)], 600, 300),      # five q-tile groups load every cached tile
                kernel_pair=mk("reuse1", [(SEG_PAGED, 0, 500), (SEG_CONTIG, 500, 100)], 600, 64),    # one group: converted in the kernel
                kernel_split=mk("short", [(SEG_PAGED, 0, 500), (SEG_CONTIG, 500, 100)], 600, 4))


def test_plan_chooses_prepass_by_reuse_of_the_cached_blocks():
    for want, p in _three_paths().items():
        path, deq, ws = _kv8_path(p)
        assert path == want, (want, path)
        if want == "prepass":
            # 500 cached tokens = 32 blocks, each listed once, in block-table order; the workspace holds their bf16 copy
            assert np.array_equal(deq, np.arange(32, dtype=np.int32))
            assert ws >= 2 * 32 * 16 * p.Hkv * p.D * 2
        else:
            # nothing but the split-KV partials a bf16 handle needs too
            from paper_2606_02964_b200 import msa_plan_create, msa_plan_destroy, msa_workspace_bytes
            hb = msa_create(p.Hq, p.Hkv, p.D, device=-1)
            R, n_req, S, n_seg = make_descriptors(p.req, p.seg_kind, p.seg_abs_start, p.seg_len, p.seg_block_off, p.seg_row_off)
            pl = msa_plan_create(hb, R, n_req, S, n_seg)
            assert ws == msa_workspace_bytes(pl)
            msa_plan_destroy(pl)
            msa_destroy(hb)
    # cfg2 loads every cached tile eight times, cfg5 once
    assert _kv8_path(W.cfg2_llama8b(layout_only=True))[0] == "prepass"
    assert _kv8_path(W.cfg5_short_query(layout_only=True))[0] == "kernel_split"


def test_quantiser_oracle_against_torch_and_closed_forms():
    rng = np.random.default_rng(11)
    x = np.concatenate([rng.standard_normal(4000) * 3, rng.uniform(-448, 448, 2000), rng.standard_normal(500) * 1e-3,
                        [0.0, -0.0, 448.0, -448.0, 2.0 ** -9, 2.0 ** -10, 3 * 2.0 ** -10]])
    x = torch.from_numpy(x).to(torch.bfloat16).double().numpy()              # what the arena can hold
    for scale in (1.0, 2.0 ** -6, 4.0):
        mine = quantize_e4m3(x * scale, scale, oracle.e4m3_to_double)
        ref = torch.from_numpy(x).float().to(torch.float8_e4m3fn).view(torch.uint8).numpy()   # library routine, |x| <= 448
        assert np.array_equal(mine, ref)
    # saturation and NaN (torch's conversion does not saturate, so these are closed forms)
    q = lambda v: int(quantize_e4m3(np.array([v]), 1.0, oracle.e4m3_to_double)[0])
    assert q(449.0) == 0x7e and q(1e30) == 0x7e and q(-1e30) == 0xfe and q(float("inf")) == 0x7e and q(float("nan")) == 0x7f
    # ties go to the even code: halfway between 1.0 (0x38) and 1.125 (0x39) -> 0x38; between 1.125 and 1.25 (0x3a) -> 0x3a
    assert q(1.0625) == 0x38 and q(1.1875) == 0x3a and q(2.0 ** -10) == 0x00 and q(3 * 2.0 ** -10) == 0x02
    # decode(quantise(v)) is the nearest representable value
    v = rng.uniform(-400, 400, 300)
    codes = quantize_e4m3(v, 1.0, oracle.e4m3_to_double)
    back = np.array([oracle.e4m3_to_double(int(c)) for c in codes])
    grid = np.array([oracle.e4m3_to_double(c) for c in range(256) if c not in (0x7f, 0xff)])
    assert np.allclose(np.abs(back - v), np.abs(grid[None, :] - v[:, None]).min(axis=1), atol=0)


# ------------------------------------------------------------------ GPU parity
def gpu_forward(p):
    with MsaSession(p) as s:
        o, lse = s.forward()
        torch.cuda.synchronize()
        return o.float().cpu().numpy().astype(np.float64), lse.cpu().numpy().astype(np.float64), s.info


def compare(p, o, lse, row_req=None, row_idx=None, strict=True, v_scale=1.0):
    """v_scale: the O tolerances are stated for V ~ N(0,1); the error of O is linear in V, so a test that scales V scales them."""
    O, LSE = oracle.forward_problem(p, row_req, row_idx)
    if row_req is not None:
        g = p.req[row_req, 0] + row_idx
        o, lse = o[g], lse[g]
    fin = np.isfinite(LSE)
    assert np.array_equal(np.isneginf(lse), ~fin), "rows without a visible key must give LSE=-inf"
    assert np.all(np.isfinite(o)), "non-finite O"
    assert np.all(o[~fin] == 0.0)
    d_o = np.abs(o - O)
    d_l = np.abs(lse[fin] - LSE[fin]) if fin.any() else np.zeros(1)
    if strict:
        assert d_o.max() <= TOL_O_MAX * v_scale, f"max|dO|={d_o.max()}"
    else:
        assert np.all(d_o <= TOL_O_MAX * v_scale * np.maximum(1.0, np.abs(O) / (2.0 * v_scale))), f"max|dO|={d_o.max()}"
    assert d_o.mean() <= TOL_O_MEAN * v_scale, f"mean|dO|={d_o.mean()}"
    assert d_l.max() <= TOL_LSE, f"max|dLSE|={d_l.max()}"
    return d_o.max(), d_o.mean(), d_l.max()


def _dequantised_twin(p8):
    """bf16 problem whose pool holds code * scale (exact in bf16 for power-of-two scales)."""
    import copy
    p = copy.copy(p8)
    for name, sc in (("pool_k", p8.k_scale), ("pool_v", p8.v_scale)):
        codes = getattr(p8, name)
        s = torch.from_numpy(np.asarray(sc, np.float32)).to(codes.device)[None, None, :, None]
        setattr(p, name, (codes.view(torch.float8_e4m3fn).float() * s).to(torch.bfloat16))
    p.k_scale = p.v_scale = None
    return p


def _against_the_bf16_kernel(p8, o, lse, v_scale=1.0):
    """code * 2^k is exactly a bf16.  The pre-pass and the two-Q-tile kernel variant feed those bf16 values to the same MMAs:
    bit-identical to the bf16 kernel on the dequantised pool.  The short-query variant multiplies the codes' f16 image and hands P
    over in f16 (three more mantissa bits than bf16): not the same bits, but the same scores up to fp32 rounding of the scale
    product and an O within the bf16 path's own distance from the oracle."""
    o2, lse2, _ = gpu_forward(_dequantised_twin(p8))
    if _kv8_path(p8, device=0)[0] != "kernel_split":
        assert np.array_equal(o, o2) and np.array_equal(lse, lse2)
    else:
        fin = np.isfinite(lse2)
        assert np.array_equal(np.isfinite(lse), fin)
        assert np.abs(lse[fin] - lse2[fin]).max() <= 1e-5 if fin.any() else True
        assert np.all(np.abs(o - o2) <= TOL_O_MAX * v_scale * np.maximum(1.0, np.abs(o2) / (2.0 * v_scale)))


CASES = [
    dict(seed=101, Hq=4, Hkv=2, D=64, max_ctx=700, max_q=96),
    dict(seed=102, Hq=8, Hkv=2, D=128, max_ctx=900, max_q=70),
    dict(seed=103, Hq=4, Hkv=4, D=128, max_ctx=600, max_q=140, n_req=4),          # G=1
    dict(seed=104, Hq=16, Hkv=2, D=64, max_ctx=500, max_q=40),                    # G=8
    dict(seed=106, Hq=6, Hkv=2, D=128, max_ctx=500, max_q=90),                    # G=3 (R=40)
    dict(seed=108, Hq=8, Hkv=2, D=128, max_ctx=600, max_q=100, hybrid=True, gaps=True),
    dict(seed=109, Hq=4, Hkv=2, D=128, max_ctx=300, max_q=8, n_req=12, max_segs=8),   # short queries
    dict(seed=110, Hq=4, Hkv=2, D=64, max_ctx=40, max_q=3, n_req=10, max_segs=4),     # tiny everything
    dict(seed=111, Hq=4, Hkv=2, D=128, max_ctx=500, max_q=64, q_to_kv=[1, 0, 0, 1]),   # custom GQA map
    dict(seed=112, Hq=8, Hkv=2, D=128, max_ctx=800, max_q=200, ragged=False),
]


@pytest.mark.gpu
@pytest.mark.parametrize("kw", CASES, ids=lambda k: f"seed{k['seed']}")
def test_kv8_random_small_problems_against_the_oracle_and_the_bf16_kernel(kw):
    p = W.random_problem(device=DEV, keep_dense=False, **kw)
    exps = [(-6, -4), (-5, -7), (-7, -5), (-4, -6)] if kw["seed"] != 112 else [(-14, 7), (7, -14)]     # 112: both ends of the range
    p8 = W.to_fp8_pool(p, k_exp=[exps[h % 4][0] for h in range(p.Hkv)], v_exp=[exps[h % 4][1] for h in range(p.Hkv)])
    o, lse, _ = gpu_forward(p8)
    compare(p8, o, lse, strict=False)
    _against_the_bf16_kernel(p8, o, lse)


@pytest.mark.gpu
@pytest.mark.parametrize("want", ["prepass", "kernel_pair", "kernel_split"])
def test_kv8_each_path_against_the_oracle_and_the_bf16_kernel(want):
    """The three ways an fp8 handle serves a batch (dequantising pre-pass + bf16 kernel; conversion in the kernel with two / one
    Q tiles) on the same context: each against the oracle, each bit-identical to the bf16 kernel on the dequantised pool."""
    p8 = W.to_fp8_pool(_three_paths(DEV)[want], k_exp=[-6, -4], v_exp=[-5, -7])
    assert _kv8_path(p8, device=0)[0] == want
    o, lse, _ = gpu_forward(p8)
    compare(p8, o, lse, strict=False)
    _against_the_bf16_kernel(p8, o, lse)


@pytest.mark.gpu
def test_kv8_cfg1_tiny_and_default_scales():
    p8 = W.to_fp8_pool(W.cfg1_tiny(device=DEV, keep_dense=False))
    o, lse, info = gpu_forward(p8)
    compare(p8, o, lse)
    assert info["visible_pairs"] == 14368


@pytest.mark.gpu
@pytest.mark.parametrize("seed", [201, 202])
def test_kv8_nan_codes_in_the_slack_never_reach_the_output(seed):
    """Block tails and unused blocks hold the NaN code 0x7f, arena gaps bf16 NaN."""
    p = W.random_problem(seed, Hq=8, Hkv=2, D=128, max_ctx=600, max_q=70, fill="nan", arena_gap=3, device=DEV)
    p8 = W.to_fp8_pool(p, k_exp=[-6, -5], v_exp=[-5, -6])
    assert (p8.pool_k == 0x7f).any()
    o, lse, _ = gpu_forward(p8)
    compare(p8, o, lse, strict=False)


@pytest.mark.gpu
def test_kv8_split_kv_and_one_token_segments():
    ctx = ContextSpec([(SEG_PAGED, 0, 3000), (SEG_CONTIG, 3000, 1777), (SEG_PAGED, 4777, 1500), (SEG_SELF, 6277, 40)])
    p = build_problem("split", 8, 2, 128, [ctx], [RunSpec(0, 6277, 40)], seed=8, device=DEV)
    p8 = W.to_fp8_pool(p)
    with MsaSession(p8) as s:
        assert s.info["num_split_items"] > 0
    o, lse, _ = gpu_forward(p8)
    compare(p8, o, lse)
    c0 = ContextSpec([(SEG_PAGED, 3, 1), (SEG_CONTIG, 4, 1), (SEG_PAGED, 9, 1)])
    c1 = ContextSpec([(SEG_PAGED, 0, 131), (SEG_CONTIG, 131, 1), (SEG_SELF, 132, 1)])
    p = build_problem("edge", 4, 2, 128, [c0, c1], [RunSpec(0, 0, 5), RunSpec(1, 132, 1)], seed=7, device=DEV, keep_dense=True,
                      fill="nan")
    p8 = W.to_fp8_pool(p, k_exp=[-6, -6], v_exp=[-6, -6])
    o, lse, _ = gpu_forward(p8)
    compare(p8, o, lse, strict=False)
    assert np.all(np.isneginf(lse[:3]))


def _gpu_forward_with_units(p):
    with MsaSession(p) as s:
        o, lse = s.forward()
        torch.cuda.synchronize()
        units = msa_plan_export(s.plan, 1)
        return o.float().cpu().numpy().astype(np.float64), lse.cpu().numpy().astype(np.float64), s.info, units


def _sample_with_plan_rows(p, units, reqs, n_random, seed, max_split=300):
    """Random and boundary rows of the runs `reqs`, the first / last row of each of their q-tile groups, and the first / last row
    of every split unit of the whole batch (the rows that go through the LSE-merge kernel), as test_msa_gpu samples them."""
    from test_msa_gpu import _plan_rows
    rr, ii = W.pick_rows(p, n_random, seed, reqs)
    rows = set(zip((int(x) for x in rr), (int(x) for x in ii)))
    grp, _ = _plan_rows(p, units, reqs, groups=True)
    spl, n_split = _plan_rows(p, units, None, groups=False)
    if len(spl) > max_split:
        pick = np.random.default_rng(seed).choice(len(spl), size=max_split, replace=False)
        spl = set(sorted(spl)[i] for i in pick)
    rows = sorted(rows | grp | spl)
    print(f"{p.name}: {len(grp)} q-tile-group edge rows, {len(spl)} split-unit edge rows ({n_split} split units in the plan)")
    return np.asarray([r for r, _ in rows], np.int32), np.asarray([i for _, i in rows], np.int32)


@pytest.mark.gpu
@pytest.mark.parametrize("k_exp,v_exp,k_mul,v_mul", [(-14, -14, 4.0, 1.0), (-10, -10, 4.0, 1.0), (7, 7, 1.0, 4096.0), (-14, 7, 4.0, 4096.0)])
def test_kv8_short_query_variant_at_the_ends_of_the_scale_range(k_exp, v_exp, k_mul, v_mul):
    """The f16 short-query variant with scales at both ends of the legal range and an arena that is not small next to them:
    arena K ~ 4 N(0,1) beside a pool whose largest K is 448 * 2^-14 = 0.027, arena and cached V ~ 4096 N(0,1) (|V| up to
    ~2^14) at the largest scale.  What the variant multiplies is code * 2^k and the arena value itself, both exact in f16,
    so the result may not depend on where a token's K / V lives or on the scale chosen."""
    ctxs, runs = [], []
    for r, (L, n) in enumerate([(700, 3), (1300, 8), (450, 1), (990, 5)]):
        ctxs.append(ContextSpec([(SEG_PAGED, 0, L - 260), (SEG_CONTIG, L - 260, 200), (SEG_PAGED, L - 60, 60), (SEG_SELF, L, n)]))
        runs.append(RunSpec(r, L, n))
    p = build_problem("scale_ends", 8, 2, 128, ctxs, runs, seed=41, device=DEV)
    p.contig_k = (p.contig_k.float() * k_mul).to(torch.bfloat16)
    p.contig_v = (p.contig_v.float() * v_mul).to(torch.bfloat16)
    p.pool_v = (p.pool_v.float() * v_mul).to(torch.bfloat16)
    p8 = W.to_fp8_pool(p, k_exp=[k_exp] * p.Hkv, v_exp=[v_exp] * p.Hkv)
    assert _kv8_path(p8, device=0)[0] == "kernel_split"
    if k_exp == -14:
        assert float(p8.contig_k.float().abs().max()) > 65504 * 2.0 ** k_exp       # beyond what arena / scale could hold in f16
    o, lse, _ = gpu_forward(p8)
    compare(p8, o, lse, strict=False, v_scale=v_mul)
    _against_the_bf16_kernel(p8, o, lse, v_scale=v_mul)


@pytest.mark.gpu
def test_kv8_handle_without_cached_segments_runs_the_bf16_kernel():
    """A plan with no PAGED segment has nothing to convert: an fp8 handle serves it with the plain kernel, bit for bit."""
    ctx = ContextSpec([(SEG_CONTIG, 0, 700), (SEG_SELF, 700, 90)])
    p = build_problem("no_paged", 8, 2, 128, [ctx, ctx], [RunSpec(0, 700, 90), RunSpec(1, 700, 3)], seed=42, device=DEV)
    o1, l1, _ = gpu_forward(p)
    p8 = W.to_fp8_pool(p, k_exp=[-6, -5], v_exp=[-5, -6])
    o2, l2, _ = gpu_forward(p8)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)
    compare(p8, o2, l2, strict=False)


@pytest.mark.gpu
def test_kv8_cfg5_short_query_every_row():
    """BASELINE.json configs[4] with the cached blocks in fp8 (the launch bench.py --workload cfg5_kv8 times)."""
    p8 = W.to_fp8_pool(W.cfg5_short_query(device=DEV))
    o, lse, info = gpu_forward(p8)
    mx, mean, dl = compare(p8, o, lse)
    print(f"cfg5_kv8: {p8.total_q} rows x {p8.Hq} heads compared, max|dO|={mx:.3e} mean|dO|={mean:.3e} max|dLSE|={dl:.3e}")


@pytest.mark.gpu
def test_kv8_cfg2_prefill_sampled_rows():
    p8 = W.to_fp8_pool(W.cfg2_llama8b(device=DEV))
    o, lse, info, units = _gpu_forward_with_units(p8)
    rr, ii = _sample_with_plan_rows(p8, units, reqs=[0, 3, 7], n_random=8, seed=3)
    mx, mean, dl = compare(p8, o, lse, rr, ii)
    print(f"cfg2_kv8: {len(rr)} rows x {p8.Hq} heads compared, max|dO|={mx:.3e} mean|dO|={mean:.3e} max|dLSE|={dl:.3e}")


@pytest.mark.gpu
@pytest.mark.parametrize("Hq,Hkv,D", [(8, 2, 128), (8, 4, 64)])
def test_kv8_append_quantises_like_the_oracle_and_feeds_the_forward(Hq, Hkv, D):
    """msa_kv_append on an fp8 handle: every destination byte equals the oracle quantiser's code (untouched blocks and block
    tails keep their canary), and a forward that reads the written blocks as PAGED segments matches the fp64 oracle."""
    p = W.random_problem(305, n_req=3, Hq=Hq, Hkv=Hkv, D=D, max_ctx=400, max_q=50, hybrid=True, device=DEV, keep_dense=False)
    p8 = W.to_fp8_pool(p, k_exp=[-6, -5, -7, -4][:Hkv], v_exp=[-5, -7, -4, -6][:Hkv])
    # a few extreme arena values: saturation, ties, tiny
    p8.contig_k = p8.contig_k.clone()
    p8.contig_k.view(-1)[:6] = torch.tensor([1000.0, -1000.0, 1.0625 * 2 ** -6, 2.0 ** -17, 0.0, -0.0], dtype=torch.bfloat16)
    bt = p8.block_table_np
    n_pool = int(p8.pool_k.shape[0])
    jobs, kind2, boff2, cursor = [], p8.seg_kind.copy(), p8.seg_block_off.copy(), len(bt)
    for s in range(len(p8.seg_kind)):
        if int(p8.seg_kind[s]) != SEG_PAGED:
            n = int(p8.seg_len[s])
            jobs.append((int(p8.seg_row_off[s]), n, cursor))
            kind2[s], boff2[s] = SEG_PAGED, cursor
            cursor += (n + 15) // 16
    extra = cursor - len(bt)
    bt2 = np.concatenate([bt, (n_pool + np.random.default_rng(5).permutation(extra)).astype(np.int32)])
    canary = 0x5a
    pool_k = torch.cat([p8.pool_k, torch.full((extra,) + tuple(p8.pool_k.shape[1:]), canary, dtype=torch.uint8, device=DEV)])
    pool_v = torch.cat([p8.pool_v, torch.full((extra,) + tuple(p8.pool_v.shape[1:]), canary, dtype=torch.uint8, device=DEV)])
    bt2_d = torch.from_numpy(bt2).to(DEV)
    h = msa_create(p8.Hq, p8.Hkv, p8.D, device=0, pool_format=MSA_POOL_FP8_E4M3, k_scale=p8.k_scale, v_scale=p8.v_scale)
    ap = msa_append_plan_create(h, jobs)
    msa_kv_append(h, ap, p8.contig_k, p8.contig_v, pool_k, pool_v, bt2_d, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    msa_append_plan_destroy(ap)
    msa_destroy(h)
    # expected bytes: the oracle's quantiser per KV head, placed by the oracle's write-back
    for pool, arena, scales in ((pool_k, p8.contig_k, p8.k_scale), (pool_v, p8.contig_v, p8.v_scale)):
        a = arena.float().cpu().double().numpy()
        codes = np.stack([quantize_e4m3(a[:, hh, :], float(scales[hh]), oracle.e4m3_to_double) for hh in range(p8.Hkv)], axis=1)
        start = np.concatenate([p8_pool.cpu().numpy() for p8_pool in (p8.pool_k if pool is pool_k else p8.pool_v,)] +
                               [np.full((extra,) + tuple(pool.shape[1:]), canary, np.uint8)])
        want = kv_append(start, codes, bt2, jobs)
        assert np.array_equal(pool.cpu().numpy(), want)
    # the forward reads what was written
    import copy
    p2 = copy.copy(p8)
    p2.pool_k, p2.pool_v, p2.block_table, p2.block_table_np = pool_k, pool_v, bt2_d, bt2
    p2.seg_kind, p2.seg_block_off, p2.num_blocks = kind2, boff2, n_pool + extra
    o, lse, _ = gpu_forward(p2)
    compare(p2, o, lse, strict=False)


@pytest.mark.gpu
@pytest.mark.parametrize("want", ["prepass", "kernel_pair", "kernel_split"])
def test_kv8_forward_writeback_is_forward_plus_quantising_append(want):
    """msa_forward_writeback on an fp8 handle: O / LSE bit-identical to msa_forward, and the pool afterwards holds, byte for
    byte, the oracle quantiser's codes of the arena rows where the oracle's write-back puts them (canary everywhere else)."""
    from paper_2606_02964_b200 import msa_forward_writeback, msa_last_launch_count, msa_plan_destroy, msa_workspace_bytes
    p8 = W.to_fp8_pool(_three_paths(DEV)[want], k_exp=[-6, -4], v_exp=[-5, -7])
    bt = p8.block_table_np
    n_pool, extra_rows = int(p8.pool_k.shape[0]), []
    jobs, cursor = [], len(bt)
    for s_ in range(len(p8.seg_kind)):
        if int(p8.seg_kind[s_]) != SEG_PAGED:
            n = int(p8.seg_len[s_])
            jobs.append((int(p8.seg_row_off[s_]), n, cursor))
            cursor += (n + 15) // 16
    extra = cursor - len(bt)
    bt2 = np.concatenate([bt, (n_pool + np.random.default_rng(6).permutation(extra)).astype(np.int32)])
    canary = 0x5a
    grow = lambda t: torch.cat([t, torch.full((extra,) + tuple(t.shape[1:]), canary, dtype=torch.uint8, device=DEV)])
    pool_k, pool_v = grow(p8.pool_k), grow(p8.pool_v)
    start_k, start_v = pool_k.cpu().numpy(), pool_v.cpu().numpy()
    bt2_d = torch.from_numpy(bt2).to(DEV)
    with MsaSession(p8) as s:
        o_ref, l_ref = s.forward()
        o_ref, l_ref, n_fwd = o_ref.clone(), l_ref.clone(), msa_last_launch_count(s.h)
        R, n_req, S, n_seg = make_descriptors(p8.req, p8.seg_kind, p8.seg_abs_start, p8.seg_len, p8.seg_block_off, p8.seg_row_off)
        plan = msa_plan_create_writeback(s.h, R, n_req, S, n_seg, jobs)
        nb = msa_workspace_bytes(plan)
        ws = torch.empty(max(nb, 16), dtype=torch.uint8, device=DEV)
        o, lse = torch.zeros_like(o_ref), torch.zeros_like(l_ref)
        msa_forward_writeback(s.h, plan, p8.q, pool_k, pool_v, bt2_d, p8.contig_k, p8.contig_v, p8.scale, o, lse, ws,
                              torch.cuda.current_stream().cuda_stream)
        assert msa_last_launch_count(s.h) == n_fwd + 1
        torch.cuda.synchronize()
        msa_plan_destroy(plan)
    assert torch.equal(o, o_ref) and torch.equal(lse, l_ref)
    for pool, start, arena, scales in ((pool_k, start_k, p8.contig_k, p8.k_scale), (pool_v, start_v, p8.contig_v, p8.v_scale)):
        a = arena.float().cpu().double().numpy()
        codes = np.stack([quantize_e4m3(a[:, hh, :], float(scales[hh]), oracle.e4m3_to_double) for hh in range(p8.Hkv)], axis=1)
        assert np.array_equal(pool.cpu().numpy(), kv_append(start, codes, bt2, jobs))


@pytest.mark.gpu
@pytest.mark.parametrize("want", ["prepass", "kernel_split"])
def test_kv8_host_buffer_call_equals_the_device_call(want):
    """msa_forward_host on an fp8 handle (the pool stays on the device; the pre-pass's copy lives in the handle's staging workspace)."""
    from paper_2606_02964_b200 import msa_forward_host
    p8 = W.to_fp8_pool(_three_paths(DEV)[want], k_exp=[-6, -4], v_exp=[-5, -7])
    with MsaSession(p8) as s:
        o_ref, l_ref = s.forward()
        torch.cuda.synchronize()
        qh, bt = p8.q.cpu().pin_memory(), p8.block_table.cpu().pin_memory()
        ck, cv = p8.contig_k.cpu().pin_memory(), p8.contig_v.cpu().pin_memory()
        oh, lh = torch.zeros_like(qh).pin_memory(), torch.zeros(p8.total_q, p8.Hq, dtype=torch.float32).pin_memory()
        msa_forward_host(s.h, s.plan, qh, p8.pool_k, p8.pool_v, bt, ck, cv, p8.scale, oh, lh, torch.cuda.current_stream().cuda_stream)
        assert torch.equal(oh, o_ref.cpu()) and torch.equal(lh, l_ref.cpu())


@pytest.mark.gpu
@pytest.mark.parametrize("name,want", [("cfg4_mixed", "prepass"), ("f1_hybrid_pod", "kernel_pair"), ("cfg3_70b_long", "prepass")])
def test_kv8_full_size_sampled_rows_on_the_other_paths(name, want):
    """The largest config through the dequantising pre-pass and the mixed prefill + decode batch through the two-Q-tile kernel
    variant (the launches `bench.py --workload <name>_kv8` times), on a row sample of a few runs."""
    base = {**W.CONFIGS, **W.EXTRA_CONFIGS}[name](device=DEV)
    p8 = W.to_fp8_pool(base)
    del base
    assert _kv8_path(p8, device=0)[0] == want
    o, lse, _, units = _gpu_forward_with_units(p8)
    reqs = list(range(0, p8.n_req, max(1, p8.n_req // 6)))[:6]
    if name == "cfg3_70b_long":          # G = 8, one request, 68 split items: rows aligned to the plan, as for the bf16 pool
        rr, ii = _sample_with_plan_rows(p8, units, reqs, n_random=12, seed=5, max_split=120)
    else:
        rr, ii = W.pick_rows(p8, n_random=6, seed=5, reqs=reqs)
    mx, mean, dl = compare(p8, o, lse, rr, ii)
    print(f"{name}_kv8 ({want}): {len(rr)} rows x {p8.Hq} heads compared, max|dO|={mx:.3e} mean|dO|={mean:.3e} max|dLSE|={dl:.3e}")

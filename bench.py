#!/usr/bin/env python
"""bench.py -- throughput of the MSA hot path on B200 (one JSON line on stdout).

A "step" is one pass of the whole hot path (plan reused; forward kernel + LSE-merge kernel)
over one synthetic batch.  Default workload = BASELINE.json configs[1] (Llama-3-8B-shaped
layer), metric = MSA attention TFLOP/s (algorithmic FLOPs = 4*D*Hq*visible pairs).
`--workload cfg5_short_query` reports the memory-bound metric (HBM GB/s) instead; at N=1
the default run appends it as `secondary`.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

N>1: launched by torchrun, one rank per GPU, every rank runs its own replica of the batch
(work units are independent: no data-path collective, "weak" scaling); time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402


def _env_int(name: str, default: int) -> int:
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def measured_peaks():
    """(tflops, gbs, label): driver-measured peaks, else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return float(d["bf16_tflops"]), float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json, burst bf16 / copy GB/s)"
    except Exception:
        return 1590.0, 6650.0, "fallback (B200_PROFILING.md)"


def sustained_tflops():
    """Seconds-long cuBLAS bf16 loop under the power cap (context for launches that run back to back for long)."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["bf16_tflops_sustained"])
    except Exception:
        return 1400.0


def committed_traffic(workload: str):
    """(dram bytes per launch of the dominant kernel, source) from the committed ncu capture, or (None, None).
    NOT measured by this run: profiles/roofline_traffic.csv holds dram__bytes_read.sum + dram__bytes_write.sum of one
    `ncu --set full` launch per workload (the .txt summary named in its `source` column)."""
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "roofline_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload:
                    return float(row["dram_bytes_per_launch"]), "profiles/%s (ncu --set full, one launch; not this run)" % row["source"]
    except Exception:
        pass
    return None, None


class ClockSampler:
    """Polls SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.hd = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.hd, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.hd, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.hd))
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join(timeout=1.0)
        med = int(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def oracle_sample(p, n_rows: int, seed: int, reqs=None):
    """Time the fp64 oracle, as it stands, on a bounded row sample.  Returns (seconds, flops, K/V bytes of the visible keys, rows)."""
    import oracle
    rng = np.random.default_rng(seed)
    if reqs is None:
        reqs = [int(rng.integers(0, p.n_req))]
    rr, ii = [], []
    per = max(1, n_rows // len(reqs))
    for r in reqs:
        T = int(p.req[r, 1])
        idx = np.sort(rng.choice(T, size=min(per, T), replace=False))
        rr += [r] * len(idx)
        ii += [int(x) for x in idx]
    rr, ii = np.asarray(rr, np.int32), np.asarray(ii, np.int32)
    arrays = p.host_arrays(reqs=reqs)
    pairs = 0
    kv_bytes = 0              # K and V bytes of the visible keys (all KV heads): one byte per cached element of an fp8 pool
    for r, i in zip(rr, ii):
        pos = int(p.req[r, 2]) + int(i)
        sb, sc = int(p.req[r, 3]), int(p.req[r, 4])
        for s in range(sb, sb + sc):
            vis = int(np.clip(pos - int(p.seg_abs_start[s]) + 1, 0, int(p.seg_len[s])))
            pairs += vis
            kv_bytes += vis * p.Hkv * p.D * 2 * (1 if (p.k_scale is not None and int(p.seg_kind[s]) == 0) else 2)
    t0 = time.perf_counter()
    oracle.forward(arrays, p.Hq, p.Hkv, p.D, p.scale, rr, ii)
    dt = time.perf_counter() - t0
    return dt, 4.0 * p.D * p.Hq * pairs, kv_bytes, len(rr)


def dist_max(value: float, device="cpu") -> float:
    """Max over ranks of a per-rank scalar (the timing rule: a multi-GPU number is the slowest rank's)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, units_per_step: float, ms: float) -> float:
    """Replicas only: every rank processes one full batch per step, no exchange on the path."""
    return world * units_per_step / (ms * 1e-3)


def all_workloads():
    """BASELINE.json's configs, the extra rows of SURVEY.md 8(f), and the batch whose residency the evictor decides."""
    import workloads as W
    from workloads.policy_trace import f3_policy_trace
    out = {**W.CONFIGS, **W.EXTRA_CONFIGS, "f3_policy_trace": f3_policy_trace}
    # the same batches with the paged pool stored as fp8 E4M3 codes: `<name>_kv8`
    for base in ("cfg2_llama8b", "cfg3_70b_long", "cfg4_mixed", "cfg5_short_query", "f1_hybrid_pod"):
        out[base + "_kv8"] = (lambda b: (lambda device="cpu", **kw: W.to_fp8_pool(out[b](device=device, **kw))))(base)
    return out


def metric_of(workload: str):
    if workload in ("cfg5_short_query", "cfg5_short_query_kv8"):
        return "msa_short_query_hbm_gbs", "GB/s", "hbm"
    return "msa_attention_tflops", "TFLOP/s", "tensor"


def run_mine(args, rank: int, world: int, local_rank: int):
    import torch
    import workloads as W
    from paper_2606_02964_b200 import (MsaSession, msa_forward_host, msa_forward_host_async, msa_forward_host_wait, msa_get_timing,
                                       msa_last_launch_count, msa_set_timing)
    import __graft_entry__ as ge
    if rank == 0:
        ge.build()
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    tfl_peak, gbs_peak, peak_label = measured_peaks()

    def bench_workload(name: str, steps: int, warmup: int, do_e2e: bool):
        metric, unit, bound = metric_of(name)
        p = all_workloads()[name](device=dev)
        alg = p.algorithmic()
        units_per_step = alg["flops"] / 1e12 if bound == "tensor" else alg["bytes"] / 1e9
        s = MsaSession(p, device=local_rank)
        stream = torch.cuda.current_stream().cuda_stream
        for _ in range(max(3, warmup)):
            s.forward(stream)
        torch.cuda.synchronize()
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        sampler = ClockSampler(local_rank)
        msa_set_timing(s.h, steps)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        sampler.start()
        e0.record()
        launches = 0
        for _ in range(steps):
            s.forward(stream)
            launches += msa_last_launch_count(s.h)
        e1.record()
        torch.cuda.synchronize()
        clocks = sampler.stop()
        ms = e0.elapsed_time(e1) / steps
        n_rec, fwd_ms, merge_ms = msa_get_timing(s.h)
        msa_set_timing(s.h, 0)
        if world > 1:
            ms = dist_max(ms, dev)
        value = whole_job_value(world, units_per_step, ms)
        kern_units = units_per_step          # the forward kernel does all algorithmic work of a step
        achieved = kern_units / (fwd_ms * 1e-3) if fwd_ms > 0 else None
        peak = tfl_peak if bound == "tensor" else gbs_peak
        traffic, traffic_source = committed_traffic(name)
        out = dict(metric=metric, value=value, unit=unit, ms_per_step=ms, gpu_launches=launches,
                   roofline=dict(bound=bound, achieved=achieved, peak=peak, unit=unit,
                                 frac=(achieved / peak) if achieved else None, traffic=traffic, traffic_source=traffic_source,
                                 algorithmic_units_per_launch=units_per_step,
                                 kernel="msa_fwd", kernel_ms=fwd_ms, merge_ms=merge_ms, steps_timed=n_rec,
                                 peak_source=peak_label,
                                 frac_of_nominal=(achieved / (2250.0 if bound == "tensor" else 8000.0)) if achieved else None,
                                 frac_of_sustained=(achieved / sustained_tflops()) if (achieved and bound == "tensor") else None),
                   clocks=clocks, plan=s.info, algorithmic=alg)
        if do_e2e:
            # End to end through the host-buffer entry of the C ABI, two steps in flight (msa_forward_host_async, two slots): step
            # i + 1 uploads while step i computes and reads back.  Every step copies its inputs from pinned host memory and lands its
            # O / LSE in host buffers of its own slot; a step counts as done when its results have landed (msa_forward_host_wait).
            qh = p.q.cpu().pin_memory()
            ck, cv = p.contig_k.cpu().pin_memory(), p.contig_v.cpu().pin_memory()
            bt = p.block_table.cpu().pin_memory()
            oh = [torch.empty_like(qh).pin_memory() for _ in range(2)]
            lh = [torch.empty(p.total_q, p.Hq, dtype=torch.float32).pin_memory() for _ in range(2)]
            k_e2e = max(3, min(steps, 20))

            def run_steps(n):
                for i in range(n):
                    msa_forward_host_async(s.h, s.plan, qh, p.pool_k, p.pool_v, bt, ck, cv, p.scale, oh[i & 1], lh[i & 1], stream, i & 1)
                    if i > 0:
                        msa_forward_host_wait(s.h, (i - 1) & 1)
                msa_forward_host_wait(s.h, (n - 1) & 1)

            run_steps(3)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            e0.record()
            run_steps(k_e2e)
            e1.record()
            torch.cuda.synchronize()
            wall_ms = (time.perf_counter() - t0) * 1e3 / k_e2e
            ems = max(e0.elapsed_time(e1) / k_e2e, wall_ms)      # results land on the handle's own streams: the host clock sees them all
            # one step alone, start to finish (the latency a single call sees)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(3):
                msa_forward_host(s.h, s.plan, qh, p.pool_k, p.pool_v, bt, ck, cv, p.scale, oh[0], lh[0], stream)
            single_ms = (time.perf_counter() - t0) * 1e3 / 3
            if world > 1:
                ems = dist_max(ems, dev)
            h2d = qh.numel() * 2 + ck.numel() * 2 + cv.numel() * 2 + bt.numel() * 4
            d2h = oh[0].numel() * 2 + lh[0].numel() * 4
            out["e2e"] = dict(value=whole_job_value(world, units_per_step, ems), unit=unit, ms_per_step=ems, steps=k_e2e,
                              h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h), single_call_ms=single_ms,
                              note="msa_forward_host_async / _wait, two steps in flight: q, block table, contiguous arena from pinned "
                                   "host memory; O and LSE back to host; the paged pool is the resident KV cache; "
                                   "single_call_ms = one msa_forward_host call start to finish.  The upload of the arena "
                                   "(recomputed runs + own chunk) is part of this definition and it is what the number measures: "
                                   "PCIe at ~52 GB/s, not the kernel's rate (`value`); in the serving step of the paper the arena is "
                                   "produced on the device by the QKV projection (PAPER.md:116-122)")
        s.close()
        return out, p

    res, p = bench_workload(args.workload, args.steps, args.warmup, do_e2e=True)
    line = dict(metric=res["metric"], value=res["value"], unit=res["unit"], n_gpus=world, steps=args.steps,
                warmup=max(3, args.warmup), ms_per_step=res["ms_per_step"], higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="bf16", data="synthetic",
                config=dict(workload=args.workload, Hq=p.Hq, Hkv=p.Hkv, head_dim=p.D, requests=p.n_req,
                            total_q=p.total_q, kv_tokens=p.kv_tokens(), block_size=16,
                            pool_format="fp8_e4m3 (power-of-two scale per KV head)" if p.k_scale is not None else "bf16",
                            l2_policy="inputs larger than L2 (%.0f MB per step), no flush" % (res["algorithmic"]["bytes"] / 1e6),
                            parallelism=f"replicas x{world}" if world > 1 else "single GPU"),
                clocks=res["clocks"], e2e=res.get("e2e"), gpu_launches=res["gpu_launches"],
                roofline=res["roofline"], plan=res["plan"])
    if rank == 0 and world == 1:
        # the oracle, as it stands, on a bounded sample of the same workload (reported baseline)
        import oracle
        reqs = list(range(min(2, p.n_req)))
        dt, fl, pairs, n = oracle_sample(p, 8, 1, reqs)                     # calibrate
        rows = int(np.clip(15.0 / max(dt / n, 1e-6), 16, 4096))
        dt, fl, pairs, n = oracle_sample(p, rows, 2, reqs)
        unit = res["unit"]
        if unit == "TFLOP/s":
            cv = fl / dt / 1e12
        else:
            cv = pairs / dt / 1e9                            # K and V bytes of the visible keys
        line["cpu_baseline"] = dict(value=cv, unit=unit, cores=oracle.num_threads(), kind="oracle",
                                    sample=f"{n} query rows of requests {reqs} (all {p.Hq} heads), {dt:.2f} s",
                                    seconds=dt)
        if args.workload == "cfg2_llama8b" and not args.no_secondary:
            # the other three performance configs of BASELINE.json, each with its own roofline block and clocks
            del p
            line["secondary"] = []
            # ... and configs[4] again with the cached blocks stored as fp8 E4M3 codes (GB/s on the fp8 bytes)
            # Compact entries, `secondary` the LAST key of the line and the short-query config (the other half of BASELINE.json's
            # metric) last inside it: a record that keeps only the tail of the line still holds every headline number.
            def r5(x):
                return None if x is None else float(f"{x:.5g}")

            for wl, k in (("cfg3_70b_long", 30), ("cfg4_mixed", 20), ("f1_hybrid_pod", 30), ("cfg5_short_query_kv8", 30),
                          ("cfg5_short_query", 50)):
                torch.cuda.empty_cache()
                time.sleep(2.0)            # each workload starts from an idle chip, not from the last one's power state
                sec, psec = bench_workload(wl, max(10, min(args.steps, k)), args.warmup, do_e2e=False)
                rf = sec["roofline"]
                line["secondary"].append(dict(workload=wl, value=r5(sec["value"]), unit=sec["unit"], ms_per_step=r5(sec["ms_per_step"]),
                                              kernel_ms=r5(rf["kernel_ms"]), merge_ms=r5(rf["merge_ms"]), bound=rf["bound"],
                                              achieved=r5(rf["achieved"]), peak=r5(rf["peak"]), frac=r5(rf["frac"]),
                                              frac_of_nominal=r5(rf["frac_of_nominal"]), traffic=rf["traffic"],
                                              gpu_launches=sec["gpu_launches"], sm_mhz=sec["clocks"].get("sm_mhz"),
                                              reasons=sec["clocks"].get("reasons")))
                del psec
            line["config"]["largest_single_gpu_config"] = "cfg4_mixed (in `secondary`; `value` is quoted on cfg2_llama8b = BASELINE.json configs[1])"
            line["secondary"] = line.pop("secondary")          # last key of the line
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line))


class Fig13Case:
    """One request of the Fig. 13 shape (workloads.f2_fig13) with the plans of every way to compute it.

    fused()            one msa_forward over all runs and segments (what MSA is)
    per_run()          'two kernel calls' of PAPER.md:353: one msa_forward per compute run, a host synchronisation after each
    per_kv_segment()   the same kernel once per KV segment of the LAST run, a host synchronisation after each call, and an
                       LSE merge of the partial results with torch ops (exact: softmax over a union = LSE-weighted mix)
    The per-* paths are baselines that exist only here (bench + tests); the product path is the fused call."""

    def __init__(self, cached_tokens: int, layout: str, device="cuda:0", keep_dense: bool = False):
        import torch
        import workloads as W
        from paper_2606_02964_b200 import make_descriptors, msa_create, msa_plan_create, msa_workspace_bytes
        self.torch = torch
        self.p = p = W.f2_fig13(cached_tokens, layout, device=device, keep_dense=keep_dense)
        self.dev = device
        self.h = msa_create(p.Hq, p.Hkv, p.D, p.q_to_kv, device=torch.device(device).index or 0)
        self.plans = {}

        def plan_of(run_ids, seg_lo, seg_hi):
            req = p.req[run_ids].copy()
            req[:, 3] = 0
            req[:, 4] = seg_hi - seg_lo
            R, n, S, m = make_descriptors(req, p.seg_kind[seg_lo:seg_hi], p.seg_abs_start[seg_lo:seg_hi], p.seg_len[seg_lo:seg_hi],
                                          p.seg_block_off[seg_lo:seg_hi], p.seg_row_off[seg_lo:seg_hi])
            pl = msa_plan_create(self.h, R, n, S, m)
            nb = msa_workspace_bytes(pl)
            ws = torch.empty(max(nb, 16), dtype=torch.uint8, device=device) if nb else None
            return pl, ws

        nseg, nrun = p.n_seg, p.n_req
        self.plans["fused"] = plan_of(list(range(nrun)), 0, nseg)
        # per run: run r sees the segments up to and including its own SELF segment
        self.run_plans = []
        for r in range(nrun):
            last = max(s for s in range(nseg) if int(p.seg_abs_start[s]) <= int(p.req[r, 2]))
            self.run_plans.append(plan_of([r], 0, last + 1))
        # per KV segment, last run only
        self.seg_plans = [plan_of([nrun - 1], s, s + 1) for s in range(nseg)]
        self.o = torch.zeros_like(p.q)
        self.lse = torch.zeros(p.total_q, p.Hq, dtype=torch.float32, device=device)
        self.o_part = [torch.zeros_like(p.q) for _ in range(nseg)]
        self.lse_part = [torch.full((p.total_q, p.Hq), float("-inf"), dtype=torch.float32, device=device) for _ in range(nseg)]

    def _fwd(self, plan, o, lse, stream):
        from paper_2606_02964_b200 import msa_forward
        p = self.p
        msa_forward(self.h, plan[0], p.q, p.pool_k, p.pool_v, p.block_table, p.contig_k, p.contig_v, p.scale, o, lse, plan[1], stream)

    def fused(self, stream, sync=True):
        self._fwd(self.plans["fused"], self.o, self.lse, stream)
        if sync:
            self.torch.cuda.synchronize()
        return self.o, self.lse

    def per_run(self, stream, sync=True):
        for pl in self.run_plans:
            self._fwd(pl, self.o, self.lse, stream)
            if sync:
                self.torch.cuda.synchronize()
        return self.o, self.lse

    def per_kv_segment(self, stream, sync=True):
        torch = self.torch
        p = self.p
        r0, n = int(p.req[-1, 0]), int(p.req[-1, 1])
        for s, pl in enumerate(self.seg_plans):
            self._fwd(pl, self.o_part[s], self.lse_part[s], stream)
            if sync:
                torch.cuda.synchronize()
        L = torch.stack([x[r0:r0 + n] for x in self.lse_part])                  # [S, n, Hq]
        lse = torch.logsumexp(L, dim=0)
        w = torch.exp(L - lse.unsqueeze(0))
        w = torch.where(torch.isfinite(L), w, torch.zeros_like(w))
        O = torch.stack([x[r0:r0 + n].float() for x in self.o_part])            # [S, n, Hq, D]
        o = (w.unsqueeze(-1) * O).sum(0).to(torch.bfloat16)
        if sync:
            torch.cuda.synchronize()
        return o, lse, (r0, n)

    def close(self):
        from paper_2606_02964_b200 import msa_destroy, msa_plan_destroy
        for pl, _ in [self.plans["fused"]] + self.run_plans + self.seg_plans:
            msa_plan_destroy(pl)
        msa_destroy(self.h)


def run_fig13(args):
    """SURVEY.md section 8 (f2), the shape of the paper's Fig. 13, Llama-3-8B heads, one request that
    "ends with 128 new tokens".  Three ways to serve it (the paper's three lines):
      prefix     caching from the prefix   [cached N][recompute R + new 128]              one call
      suffix x2  caching from the suffix   [recompute R][cached N][new 128]               one call per compute run ("two kernel calls")
      suffix MSA caching from the suffix, same layout                                      ONE fused msa_forward
    plus the round-1 row [cached N][new 128]: fused against one call per KV segment + LSE merge.  R = N (DESIGN.md c18).
    Every variant is timed twice: host wall clock per attention call including the synchronisation(s) a caller needs, and
    device time (CUDA events around `steps` back-to-back calls without host synchronisation)."""
    import torch
    import __graft_entry__ as ge
    ge.build()
    dev = "cuda:0"
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream().cuda_stream
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timed(fn):
        for _ in range(max(3, args.warmup)):
            fn(stream)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            fn(stream)
        wall = (time.perf_counter() - t0) / args.steps * 1e6
        torch.cuda.synchronize()
        e0.record()
        for _ in range(args.steps):
            fn(stream, sync=False)
        e1.record()
        torch.cuda.synchronize()
        return wall, e0.elapsed_time(e1) / args.steps * 1e3

    rows = []
    for N in (1024, 2048, 4096, 8192, 10240):
        row = dict(cached_tokens=N, recompute_tokens=N, new_tokens=128)
        c = Fig13Case(N, "prefix", dev)
        row["prefix_wall_us"], row["prefix_dev_us"] = timed(c.fused)
        c.close()
        c = Fig13Case(N, "suffix", dev)
        row["suffix_msa_wall_us"], row["suffix_msa_dev_us"] = timed(c.fused)
        o1, l1 = (x.clone() for x in c.fused(stream))
        row["suffix_two_calls_wall_us"], row["suffix_two_calls_dev_us"] = timed(c.per_run)
        o2, l2 = c.per_run(stream)
        row["two_calls_max_abs_dO"] = float((o1.float() - o2.float()).abs().max())
        row["two_calls_max_abs_dLSE"] = float((l1 - l2).abs().max())
        c.close()
        c = Fig13Case(N, "prefix_new", dev)
        row["new128_fused_wall_us"], row["new128_fused_dev_us"] = timed(c.fused)
        o1, l1 = (x.clone() for x in c.fused(stream))
        row["new128_per_segment_wall_us"], row["new128_per_segment_dev_us"] = timed(c.per_kv_segment)
        o2, l2, (r0, n) = c.per_kv_segment(stream)
        row["per_segment_max_abs_dO"] = float((o1[r0:r0 + n].float() - o2.float()).abs().max())
        row["per_segment_max_abs_dLSE"] = float((l1[r0:r0 + n] - l2).abs().max())
        c.close()
        row["two_calls_overhead_us"] = row["suffix_two_calls_wall_us"] - row["suffix_msa_wall_us"]
        row["suffix_vs_prefix"] = row["suffix_msa_wall_us"] / row["prefix_wall_us"]
        rows.append(row)
    mean_overhead = float(np.mean([r["two_calls_overhead_us"] for r in rows]))
    print(json.dumps(dict(metric="msa_two_call_overhead_us_per_attention_call", value=mean_overhead, unit="us", n_gpus=1, steps=args.steps,
                          warmup=max(3, args.warmup), higher_is_better=False, dtype="bf16", data="synthetic", vs_baseline=None,
                          config=dict(workload="fig13", Hq=32, Hkv=8, head_dim=128, new_tokens=128,
                                      timing="wall = host clock per call incl. the synchronisation(s) a caller needs; dev = CUDA events, no host sync"),
                          fig13=rows, gpu_launches=args.steps * 2 * 7)))


def run_evictor(args):
    """control-plane cost of one eviction (+ the re-insertion that follows) with the O(log n)
    evictor (Algorithm 1) against the O(n) scan the paper compares with, at 8 K and 100 K cached blocks."""
    import __graft_entry__ as ge
    ge.build()
    from paper_2606_02964_b200 import MsaEvictor
    rng = np.random.default_rng(7)
    rows = []
    for n in (8192, 100_000):
        for linear in (False, True):
            ev = MsaEvictor(alpha=600.0, beta=15.0, tau0=540.0, k5=2.5e-9, c0=3.0e-5)
            pos = rng.integers(0, 32768, size=n) * 16
            last = rng.uniform(0.0, 3000.0, size=n)
            for b in range(n):
                ev.add(b, int(pos[b]), float(last[b]))
            ops = 20000 if not linear else (2000 if n <= 8192 else 300)
            t, nid = 3000.0, n
            t0 = time.perf_counter()
            for i in range(ops):
                t += 0.05
                ev.evict(t, linear=linear)
                ev.add(nid, int(pos[i % n]), t)          # the freed block is reused and becomes evictable again
                nid += 1
            dt = time.perf_counter() - t0
            rows.append(dict(blocks=n, strategy="linear scan" if linear else "two ordered sets (Algorithm 1)",
                             us_per_evict_plus_add=dt / ops * 1e6, ops=ops))
            ev.close()
    fast = {r["blocks"]: r["us_per_evict_plus_add"] for r in rows if r["strategy"].startswith("two")}
    slow = {r["blocks"]: r["us_per_evict_plus_add"] for r in rows if r["strategy"].startswith("linear")}
    print(json.dumps(dict(metric="msa_evictor_us_per_eviction", value=fast[100_000], unit="us", n_gpus=0, steps=1, warmup=0,
                          higher_is_better=False, dtype="f64", data="synthetic", vs_baseline=None,
                          config=dict(workload="evictor", note="host only; includes the ctypes call overhead of both strategies alike"),
                          evictor=rows, speedup_8k=slow[8192] / fast[8192], speedup_100k=slow[100_000] / fast[100_000],
                          gpu_launches=0)))


def run_costmodel(args):
    """refit the attention part of the paper's latency model from measured msa_forward times.
    Layout of Eq. (4): [cached l1][compute q1][cached l2][compute q2], one request, Llama-3-8B heads.
    Eq. (4): T = k1 l1 + k2 q1 + k3 l2 + k4 q2 + k5 q1 (l1+q1) + k6 q2 (l1+q1+l2+q2) + b;  Eq. (6) replaces the k5 term by
    k5 (l1+q1)^2 so that dT_B = 2 k5 pos + const (Eq. (7)).  Least squares over the grid, R^2 of both forms."""
    import torch
    import workloads as W
    from paper_2606_02964_b200 import MsaSession, msa_get_timing, msa_set_timing
    import __graft_entry__ as ge
    ge.build()
    dev = "cuda:0"
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream().cuda_stream
    grid = [(l1, q1, l2, q2) for l1 in (1024, 4096, 8192, 16384) for q1 in (256, 1024, 2048)
            for l2 in (1024, 4096, 8192) for q2 in (256, 1024, 2048)]
    X4, X6, y = [], [], []
    for (l1, q1, l2, q2) in grid:
        ctx = W.ContextSpec([(W.SEG_PAGED, 0, l1), (W.SEG_SELF, l1, q1), (W.SEG_PAGED, l1 + q1, l2), (W.SEG_SELF, l1 + q1 + l2, q2)])
        p = W.build_problem("costmodel", 32, 8, 128, [ctx], [W.RunSpec(0, l1, q1), W.RunSpec(0, l1 + q1 + l2, q2)],
                            seed=77, device=dev)
        with MsaSession(p) as sess:
            for _ in range(3):
                sess.forward(stream)
            msa_set_timing(sess.h, 10)
            for _ in range(10):
                sess.forward(stream)
            torch.cuda.synchronize()
            _, fwd_ms, merge_ms = msa_get_timing(sess.h)
        lin = [l1, q1, l2, q2]
        X4.append(lin + [q1 * (l1 + q1), q2 * (l1 + q1 + l2 + q2), 1.0])
        X6.append(lin + [(l1 + q1) ** 2, q2 * (l1 + q1 + l2 + q2), 1.0])
        y.append((fwd_ms + merge_ms) * 1e-3)
        del p
    y = np.asarray(y)

    def fit(X):
        X = np.asarray(X, np.float64)
        k, *_ = np.linalg.lstsq(X, y, rcond=None)
        r = y - X @ k
        return k, 1.0 - float(r @ r) / float(((y - y.mean()) ** 2).sum())

    k4, r2_4 = fit(X4)
    k6, r2_6 = fit(X6)
    names = ["k1", "k2", "k3", "k4", "k5", "k6", "beta"]
    print(json.dumps(dict(metric="msa_costmodel_r2_eq4", value=r2_4, unit="R^2", n_gpus=1, steps=10, warmup=3, higher_is_better=True,
                          dtype="bf16", data="synthetic", vs_baseline=None,
                          config=dict(workload="costmodel", points=len(grid), seconds_min=float(y.min()), seconds_max=float(y.max())),
                          eq4=dict(r2=r2_4, coeff=dict(zip(names, map(float, k4)))),
                          eq6=dict(r2=r2_6, coeff=dict(zip(names, map(float, k6))),
                                   evictor_k5=float(k6[4]), evictor_c0=float(k6[1] - k6[2] + k6[4])),
                          gpu_launches=len(grid) * 26)))


def run_kv_append(args):
    """write the recomputed and own K/V of the cfg2 batch (every CONTIG / SELF segment) into
    fresh paged blocks.  HBM-bound copy: algorithmic bytes = 2 (read + write) x tokens x Hkv x D x 2 B x 2 (K, V)."""
    import torch
    import workloads as W
    from paper_2606_02964_b200 import msa_append_plan_create, msa_append_plan_destroy, msa_create, msa_destroy, msa_kv_append
    import __graft_entry__ as ge
    ge.build()
    dev = "cuda:0"
    torch.cuda.set_device(0)
    _, gbs_peak, peak_label = measured_peaks()
    p = W.cfg2_llama8b(device=dev)
    jobs, cursor, tokens = [], int(p.block_table.numel()), 0
    for sidx in range(len(p.seg_kind)):
        if int(p.seg_kind[sidx]) != W.SEG_PAGED:
            n = int(p.seg_len[sidx])
            jobs.append((int(p.seg_row_off[sidx]), n, cursor))
            cursor += (n + 15) // 16
            tokens += n
    extra = cursor - int(p.block_table.numel())
    n_pool = int(p.pool_k.shape[0])
    perm = torch.randperm(extra, generator=torch.Generator().manual_seed(9)).to(torch.int32) + n_pool
    bt = torch.cat([p.block_table, perm.to(dev)]).contiguous()
    pool_k = torch.cat([p.pool_k, torch.zeros((extra,) + tuple(p.pool_k.shape[1:]), dtype=torch.bfloat16, device=dev)]).contiguous()
    pool_v = torch.cat([p.pool_v, torch.zeros((extra,) + tuple(p.pool_v.shape[1:]), dtype=torch.bfloat16, device=dev)]).contiguous()
    h = msa_create(p.Hq, p.Hkv, p.D, p.q_to_kv, device=0)
    ap = msa_append_plan_create(h, jobs)
    stream = torch.cuda.current_stream().cuda_stream
    for _ in range(max(3, args.warmup)):
        msa_kv_append(h, ap, p.contig_k, p.contig_v, pool_k, pool_v, bt, stream)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    e0.record()
    for _ in range(args.steps):
        msa_kv_append(h, ap, p.contig_k, p.contig_v, pool_k, pool_v, bt, stream)
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1) / args.steps
    nbytes = 2.0 * tokens * p.Hkv * p.D * 2 * 2
    gbs = nbytes / (ms * 1e-3) / 1e9
    # the same write-back fused into the forward launch (msa_forward_writeback) against forward + msa_kv_append
    from paper_2606_02964_b200 import (make_descriptors, msa_forward, msa_forward_writeback, msa_plan_create_writeback,
                                       msa_plan_destroy, msa_workspace_bytes)
    R, n, S, m = make_descriptors(p.req, p.seg_kind, p.seg_abs_start, p.seg_len, p.seg_block_off, p.seg_row_off)
    plan = msa_plan_create_writeback(h, R, n, S, m, jobs)
    nb = msa_workspace_bytes(plan)
    ws = torch.empty(max(nb, 16), dtype=torch.uint8, device=dev) if nb else None
    o = torch.zeros_like(p.q)
    lse = torch.zeros(p.total_q, p.Hq, dtype=torch.float32, device=dev)

    def timed(fn):
        for _ in range(max(3, args.warmup)):
            fn()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(args.steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps

    fwd_only = timed(lambda: msa_forward(h, plan, p.q, pool_k, pool_v, bt, p.contig_k, p.contig_v, p.scale, o, lse, ws, stream))
    two = timed(lambda: (msa_forward(h, plan, p.q, pool_k, pool_v, bt, p.contig_k, p.contig_v, p.scale, o, lse, ws, stream),
                         msa_kv_append(h, ap, p.contig_k, p.contig_v, pool_k, pool_v, bt, stream)))
    fused = timed(lambda: msa_forward_writeback(h, plan, p.q, pool_k, pool_v, bt, p.contig_k, p.contig_v, p.scale, o, lse, ws, stream))
    msa_plan_destroy(plan)
    msa_append_plan_destroy(ap)
    msa_destroy(h)
    # the same jobs into an fp8 (E4M3) pool: the rows are quantised on the way (2 bytes read, 1 written per element)
    from paper_2606_02964_b200 import MSA_POOL_FP8_E4M3
    scales = np.full(p.Hkv, 2.0 ** -6, np.float32)
    h8 = msa_create(p.Hq, p.Hkv, p.D, p.q_to_kv, device=0, pool_format=MSA_POOL_FP8_E4M3, k_scale=scales, v_scale=scales)
    ap8 = msa_append_plan_create(h8, jobs)
    pk8 = torch.zeros(tuple(pool_k.shape), dtype=torch.uint8, device=dev)
    pv8 = torch.zeros(tuple(pool_v.shape), dtype=torch.uint8, device=dev)
    ms8 = timed(lambda: msa_kv_append(h8, ap8, p.contig_k, p.contig_v, pk8, pv8, bt, stream))
    nbytes8 = 1.5 * tokens * p.Hkv * p.D * 2 * 2
    msa_append_plan_destroy(ap8)
    msa_destroy(h8)
    print(json.dumps(dict(metric="msa_kv_append_hbm_gbs", value=gbs, unit="GB/s", n_gpus=1, steps=args.steps, warmup=max(3, args.warmup),
                          ms_per_step=ms, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="bf16", data="synthetic",
                          config=dict(workload="kv_append", tokens=tokens, jobs=len(jobs), bytes_per_step=nbytes,
                                      l2_policy="working set %.0f MB per step (read + write), larger than L2" % (nbytes / 1e6)),
                          fp8_pool=dict(ms_per_step=ms8, bytes_per_step=nbytes8, gbs=nbytes8 / (ms8 * 1e-3) / 1e9,
                                        frac=nbytes8 / (ms8 * 1e-3) / 1e9 / gbs_peak, kernel="msa_kv_append_q8_kernel"),
                          clocks=clocks, gpu_launches=args.steps,
                          fused=dict(forward_only_ms=fwd_only, forward_plus_kv_append_ms=two, forward_writeback_ms=fused,
                                     writeback_cost_ms=fused - fwd_only, separate_cost_ms=two - fwd_only,
                                     note="cfg2 batch: msa_forward_writeback stores the recomputed + own K/V from the forward "
                                          "kernel's shared-memory tiles (no second read of the arena, no second launch)"),
                          roofline=dict(bound="hbm", achieved=gbs, peak=gbs_peak, unit="GB/s", frac=gbs / gbs_peak, traffic=None,
                                        kernel="msa_kv_append", kernel_ms=ms, peak_source=peak_label))))


def run_reference(args, rank: int, world: int):
    """The reference arm of this tier = the fp64 CPU oracle on the box's host cores (rank 0 only)."""
    if rank != 0:
        return
    import oracle
    import workloads as W
    oracle.build()                      # the C oracle only: this arm never maps libmsa.so
    metric, unit, bound = metric_of(args.workload)
    p = W.CONFIGS[args.workload](device="cpu") if args.workload in ("cfg1_tiny",) else None
    if p is None:
        # values on the CPU; only the requests sampled are ever read
        small = dict(cfg2_llama8b=dict(n_req=2), cfg4_mixed=dict(n_req=4), cfg5_short_query=dict(n_req=8),
                     f1_hybrid_pod=dict(n_prefill=1, n_decode=2))
        if args.workload == "f3_policy_trace":
            raise SystemExit("the oracle arm covers BASELINE.json's configs and f1 (f3's residency is decided by the product's evictor)")
        base = args.workload[:-4] if args.workload.endswith("_kv8") else args.workload
        p = {**W.CONFIGS, **W.EXTRA_CONFIGS}[base](device="cpu", **small.get(base, {}))
        if base != args.workload:
            p = W.to_fp8_pool(p)
    reqs = list(range(min(2, p.n_req)))
    dt, fl, pairs, n = oracle_sample(p, 8, 1, reqs)
    total = max(1, args.steps + args.warmup)
    rows = int(np.clip((90.0 / total) / max(dt / n, 1e-6), 4, 2048))
    for _ in range(args.warmup):
        oracle_sample(p, rows, 3, reqs)
    t_sum, f_sum, p_sum, n_sum = 0.0, 0.0, 0, 0
    for k in range(args.steps):
        dt, fl, pairs, n = oracle_sample(p, rows, 10 + k, reqs)
        t_sum, f_sum, p_sum, n_sum = t_sum + dt, f_sum + fl, p_sum + pairs, n_sum + n
    if bound == "tensor":
        value = f_sum / t_sum / 1e12
    else:
        value = p_sum / t_sum / 1e9                            # K and V bytes of the visible keys
    sample = f"{n_sum // max(1, args.steps)} query rows per step of requests {reqs} (all {p.Hq} heads)"
    line = dict(impl="reference", metric=metric, value=value, unit=unit, n_gpus=world, steps=args.steps,
                warmup=args.warmup, ms_per_step=1e3 * t_sum / max(1, args.steps), higher_is_better=True,
                scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=args.workload, Hq=p.Hq, Hkv=p.Hkv, head_dim=p.D, sample=sample),
                cpu_baseline=dict(value=value, unit=unit, cores=oracle.num_threads(), kind="oracle", sample=sample),
                e2e=dict(value=value, unit=unit, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="mine", choices=["mine", "reference"])
    ap.add_argument("--workload", default="cfg2_llama8b",
                    choices=["cfg2_llama8b", "cfg3_70b_long", "cfg4_mixed", "cfg5_short_query", "f1_hybrid_pod", "f3_policy_trace",
                             "cfg2_llama8b_kv8", "cfg3_70b_long_kv8", "cfg4_mixed_kv8", "cfg5_short_query_kv8", "f1_hybrid_pod_kv8",
                             "fig13", "evictor", "costmodel", "kv_append"])
    ap.add_argument("--no-secondary", action="store_true")
    args = ap.parse_args()
    rank, world, local_rank = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1), _env_int("LOCAL_RANK", 0)
    if args.impl == "reference":
        run_reference(args, rank, world)
    elif args.workload == "fig13":
        if rank == 0:
            run_fig13(args)
    elif args.workload == "evictor":
        if rank == 0:
            run_evictor(args)
    elif args.workload == "costmodel":
        if rank == 0:
            run_costmodel(args)
    elif args.workload == "kv_append":
        if rank == 0:
            run_kv_append(args)
    else:
        run_mine(args, rank, world, local_rank)


if __name__ == "__main__":
    main()

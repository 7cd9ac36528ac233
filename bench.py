#!/usr/bin/env python
"""bench.py -- the dyplan hot path on N B200s of one node (contract: the task statement / DESIGN.md section 9).

A "step" is one pass of the whole hot path (K_stage -> K_seed -> K_plan -> K_fscore / K_score with the fused final
reduce and bundle emission) over one batch of synthetic requests.  With no flags the run covers ALL FIVE configurations
of BASELINE.json in one process (`"configs": [...]` in the JSON line, one entry each: Geval/s, plans/s, requests/s,
ms_per_step, kernel_ms, roofline, e2e through the *_host C-ABI call, cpu_baseline = the oracle on a bounded sample),
plus a wide-class line (configs[1] with latencies x 3000: requests beyond the fp32 scorer's plain range), an int32-scorer
line (configs[1] with one zero-factor option per request: the requests only k_score takes) and the
variant selector (selects/s after configs[1], [2], [4]).  The headline `value` / `ms_per_step` / `config.workload` are
those of the largest single-GPU configuration, configs[4] (2.79e11 (plan, level) evaluations per step).  Requests are
independent, so with N > 1 every rank compiles its own batch of the same shape (different seed) and no data-path
collective exists ("scaling": "weak").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--configs 0,1,2,3,4] [--impl dyplan|reference]

`--gpus N` without a torch.distributed environment re-launches itself as N ranks (torch.distributed.run, 127.0.0.1).
`--impl reference` times the fp64 CPU oracle (oracle/, test infrastructure) on the host cores on the headline config's
cpu_baseline sample.  Prints ONE JSON line on stdout (rank 0).
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import socket
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
sys.path.insert(1, os.path.join(ROOT, "tests"))    # tests/support/workloads.py: the seeded input generator

METRIC = "plan_level_evaluations_per_s"
UNIT = "Geval/s"
SM_LANES = 128            # FP32/INT32 lanes per SM = 4 SMSPs x 32 (one warp instruction per clock per SMSP)
HEADLINE_CFG = 4
ALL_CFGS = (0, 1, 2, 3, 4)
WIDE_FACTOR = 3000        # wide leg: configs[1] with every latency x 3000 (seconds)
ORACLE_SAMPLE_EVALS = 2.2e9   # per config: about 7 s of the oracle on 16 host threads (0.3 Geval/s)
# dram__bytes_read.sum + dram__bytes_write.sum of the scoring kernel per launch come from the committed ncu capture
# summary named here (one row per workload, from `ncu --set full` reports; each row names the commit it was captured at).
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r2_scorer_dram_bytes.csv")


def alg_ops_per_eval(w) -> float:
    """Algorithmic thread-instructions per (plan, level) evaluation, SURVEY.md 8(d) D.4 / DESIGN.md section 9:
    per (plan, level) one add(-max), one SLO compare, one best compare; per plan one multiply, one demand add and
    B cap compares (only when caps exist); outer-digit repairs are amortised by 1/K and not counted."""
    nb = w.batch.B if w.batch.cap is not None else 0
    per_plan = 1.0 + (1.0 + nb if nb else 0.0)
    return 3.0 + per_plan / w.L


def committed_traffic(tag: str):
    """(bytes per launch, source) of the scoring kernel for workload `tag` from profiles/r2_scorer_dram_bytes.csv."""
    try:
        with open(TRAFFIC_CSV) as f:
            for row in csv.DictReader(l for l in f if not l.startswith("#")):
                if row["workload"] == tag:
                    return float(row["dram_bytes_per_launch"]), \
                        f"profiles/{os.path.basename(TRAFFIC_CSV)} ({row['kernel']}, captured at commit {row['commit']})"
    except (OSError, KeyError, ValueError):
        pass
    return None, None


class ClockSampler:
    """SM clock / power / throttle reasons DURING the timed regions, via NVML (the same counters as the
    B200_PROFILING.md nvidia-smi clocks line), sampled every few ms because a timed region lasts tens of ms.
    resume() / pause() bracket each timed region, so idle gaps between legs are not sampled."""
    REASONS = (("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20),
               ("sw_power_cap", 0x4))

    def __init__(self, index: int, period_s: float = 0.004):
        self.index, self.period, self.rows, self._stop, self._t, self.h, self.nv = index, period_s, [], threading.Event(), None, None, None
        self._on = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = index
            if vis:
                ids = [x for x in vis.split(",") if x.strip() != ""]
                if index < len(ids) and ids[index].strip().isdigit():
                    phys = int(ids[index])
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.nv = pynvml
        except Exception:
            self.h = None

    def max_sm_mhz(self, default: float = 1965.0) -> float:
        try:
            return float(self.nv.nvmlDeviceGetMaxClockInfo(self.h, self.nv.NVML_CLOCK_SM))
        except Exception:
            return default

    def _sample(self):
        nv, h = self.nv, self.h
        try:
            self.rows.append((nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM), nv.nvmlDeviceGetPowerUsage(h) / 1000.0,
                              nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)))
        except Exception:
            pass

    def _run(self):
        while not self._stop.is_set():
            if self._on.is_set():
                self._sample()
            self._stop.wait(self.period)

    def start(self):
        if self.h is None:
            return
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()

    def resume(self):
        self._on.set()

    def pause(self):
        self._on.clear()

    def stop(self) -> dict:
        self._stop.set()
        if self._t:
            self._t.join(timeout=2)
        if self.h is None or not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        mask = 0
        for r in self.rows:
            mask |= r[2]
        return {"sm_mhz": statistics.median(r[0] for r in self.rows), "sm_min_mhz": min(r[0] for r in self.rows),
                "sm_max_mhz": self.max_sm_mhz(None), "power_w_max": max(r[1] for r in self.rows), "samples": len(self.rows),
                "reasons": [n for n, bit in self.REASONS if mask & bit]}


def make_workload(cfg: int, rank: int, requests: int | None, wide=False):
    from support import workloads as wl
    # rank 0 runs the config's own seed; other ranks an independent batch of the same shape
    from paper_2607_02942_b200.multi import rank_seed
    w = wl.make_config(cfg, R=requests, seed=rank_seed(cfg, rank))
    if wide == "int32":
        # one zero-factor option per request (v = 1, a = 0: that option gives C = 0): the fp32 screen needs C32 > 0 for
        # real plans, so k_stage routes every such request to the int32 scorer k_score
        b = w.batch
        for r in range(b.R):
            n = int(b.node_off[r]) + (r % b.n_nodes(r))
            b.vuln[n] = 1.0
            b.acc[int(b.opt_off[n])] = 0.0
        w.name = w.name + " with one zero-factor option per request"
    elif wide:
        # the paper's own latencies are seconds to minutes per request (Fig. 2: 4.2 s ... 414.5 s): scale
        # every duration and the SLO so that the requests leave the fp32 scorer's plain exact-integer range
        w.batch.lat_us = (w.batch.lat_us.astype(np.int64) * WIDE_FACTOR).astype(np.int32)
        w.batch.slo_us = (w.batch.slo_us.astype(np.int64) * WIDE_FACTOR).astype(np.int32)
        w.name = w.name + f" x{WIDE_FACTOR} latencies"
    return w


def workload_tag(cfg: int, wide) -> str:
    return f"cfg{cfg}" + ("_int32" if wide == "int32" else "_wide" if wide else "")


def workload_label(cfg: int, wide) -> str:
    if wide == "int32":
        return f"BASELINE.json configs[{cfg}] with one zero-factor option per request (int32 scorer k_score)"
    return f"BASELINE.json configs[{cfg}]" + (f" with latencies x {WIDE_FACTOR} (seconds, PAPER.md:68)" if wide else "")


def oracle_sample(w):
    """(sub-workload, description): a bounded sample of `w` for the CPU legs.  The oracle enumerates whole requests:
    the first requests of the workload are taken until their (plan, level) evaluations pass ORACLE_SAMPLE_EVALS; when
    ONE request is already much larger (configs[4]: 6^12 x 8 = 1.7e10), request 0 is scored at pressure level 0 only."""
    from dataclasses import replace
    R = w.batch.R
    tot, keep = 0, 0
    for r in range(R):
        e = w.subset([r]).n_plans_total() * w.L
        if keep and tot + e > ORACLE_SAMPLE_EVALS:
            break
        tot += e
        keep += 1
        if tot > ORACLE_SAMPLE_EVALS:
            break
    sub = w.subset(list(range(keep)))
    if keep == 1 and tot > 2 * ORACLE_SAMPLE_EVALS and w.kind == "compile" and w.L > 1:
        sub = replace(sub, L=1, mult_pm=np.ascontiguousarray(np.asarray(w.mult_pm).reshape(w.L, w.batch.B)[0]))
        return sub, f"request 0 of {R}, every plan, pressure level 0 of {w.L}"
    return sub, f"first {keep} of {R} requests, every plan, all {w.L} levels"


def time_oracle(w_sample):
    from oracle import oracle
    oracle.build()
    t0 = time.perf_counter()
    oracle.run(w_sample)
    dt = time.perf_counter() - t0
    plans = w_sample.n_plans_total()
    return dt, plans * w_sample.L, oracle.num_threads()


def headline_config(cfg: int, w, world: int) -> dict:
    """The `config` object of the JSON line -- identical in the dyplan arm and the reference arm."""
    return {"workload": workload_label(cfg, False), "requests_per_gpu": int(w.batch.R), "plans_per_gpu": int(w.n_plans_total()),
            "levels": int(w.L), "l2": "flushed between timed iterations (256 MiB fill)",
            "parallelism": f"independent request batches x{world}, no collective"}


def run_reference(args, rank: int, world: int):
    """--impl reference: the oracle as it stands on the host cores (rank 0 only), on the SAME bounded sample of the
    headline workload that the dyplan arm's cpu_baseline leg times."""
    if rank != 0:
        return
    cfg = args.headline
    w = make_workload(cfg, 0, args.requests)
    sample, what = oracle_sample(w)
    from oracle import oracle
    oracle.build()
    from support import workloads as wl
    tiny = wl.make_config(0)
    for _ in range(args.warmup):
        oracle.run(tiny)                 # warm-up: library load and thread pool (the oracle keeps no state between runs)
    tot, evals, cores = 0.0, 0, 1
    for _ in range(args.steps):
        dt, ev, cores = time_oracle(sample)
        tot += dt
        evals += ev
    v = evals / tot / 1e9
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64+int64", "data": "synthetic",
        "config": headline_config(cfg, w, world),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{what} per step; warm-up steps run configs[0]"},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "requests_per_s": sample.batch.R * args.steps / tot,
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def pinned_host_call(binding, ctx, torch, w, stream):
    """The *_host C-ABI call on pinned HOST buffers: returns (callable, pinned output tensors, keep-alive)."""
    hb = binding.make_batch(w.batch, None)
    keep = {}
    for k, a in hb.arrays.items():
        if a is None:
            continue
        t = torch.from_numpy(a.view({np.dtype(np.uint32): np.int32}.get(a.dtype, a.dtype))).pin_memory()
        keep[k] = t
        setattr(hb.cstruct, k, t.data_ptr())
    hout = binding.alloc_bundle(w.batch.R, w.L, w.batch.B, None, True)
    pin_out = {}
    for k, a in hout.arrays.items():
        t = torch.from_numpy(a.view({np.dtype(np.uint64): np.int64}.get(a.dtype, a.dtype))).pin_memory()
        pin_out[k] = t
        setattr(hout.cstruct, k, t.data_ptr())

    def pin(a, dt):
        return torch.from_numpy(np.ascontiguousarray(a, dtype=dt).view(np.int32 if dt == np.uint32 else dt)).pin_memory()

    if w.kind == "compile":
        hm = pin(w.mult_pm, np.int32)
        call = lambda: ctx.dyplan_compile_host(hb, w.L, hm, hout, stream)
        keep["m"] = hm
    else:
        hm, hd, hf = pin(w.live_mult_pm, np.int32), pin(w.dispatched_mask, np.uint32), pin(w.fixed_choice, np.uint8)
        call = lambda: ctx.dyplan_replan_host(hb, hd, hf, hm, int(w.flags), hout, stream)
        keep["m"] = (hm, hd, hf)
    return call, pin_out, (hb, hout, keep)


def bench_one(args, ctx, binding, torch, dist, dev, rank, world, cfg, wide, peaks, sampler, flush, stream, prune_flags):
    """Device-resident leg + end-to-end leg of one workload.  Returns (entry for rank 0 | None, workload, device buffers)."""
    from paper_2607_02942_b200.multi import max_over_ranks, whole_job_rate
    w = make_workload(cfg, rank, args.requests, wide)
    dw = binding.upload(w, dev, corr64=True)
    plans = w.n_plans_total()
    evals = plans * w.L

    def barrier():
        if world > 1:
            dist.barrier()

    # ---- device-resident leg ---------------------------------------------------------------------------------
    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            binding.launch(ctx, dw, stream)
        stream.synchronize()
        st = ctx.dyplan_last_stats()
        # dominance pruning shrinks the enumerated space; stats report the plans actually enumerated
        assert st["plans"] == plans or (prune_flags & binding.PRUNE_DOMINATED and st["plans"] <= plans), (st, plans)
        launches_per_step = st["launches"]
        barrier()
        torch.cuda.synchronize()
        sampler.resume()
        e0 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
        e1 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
        score_ms = []
        for i in range(args.steps):
            flush.fill_(i & 0xFF)                    # L2 flush between timed iterations (outside the event pair)
            e0[i].record(stream)
            binding.launch(ctx, dw, stream)
            e1[i].record(stream)
            score_ms.append(ctx.dyplan_last_stats()["score_ms"])   # syncs the stream; the scorers' own event pair
        torch.cuda.synchronize()
        sampler.pause()
        barrier()
        step_ms = [a.elapsed_time(b) for a, b in zip(e0, e1)]

    # ---- end-to-end leg: the *_host C-ABI call, pinned host buffers, copies inside the timed region -------------
    host_call, pin_out, _keep = pinned_host_call(binding, ctx, torch, w, stream)
    for _ in range(args.warmup):
        h2d, d2h = host_call()
    barrier()
    torch.cuda.synchronize()
    e2e_ms = 0.0
    sampler.resume()
    for i in range(args.steps):
        flush.fill_(i & 0xFF)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        h2d, d2h = host_call()                       # returns after the results are in the host buffers
        e2e_ms += 1e3 * (time.perf_counter() - t0)
    sampler.pause()
    barrier()
    # the host leg must reproduce the device leg bit for bit
    dres = dw.out.host()
    assert np.array_equal(dres["plan_idx"], pin_out["plan_idx"].numpy().view(np.uint64)), "host/device legs disagree"

    tot_ms, k_ms, e2e_ms = max_over_ranks([sum(step_ms), sum(score_ms), e2e_ms], device=dev)
    entry = None
    if rank == 0:
        k_eval_s = evals * args.steps / (k_ms * 1e-3)
        aops = alg_ops_per_eval(w)
        achieved = k_eval_s * aops / 1e12
        fast = bool(st.get("fast_requests", 0))
        kernel = "k_fscore" if fast else "k_score"
        traffic, traffic_src = committed_traffic(workload_tag(cfg, wide)) if args.requests is None else (None, None)
        entry = {
            "workload": workload_label(cfg, wide), "cfg": cfg, "wide": wide, "name": w.name, "kind": w.kind,
            "requests_per_gpu": int(w.batch.R), "plans_per_gpu": int(plans), "levels": int(w.L),
            "fast_requests": int(st.get("fast_requests", 0)), "approx_requests": int(st.get("approx_requests", 0)),
            "value": whole_job_rate(evals, world, args.steps, tot_ms) / 1e9, "unit": UNIT,
            "ms_per_step": tot_ms / args.steps, "kernel_ms": k_ms / args.steps,
            "plans_per_s": world * plans * args.steps / (tot_ms * 1e-3),
            "requests_per_s": world * w.batch.R * args.steps / (tot_ms * 1e-3),
            "e2e": {"value": world * evals * args.steps / (e2e_ms * 1e-3) / 1e9, "unit": UNIT,
                    "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms / args.steps,
                    "api": "dyplan_compile_host" if w.kind == "compile" else "dyplan_replan_host"},
            "gpu_launches": launches_per_step * args.steps,
            "roofline": {"bound": "alu", "kernel": kernel, "achieved": achieved, "unit": "Tinst/s",
                         "peak": peaks["peak"], "frac": achieved / peaks["peak"],
                         "peak_nominal": peaks["peak_nominal"], "frac_of_nominal": achieved / peaks["peak_nominal"],
                         "traffic": traffic, "traffic_source": traffic_src,
                         "ops_per_eval": aops, "kernel_ms": k_ms / args.steps},
        }
        if prune_flags:
            # DESIGN.md 7.8/7.9: records identical to the exhaustive run, but plans are skipped, so `value` counts the
            # (plan, level) evaluations COVERED, not executed: not the headline metric and no roofline claim.
            entry["pruning"] = f"{args.prune} (exact; value = evaluations covered, not executed; not the headline)"
            entry["bound_skipped_outer"] = int(st.get("bound_skipped", 0))
            entry["plans_enumerated_per_gpu"] = int(st["plans"])
            entry["roofline"]["frac"] = entry["roofline"]["achieved"] = entry["roofline"]["frac_of_nominal"] = None
    return entry, w, dw


def select_leg(args, ctx, binding, torch, dev, rank, w, dw, stream):
    """S8: after a compile, 100 live multiplier vectors ~ U{1000..4000}: dyplan_select, parity against the oracle's
    selector on every vector, selects/s on the device."""
    rng = np.random.default_rng(4242 + rank)
    b = w.batch
    lives = rng.integers(1000, 4001, size=(100, b.B)).astype(np.int32)
    d_lives = torch.from_numpy(lives).to(dev)
    variant = torch.full((100, b.R), -9, dtype=torch.int32, device=dev)
    with torch.cuda.stream(stream):
        for i in range(3):
            ctx.dyplan_select(dw.batch, dw.out, w.L, d_lives[i], variant[i], None, stream)
        stream.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for i in range(100):
            ctx.dyplan_select(dw.batch, dw.out, w.L, d_lives[i], variant[i], None, stream)
        e1.record(stream)
        stream.synchronize()
    ms = e0.elapsed_time(e1)
    out = {"live_vectors": 100, "requests": int(b.R), "levels": int(w.L), "selects_per_s": 100 * b.R / (ms * 1e-3),
           "us_per_call": 1e3 * ms / 100, "gpu_launches": 100}
    if rank == 0 and not args.no_cpu_baseline:
        from oracle import oracle
        g = dw.out.host()
        v = variant.cpu().numpy()
        for i in range(100):
            rs = oracle.select(b, w.L, g["choice"], g["status"], lives[i])
            assert np.array_equal(v[i], rs["variant"]), f"select parity, live vector {i}"
        out["parity"] = "identical to the oracle's selector on all 100 vectors"
    return out


def measured_peaks(ctx, sm_count: int, sm_max_mhz: float) -> dict:
    """M0 (dyplan_measure_issue_rates): the issue rates measured on this device, and the peaks derived from them."""
    ctx.dyplan_measure_issue_rates()                      # warm-up pass (clocks)
    rates, mhz = ctx.dyplan_measure_issue_rates()
    by = {r["name"]: r["rate"] for r in rates}
    full = max(by.get("FFMA", 0.0), by.get("FADD.SAT", 0.0), by.get("FMUL", 0.0))
    mix = next((r["rate"] for r in rates if r["name"].startswith("mix: 2 FADD.SAT")), None)
    nominal = sm_count * SM_LANES * sm_max_mhz * 1e6 / 1e12
    return {"peak_nominal": nominal, "peak": nominal * full, "full_rate": full, "mix_rate": mix,
            "mix_ceiling": nominal * mix if mix else None, "sm_clock_mhz_observed": mhz,
            "rates": {r["name"]: round(r["rate"], 4) for r in rates}}


def run_dyplan(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist
    from paper_2607_02942_b200 import binding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the dyplan path has no CPU fallback)")
    if local_rank >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: rank {rank} needs cuda:{local_rank} but only {torch.cuda.device_count()} device(s) are visible")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    ctx = binding.Context(local_rank)
    prune_flags = {"none": 0, "dominated": binding.PRUNE_DOMINATED, "bounds": binding.PRUNE_BOUNDS,
                   "both": binding.PRUNE_DOMINATED | binding.PRUNE_BOUNDS}[args.prune]
    if prune_flags:
        ctx.dyplan_set_flags(prune_flags)
    stream = torch.cuda.Stream(device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2
    sampler = ClockSampler(local_rank)
    sampler.start()
    sm_count = ctx.dyplan_last_stats()["sm_count"]
    sm_max = sampler.max_sm_mhz(1965.0)
    peaks = measured_peaks(ctx, sm_count, sm_max)

    legs = [(c, False) for c in args.cfg_list]
    if args.wide and not prune_flags:
        legs.append((1, True))
        legs.append((1, "int32"))
    entries, selects = [], []
    for cfg, wide in legs:
        entry, w, dw = bench_one(args, ctx, binding, torch, dist, dev, rank, world, cfg, wide, peaks, sampler, flush, stream, prune_flags)
        if not wide and cfg in (1, 2, 4) and not args.no_select and w.kind == "compile" and not prune_flags:
            s = select_leg(args, ctx, binding, torch, dev, rank, w, dw, stream)
            s["after"] = workload_label(cfg, False)
            selects.append(s)
        if rank == 0:
            if world == 1 and not args.no_cpu_baseline:
                sample, what = oracle_sample(w)
                dt, ev, cores = time_oracle(sample)
                entry["cpu_baseline"] = {"value": ev / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
                                         "sample": f"{what} ({dt:.1f} s)"}
            entries.append(entry)
        del dw
    clocks = sampler.stop()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    head = next((e for e in entries if e["cfg"] == args.headline and not e["wide"]), entries[0])
    hw = make_workload(head["cfg"], 0, args.requests)
    line = {
        "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32+f32", "data": "synthetic",
        "config": headline_config(head["cfg"], hw, world),
        "plans_per_s": head["plans_per_s"], "requests_per_s": head["requests_per_s"],
        "e2e": head["e2e"],
        "gpu_launches": head["gpu_launches"],
        "gpu_launches_all_legs": sum(e["gpu_launches"] for e in entries) + sum(s["gpu_launches"] for s in selects),
        "clocks": clocks,
        "roofline": dict(head["roofline"],
                         peak_how=f"{sm_count} SMs x 128 lanes x {sm_max:.0f} MHz x {peaks['full_rate']:.3f} warp-inst/clk/SMSP measured "
                                  f"on this device (dyplan_measure_issue_rates: FFMA / FADD.SAT / FMUL chains); "
                                  f"peak_nominal = 1.0 warp-inst/clk/SMSP; DESIGN.md section 9",
                         mix_ceiling=peaks["mix_ceiling"], mix_rate=peaks["mix_rate"],
                         sm_clock_mhz_observed=peaks["sm_clock_mhz_observed"], issue_rates=peaks["rates"]),
        "configs": entries,
        "select": selects,
    }
    if "cpu_baseline" in head:
        line["cpu_baseline"] = head["cpu_baseline"]
    for k in ("pruning", "bound_skipped_outer", "plans_enumerated_per_gpu"):
        if k in head:
            line[k] = head[k]
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


LINEAR_PARAMS = dict(lambda_f=0.5, lambda_c=0.1, lambda_l=0.0002, lambda_ld=0.0001, beta=0.5, effort=1.0)
LINEAR_LEVELS = [0.0, 1.5, 3.0]          # the paper's levels


def run_linear(args, rank: int, world: int, local_rank: int):
    """--objective linear: dyplan_compile_linear (the paper's Eq.(4)/(5)) on the configured shape, cost ~ U[0,1]."""
    import torch
    import torch.distributed as dist
    from paper_2607_02942_b200 import binding
    from paper_2607_02942_b200.multi import max_over_ranks, whole_job_rate
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the dyplan path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    ctx = binding.Context(local_rank)
    cfg = args.cfg_list[0] if len(args.cfg_list) == 1 else 1
    w = make_workload(cfg, rank, args.requests)
    b = w.batch
    cost = np.random.default_rng(7 + rank).uniform(0.0, 1.0, size=b.lat_us.size).astype(np.float32)
    L = len(LINEAR_LEVELS)
    plans = w.n_plans_total()
    evals = plans * L
    stream = torch.cuda.Stream(device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    db = binding.make_batch(b, dev)
    out = binding.alloc_bundle(b.R, L, b.B, dev, True)
    dcost = torch.from_numpy(cost).to(dev)
    sampler = ClockSampler(local_rank)
    sampler.start()
    sm_count = ctx.dyplan_last_stats()["sm_count"]
    peaks = measured_peaks(ctx, sm_count, sampler.max_sm_mhz(1965.0))
    with torch.cuda.stream(stream):
        for _ in range(max(args.warmup, 3)):
            ctx.dyplan_compile_linear(db, dcost, LINEAR_PARAMS, LINEAR_LEVELS, out, stream=stream)
        stream.synchronize()
        st = ctx.dyplan_last_stats()
        assert st["plans"] == plans, (st, plans)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        sampler.resume()
        e0 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
        e1 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
        for i in range(args.steps):
            flush.fill_(i & 0xFF)
            e0[i].record(stream)
            ctx.dyplan_compile_linear(db, dcost, LINEAR_PARAMS, LINEAR_LEVELS, out, stream=stream)
            e1[i].record(stream)
        torch.cuda.synchronize()
        clocks = sampler.stop()
        tot_ms = sum(a.elapsed_time(c) for a, c in zip(e0, e1))
    # end to end through the C ABI's host call: pinned host arrays in, records in pinned host arrays out
    hb = binding.make_batch(b, None)
    keep = []
    for k, a in hb.arrays.items():
        if a is None:
            continue
        t = torch.from_numpy(a.view({np.dtype(np.uint32): np.int32}.get(a.dtype, a.dtype))).pin_memory()
        keep.append(t)
        setattr(hb.cstruct, k, t.data_ptr())
    hout = binding.alloc_bundle(b.R, L, b.B, None, True)
    pin_out = {}
    for k, a in hout.arrays.items():
        t = torch.from_numpy(a.view({np.dtype(np.uint64): np.int64}.get(a.dtype, a.dtype))).pin_memory()
        pin_out[k] = t
        setattr(hout.cstruct, k, t.data_ptr())
    pcost = torch.from_numpy(cost).pin_memory()
    h2d = d2h = 0
    e2e_ms = 0.0
    for i in range(args.steps + 1):
        flush.fill_(i & 0xFF)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        h2d, d2h = ctx.dyplan_compile_linear_host(hb, pcost, LINEAR_PARAMS, LINEAR_LEVELS, hout, stream=stream)
        if i:
            e2e_ms += 1e3 * (time.perf_counter() - t0)
    assert np.array_equal(out.host()["plan_idx"], pin_out["plan_idx"].numpy().view(np.uint64)), "host/device legs disagree"
    tot_ms, e2e_ms = max_over_ranks([tot_ms, e2e_ms], device=dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    aops = 2.0 + 5.0 / L      # per (plan, level): FFMA + compare; per plan: add-min (2), two sums, one FFMA
    k_eval_s = evals * args.steps / (tot_ms * 1e-3)
    lin_traffic, lin_traffic_src = committed_traffic(f"linear_cfg{cfg}") if args.requests is None else (None, None)
    line = {
        "metric": METRIC, "value": whole_job_rate(evals, world, args.steps, tot_ms) / 1e9, "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": tot_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{cfg}] shapes ({w.name}) under the paper's linear objective "
                               f"Eq.(4)/(5), levels {LINEAR_LEVELS}, cost ~ U[0,1]", "requests_per_gpu": b.R,
                   "plans_per_gpu": plans, "levels": L, "l2": "flushed between timed iterations (256 MiB fill)"},
        "requests_per_s": world * b.R * args.steps / (tot_ms * 1e-3),
        "e2e": {"value": world * evals * args.steps / (e2e_ms * 1e-3) / 1e9, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms / args.steps, "api": "dyplan_compile_linear_host"},
        "gpu_launches": st["launches"] * args.steps, "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": "k_lscore", "achieved": k_eval_s * aops / 1e12, "peak": peaks["peak"],
                     "unit": "Tinst/s", "frac": k_eval_s * aops / 1e12 / peaks["peak"], "peak_nominal": peaks["peak_nominal"],
                     "traffic": lin_traffic, "traffic_source": lin_traffic_src, "ops_per_eval": aops, "kernel_ms": st["score_ms"]},
    }
    if world == 1 and not args.no_cpu_baseline:
        from oracle import linear as lo
        nthr = os.cpu_count() or 1
        nreq = min(b.R, nthr)        # the oracle's OpenMP loop runs one request per thread: a sample that fills the host cores
        sub = w.subset(list(range(nreq)))
        c0 = cost[: sub.batch.lat_us.size]
        t0 = time.perf_counter()
        lo.compile(sub.batch, c0, LINEAR_PARAMS, LINEAR_LEVELS)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": sub.n_plans_total() * L / dt / 1e9, "unit": UNIT, "cores": nreq, "kind": "oracle",
                                "sample": f"first {nreq} of {b.R} requests, every plan, all levels ({dt:.1f} s; one request per thread)"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--configs", default=None, help="comma-separated BASELINE.json configs indices (default: all five)")
    ap.add_argument("--config", type=int, default=None, help="one config only (it is then the headline)")
    ap.add_argument("--requests", type=int, default=None, help="override the request count (down-scaled runs)")
    ap.add_argument("--impl", default="dyplan", choices=["dyplan", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-select", action="store_true")
    ap.add_argument("--no-wide", dest="wide", action="store_false", help="skip the configs[1] x 3000-latency leg and the int32-scorer leg")
    ap.add_argument("--objective", default="product", choices=["product", "linear"],
                    help="product: north_star's constrained objective (default); linear: the paper's Eq.(4)/(5)")
    ap.add_argument("--prune", default="none", choices=["none", "dominated", "bounds", "both"],
                    help="opt-in exact pruning (DESIGN.md 7.8/7.9); the default, headline line never prunes")
    args = ap.parse_args()
    if args.config is not None:
        args.cfg_list = [args.config]
        args.wide = False
    elif args.configs:
        args.cfg_list = [int(x) for x in args.configs.split(",")]
    else:
        args.cfg_list = list(ALL_CFGS)
    args.headline = HEADLINE_CFG if HEADLINE_CFG in args.cfg_list else args.cfg_list[-1]
    args.warmup = max(args.warmup, 3) if args.impl == "dyplan" else args.warmup
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")

    # --gpus N outside a torch.distributed launch: start the N ranks ourselves (one process per GPU, 127.0.0.1)
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        if args.impl == "dyplan" or args.objective == "linear":
            import torch
            n = torch.cuda.device_count() if torch.cuda.is_available() else 0
            if n < args.gpus:
                raise SystemExit(f"bench.py: --gpus {args.gpus} requested but {n} CUDA device(s) are visible")
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world} (launch one rank per GPU)")
    if args.objective == "linear":
        run_linear(args, rank, world, local_rank)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_dyplan(args, rank, world, local_rank)


if __name__ == "__main__":
    main()

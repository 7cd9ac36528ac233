#!/usr/bin/env python
"""bench.py -- the dyplan hot path on N B200s of one node (contract: see the task statement / DESIGN.md section 9).

A "step" is one pass of the whole hot path (K_stage -> K_plan -> K_fscore / K_score with the fused final reduce and
bundle emission) over one batch of synthetic requests: BASELINE.json configs[1] by default (256 requests, 8-node layered
DAGs, 8 options per node, 4 pressure levels: 4.29e9 plans, 1.72e10 (plan, level) evaluations).  Requests are
independent, so with N > 1 every rank compiles its own batch of the same shape (different seed) and no data-path
collective exists ("scaling": "weak").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl dyplan|reference]

`--impl reference` times the fp64 CPU oracle (oracle/, test infrastructure) on the host cores instead.
Prints ONE JSON line on stdout (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "plan_level_evaluations_per_s"
UNIT = "Geval/s"
SM_LANES = 128            # FP32/INT32 lanes per SM = 4 SMSPs x 32 (one warp instruction per clock per SMSP)
# dram__bytes_read.sum + dram__bytes_write.sum of the scoring kernel, per launch, from the `ncu --set full` captures of
# profiles/r1g_k_fscore.md (bytes).  The kernel is issue-bound; this is reported to show the traffic is negligible
# (cfg4's is local-memory write-back).  None for a workload that was not captured (cfg0, down-scaled runs).
NCU_DRAM_BYTES = {1: 13.85e6, 2: 33.97e6, 3: 94.34e6, 4: 232.98e6}


def alg_ops_per_eval(w) -> float:
    """Algorithmic thread-instructions per (plan, level) evaluation, SURVEY.md 8(d) D.4 / DESIGN.md section 9:
    per (plan, level) one add(-max), one SLO compare, one best compare; per plan one multiply, one demand add and
    B cap compares (only when caps exist); outer-digit repairs are amortised by 1/K and not counted."""
    nb = w.batch.B if w.batch.cap is not None else 0
    per_plan = 1.0 + (1.0 + nb if nb else 0.0)
    return 3.0 + per_plan / w.L


class ClockSampler:
    """SM clock / power / throttle reasons DURING the timed region, via NVML (the same counters as the
    B200_PROFILING.md nvidia-smi clocks line), sampled every few ms because a timed region lasts tens of ms."""
    REASONS = (("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20),
               ("sw_power_cap", 0x4))

    def __init__(self, index: int, period_s: float = 0.004):
        self.index, self.period, self.rows, self._stop, self._t, self.h, self.nv = index, period_s, [], threading.Event(), None, None, None
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

    def _sample(self):
        nv, h = self.nv, self.h
        try:
            self.rows.append((nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM), nv.nvmlDeviceGetPowerUsage(h) / 1000.0,
                              nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)))
        except Exception:
            pass

    def _run(self):
        while not self._stop.is_set():
            self._sample()
            self._stop.wait(self.period)

    def start(self):
        if self.h is None:
            return
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._t:
            self._t.join(timeout=2)
        if self.h is None or not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        try:
            mx = float(self.nv.nvmlDeviceGetMaxClockInfo(self.h, self.nv.NVML_CLOCK_SM))
        except Exception:
            mx = None
        mask = 0
        for r in self.rows:
            mask |= r[2]
        return {"sm_mhz": statistics.median(r[0] for r in self.rows), "sm_min_mhz": min(r[0] for r in self.rows),
                "sm_max_mhz": mx, "power_w_max": max(r[1] for r in self.rows), "samples": len(self.rows),
                "reasons": [n for n, bit in self.REASONS if mask & bit]}


def make_workload(cfg: int, rank: int, requests: int | None):
    from paper_2607_02942_b200 import workloads as wl
    # rank 0 runs the config's own seed; other ranks an independent batch of the same shape
    from paper_2607_02942_b200.multi import rank_seed
    return wl.make_config(cfg, R=requests, seed=rank_seed(cfg, rank))


ORACLE_SAMPLE_EVALS = 8e9   # about 25 s of the oracle on 16 host threads (0.3 Geval/s)


def oracle_sample(w, n_req: int):
    """The first n_req requests of the workload, cut where their (plan, level) evaluations pass ORACLE_SAMPLE_EVALS
    (a bounded sample for the CPU legs; the oracle enumerates whole requests, so at least one: configs[4]'s
    6^12 x 8 = 1.7e10 evaluations per request take it about a minute)."""
    n = min(n_req, w.batch.R)
    if n > 1:
        per = [w.subset([r]).n_plans_total() * w.L for r in range(n)]
        tot, keep = 0, 0
        for e in per:
            if keep and tot + e > ORACLE_SAMPLE_EVALS:
                break
            tot += e
            keep += 1
        n = keep
    return w.subset(list(range(n)))


def time_oracle(w_sample):
    from oracle import oracle
    oracle.build()
    t0 = time.perf_counter()
    oracle.run(w_sample)
    dt = time.perf_counter() - t0
    plans = w_sample.n_plans_total()
    return dt, plans * w_sample.L, oracle.num_threads()


def run_reference(args, rank: int, world: int):
    """--impl reference: the oracle as it stands on the host cores (rank 0 only)."""
    if rank != 0:
        return
    w = make_workload(args.config, 0, args.requests)
    sample = oracle_sample(w, args.ref_requests)
    for _ in range(args.warmup):
        time_oracle(oracle_sample(w, 1))
    tot, evals, cores = 0.0, 0, 1
    for _ in range(args.steps):
        dt, ev, cores = time_oracle(sample)
        tot += dt
        evals += ev
    v = evals / tot / 1e9
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64+int64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config}]", "sample": f"first {sample.batch.R} of {w.batch.R} requests per step"},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"first {sample.batch.R} of {w.batch.R} requests of configs[{args.config}], every plan, all levels"},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "requests_per_s": sample.batch.R * args.steps / tot,
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_dyplan(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist
    from paper_2607_02942_b200 import binding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the dyplan path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    ctx = binding.Context(local_rank)
    prune_flags = {"none": 0, "dominated": binding.PRUNE_DOMINATED, "bounds": binding.PRUNE_BOUNDS,
                   "both": binding.PRUNE_DOMINATED | binding.PRUNE_BOUNDS}[args.prune]
    if prune_flags:
        ctx.dyplan_set_flags(prune_flags)
    w = make_workload(args.config, rank, args.requests)
    dw = binding.upload(w, dev, corr64=True)
    stream = torch.cuda.Stream(device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2
    plans = w.n_plans_total()
    evals = plans * w.L

    def barrier():
        if world > 1:
            dist.barrier()

    # ---- device-resident leg -------------------------------------------------------------------------------
    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            binding.launch(ctx, dw, stream)
        stream.synchronize()
        st = ctx.dyplan_last_stats()
        # dominance pruning shrinks the enumerated space; stats report the plans actually enumerated
        assert st["plans"] == plans or (prune_flags & binding.PRUNE_DOMINATED and st["plans"] <= plans), (st, plans)
        launches_per_step = st["launches"]
        sampler = ClockSampler(local_rank)
        barrier()
        torch.cuda.synchronize()
        sampler.start()
        e0 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
        e1 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
        score_ms = []
        for i in range(args.steps):
            flush.fill_(i & 0xFF)                    # L2 flush between timed iterations (outside the event pair)
            e0[i].record(stream)
            binding.launch(ctx, dw, stream)
            e1[i].record(stream)
            score_ms.append(ctx.dyplan_last_stats()["score_ms"])   # syncs the stream; K_score's own event pair
        torch.cuda.synchronize()
        clocks = sampler.stop()
        barrier()
        step_ms = [a.elapsed_time(b) for a, b in zip(e0, e1)]
    tot_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device=dev)
    k_ms = torch.tensor([sum(score_ms)], dtype=torch.float64, device=dev)

    # ---- end-to-end leg: the *_host C-ABI call, pinned host buffers, copies inside the timed region -------------
    hb = binding.make_batch(w.batch, None)
    pinned = {}
    for k, a in hb.arrays.items():
        if a is None:
            continue
        t = torch.from_numpy(a.view({np.dtype(np.uint32): np.int32}.get(a.dtype, a.dtype))).pin_memory()
        pinned[k] = t
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
        host_call = lambda: ctx.dyplan_compile_host(hb, w.L, hm, hout, stream)
    else:
        hm, hd, hf = pin(w.live_mult_pm, np.int32), pin(w.dispatched_mask, np.uint32), pin(w.fixed_choice, np.uint8)
        host_call = lambda: ctx.dyplan_replan_host(hb, hd, hf, hm, int(w.flags), hout, stream)
    for _ in range(args.warmup):
        h2d, d2h = host_call()
    barrier()
    torch.cuda.synchronize()
    e2e_ms = 0.0
    for i in range(args.steps):
        flush.fill_(i & 0xFF)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        h2d, d2h = host_call()                       # returns after the results are in the host buffers
        e2e_ms += 1e3 * (time.perf_counter() - t0)
    barrier()
    e2e_t = torch.tensor([e2e_ms], dtype=torch.float64, device=dev)
    # the host leg must reproduce the device leg bit for bit
    dres = dw.out.host()
    assert np.array_equal(dres["plan_idx"], pin_out["plan_idx"].numpy().view(np.uint64)), "host/device legs disagree"

    from paper_2607_02942_b200.multi import max_over_ranks, whole_job_rate
    tot_ms, k_ms, e2e_ms = max_over_ranks([float(tot_ms), float(k_ms), float(e2e_t)], device=dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    sm_count = st["sm_count"]
    value = whole_job_rate(evals, world, args.steps, tot_ms) / 1e9
    k_eval_s = evals * args.steps / (k_ms * 1e-3)
    aops = alg_ops_per_eval(w)
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak = sm_count * SM_LANES * sm_max * 1e6 / 1e12            # T thread-inst/s at the max SM clock
    achieved = k_eval_s * aops / 1e12
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": tot_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32+f32", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config}] ({w.name})", "requests_per_gpu": w.batch.R,
                   "plans_per_gpu": plans, "levels": w.L, "l2": "flushed between timed iterations (256 MiB fill)",
                   "parallelism": f"independent request batches x{world}, no collective"},
        "plans_per_s": world * plans * args.steps / (tot_ms * 1e-3),
        "requests_per_s": world * w.batch.R * args.steps / (tot_ms * 1e-3),
        "e2e": {"value": world * evals * args.steps / (e2e_ms * 1e-3) / 1e9, "unit": UNIT,
                "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms / args.steps,
                "api": "dyplan_compile_host" if w.kind == "compile" else "dyplan_replan_host"},
        "gpu_launches": launches_per_step * args.steps,
        "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": "k_fscore" if st.get("fast_requests", 0) else "k_score", "achieved": achieved, "peak": peak, "unit": "Tinst/s",
                     "frac": achieved / peak,
                     "traffic": NCU_DRAM_BYTES.get(args.config) if args.requests is None else None,
                     "ops_per_eval": aops, "kernel_ms": k_ms / args.steps,
                     "peak_how": f"{sm_count} SMs x 128 lanes x {sm_max:.0f} MHz (B300_MICROARCH.md: 1 warp-inst/clk/SMSP); DESIGN.md section 9"},
    }
    if prune_flags:
        # DESIGN.md 7.8/7.9: records identical to the exhaustive run, but plans are skipped, so `value` counts the
        # (plan, level) evaluations COVERED, not executed: not the headline metric and no roofline claim.
        line["config"]["pruning"] = f"{args.prune} (exact; value = evaluations covered, not executed; not the headline)"
        line["bound_skipped_outer"] = int(st.get("bound_skipped", 0))
        line["plans_enumerated_per_gpu"] = int(st["plans"])
        line["roofline"]["frac"] = line["roofline"]["achieved"] = None
    if world == 1 and not args.no_cpu_baseline:
        sample = oracle_sample(w, args.cpu_requests)
        dt, ev, cores = time_oracle(sample)
        line["cpu_baseline"] = {"value": ev / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"first {sample.batch.R} of {w.batch.R} requests, every plan, all levels ({dt:.1f} s)"}
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
    w = make_workload(args.config, rank, args.requests)
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
    with torch.cuda.stream(stream):
        for _ in range(max(args.warmup, 3)):
            ctx.dyplan_compile_linear(db, dcost, LINEAR_PARAMS, LINEAR_LEVELS, out, stream=stream)
        stream.synchronize()
        st = ctx.dyplan_last_stats()
        assert st["plans"] == plans, (st, plans)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        sampler.start()
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
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak = st["sm_count"] * SM_LANES * sm_max * 1e6 / 1e12
    k_eval_s = evals * args.steps / (tot_ms * 1e-3)
    line = {
        "metric": METRIC, "value": whole_job_rate(evals, world, args.steps, tot_ms) / 1e9, "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": tot_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config}] shapes ({w.name}) under the paper's linear objective "
                               f"Eq.(4)/(5), levels {LINEAR_LEVELS}, cost ~ U[0,1]", "requests_per_gpu": b.R,
                   "plans_per_gpu": plans, "levels": L, "l2": "flushed between timed iterations (256 MiB fill)"},
        "requests_per_s": world * b.R * args.steps / (tot_ms * 1e-3),
        "e2e": {"value": world * evals * args.steps / (e2e_ms * 1e-3) / 1e9, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms / args.steps, "api": "dyplan_compile_linear_host"},
        "gpu_launches": st["launches"] * args.steps, "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": "k_lscore", "achieved": k_eval_s * aops / 1e12, "peak": peak,
                     "unit": "Tinst/s", "frac": k_eval_s * aops / 1e12 / peak, "traffic": None, "ops_per_eval": aops,
                     "kernel_ms": st["score_ms"]},
    }
    if world == 1 and not args.no_cpu_baseline:
        from oracle import linear as lo
        sub = w.subset([0])
        c0 = cost[: sub.batch.lat_us.size]
        t0 = time.perf_counter()
        lo.compile(sub.batch, c0, LINEAR_PARAMS, LINEAR_LEVELS)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": sub.n_plans_total() * L / dt / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"request 0 of {b.R}, every plan, all levels ({dt:.1f} s; one request runs on one core)"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index (default 1)")
    ap.add_argument("--requests", type=int, default=None, help="override the request count (down-scaled runs)")
    ap.add_argument("--impl", default="dyplan", choices=["dyplan", "reference"])
    ap.add_argument("--cpu-requests", type=int, default=32, help="oracle sample size of the cpu_baseline leg")
    ap.add_argument("--ref-requests", type=int, default=4, help="oracle sample size per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--objective", default="product", choices=["product", "linear"],
                    help="product: north_star's constrained objective (default); linear: the paper's Eq.(4)/(5)")
    ap.add_argument("--prune", default="none", choices=["none", "dominated", "bounds", "both"],
                    help="opt-in exact pruning (DESIGN.md 7.8/7.9); the default, headline line never prunes")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "dyplan" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.objective == "linear":
        run_linear(args, rank, world, local_rank)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_dyplan(args, rank, world, local_rank)


if __name__ == "__main__":
    main()

"""-m gpu: differential runs of the CUDA path against itself on many random shapes.

Every way the library has of computing the same bundle must give the same bytes: the admission path (k_small) and the
batched scorers, the exhaustive enumeration and the two exact prunings, the ctx's own scratch and the static scratch of
dyplan_compile_static.  No oracle here (tests/test_gpu_parity.py compares with it): the point is breadth -- a few
hundred shapes per run, with second-scale latencies (approx class) and zero-factor options (int32 scorer) mixed into
the batches -- at a cost of seconds.
"""
from __future__ import annotations

import numpy as np
import pytest

from support import workloads as wl

pytestmark = pytest.mark.gpu

KEYS = ("status", "plan_idx", "choice", "corr", "corr64", "lat", "dem", "dom_model")


@pytest.fixture(scope="module")
def dy():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    from paper_2607_02942_b200 import binding
    ctx = binding.Context(0)
    yield binding, ctx
    ctx.dyplan_set_flags(0)
    ctx.close()


def run(dy, w, flags, static=False):
    import torch
    binding, ctx = dy
    ctx.dyplan_set_flags(flags)
    dw = binding.upload(w, "cuda:0")
    for k in ("plan_idx", "corr", "lat", "status"):       # every record must be written by this call
        dw.out.arrays[k].fill_(0x5A if k == "status" else 77)
    if static:
        ctx.dyplan_compile_static(dw.batch, dw.L, dw.mult, dw.out)
    else:
        binding.launch(ctx, dw)
    torch.cuda.synchronize()
    return dw.out.host(), ctx.dyplan_last_stats()


def same(w, a, b, what, params):
    for k in KEYS:
        assert np.array_equal(a[k], b[k]), f"{what}: {k} differs for {params}"


def draw(rng, small_call: bool):
    R = int(rng.integers(1, 33)) if small_call else int(rng.integers(33, 400))
    L, B, caps = int(rng.integers(1, 9)), int(rng.integers(1, 9)), bool(rng.integers(0, 2))
    if small_call:
        nmax = int(rng.integers(1, 17))
        kmax = int(rng.integers(1, 17 if nmax <= 5 else (5 if nmax <= 9 else 3)))
    else:
        nmax = int(rng.integers(3, 9))
        kmax = int(rng.integers(2, 8 if nmax <= 6 else 5))
    seed, kind = int(rng.integers(0, 1 << 30)), int(rng.integers(0, 3))
    params = dict(R=R, L=L, B=B, caps=caps, nmax=nmax, kmax=kmax, seed=seed, kind=kind)
    if kind == 0:
        w = wl.random_workload(seed, R=R, nmin=1, nmax=nmax, kmin=1, kmax=kmax, B=B, M=3, L=L, caps=caps,
                               tool_p=float(rng.uniform(0, 0.4)), edge_p=float(rng.uniform(0.1, 0.8)), slo_q=float(rng.uniform(0.05, 0.95)))
    else:
        w = wl.random_replan_workload(seed, R=R, nmin=1, nmax=nmax, kmin=1, kmax=kmax, B=B, M=3, caps=caps,
                                      flags=(wl.FLAG_FIXED_IN_PLACE if kind == 1 else wl.FLAG_RESIDUAL))
    return w, params


def test_small_calls_every_path_gives_the_same_bytes(dy):
    binding, _ = dy
    rng = np.random.default_rng(20260711)
    n = smalls = 0
    for _ in range(250):
        w, params = draw(rng, small_call=True)
        if w.n_plans_total() > 2e8:
            continue
        a, st = run(dy, w, 0)
        same(w, a, run(dy, w, binding.NO_SMALL_PATH)[0], "k_small vs the batched scorers", params)
        same(w, a, run(dy, w, binding.NO_SMALL_PATH | binding.PRUNE_BOUNDS)[0], "exhaustive vs subtree bounds", params)
        if w.kind == "compile":
            same(w, a, run(dy, w, 0, static=True)[0], "ctx scratch vs static scratch", params)
        n += 1
        smalls += st["small_requests"]
    assert n >= 200 and smalls >= 1000


def test_batched_calls_every_path_gives_the_same_bytes(dy):
    binding, _ = dy
    rng = np.random.default_rng(20260712)
    n = approx = 0
    for _ in range(60):
        w, params = draw(rng, small_call=False)
        if w.n_plans_total() * w.L > 2e9:
            continue
        b = w.batch
        for r in range(0, b.R, 7):      # second-scale latencies (approx class) and zero factors (int32 scorer) in the same batch
            a0, e0 = int(b.opt_off[b.node_off[r]]), int(b.opt_off[b.node_off[r + 1]])
            if e0 <= a0:
                continue
            if r % 14 == 0:
                b.lat_us[a0:e0] = np.minimum(b.lat_us[a0:e0].astype(np.int64) * 3000, 2**30).astype(np.int32)
                b.slo_us[r] = int(min(int(b.slo_us[r]) * 3000, 2**31 - 1))
            else:
                nn = int(b.node_off[r])
                b.vuln[nn] = 1.0
                b.acc[int(b.opt_off[nn])] = 0.0
        a, st = run(dy, w, 0)
        same(w, a, run(dy, w, binding.PRUNE_BOUNDS)[0], "exhaustive vs subtree bounds", params)
        same(w, a, run(dy, w, binding.PRUNE_DOMINATED)[0], "exhaustive vs dominance pruning", params)
        if w.kind == "compile" and b.R <= binding.STATIC_MAX_REQUESTS:
            same(w, a, run(dy, w, 0, static=True)[0], "ctx scratch vs static scratch", params)
        n += 1
        approx += st["approx_requests"]
    assert n >= 40 and approx >= 40

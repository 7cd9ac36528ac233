"""-m gpu: dyplan_compile_static (include/dyplan.h) -- the compile call whose scratch is the library's file-scope
static device array, for callers that cannot call cudaMalloc -- against the existing dyplan_compile path.

The records must be identical bit for bit (same kernels, same launch geometry; only where the scratch lives and the
work-item budget differ, and neither changes a record).  The calls run back to back on ONE stream: they share the
array, which keeps the previous call's contents, so each case follows a call of a different shape.

This file is named to be collected last: the run uses `pytest -x`.
"""
from __future__ import annotations

import numpy as np
import pytest

from support import workloads as wl

pytestmark = pytest.mark.gpu

RECORD_KEYS = ("status", "plan_idx", "choice", "corr", "corr64", "lat", "dem", "dom_model")


@pytest.fixture(scope="module")
def dy():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    from paper_2607_02942_b200 import binding
    ctx = binding.Context(0)
    yield binding, ctx
    ctx.close()


def existing_path(binding, ctx, w):
    import torch
    dw = binding.upload(w, "cuda:0")
    binding.launch(ctx, dw)
    torch.cuda.synchronize()
    return dw.out.host()


def static_path(binding, ctx, w):
    import torch
    dw = binding.upload(w, "cuda:0")
    for k in ("plan_idx", "corr", "lat", "status"):      # poison the outputs: every record must be written by this call
        dw.out.arrays[k].fill_(0x5A if k == "status" else 77)
    ctx.dyplan_compile_static(dw.batch, dw.L, dw.mult, dw.out)
    torch.cuda.synchronize()
    return dw.out.host()


def assert_same(w, a, b, what):
    for k in RECORD_KEYS:
        assert np.array_equal(a[k], b[k]), f"{w.name}: {k} differs ({what})"


def cases():
    big = wl.random_workload(seed=9101, R=200, nmin=5, nmax=8, kmin=2, kmax=5, B=3, M=3, L=4)        # batched scorers
    small = wl.random_workload(seed=9102, R=5, nmin=3, nmax=6, kmin=2, kmax=4, B=2, M=3, L=3)         # k_small
    mixed = wl.make_config(1, R=3)                                                                    # R <= 32, too large for k_small
    nocap = wl.random_workload(seed=9103, R=64, nmin=4, nmax=9, kmin=1, kmax=4, B=2, M=2, L=8, caps=False)
    return [big, small, mixed, nocap]


def test_static_scratch_calls_in_a_row_match_the_existing_path(dy):
    binding, ctx = dy
    ws = cases()
    ref = [existing_path(binding, ctx, w) for w in ws]
    # two passes over the cases, every call on the same (default) stream, the array reused from call to call
    for rep in range(2):
        for w, r in zip(ws, ref):
            g = static_path(binding, ctx, w)
            assert_same(w, g, r, f"dyplan_compile_static vs dyplan_compile, pass {rep}")
            assert (r["status"] == 0).any(), w.name
    # the same workload twice in a row
    g1 = static_path(binding, ctx, ws[0])
    g2 = static_path(binding, ctx, ws[0])
    assert_same(ws[0], g1, ref[0], "first of two identical calls")
    assert_same(ws[0], g2, ref[0], "second of two identical calls")


def test_static_scratch_matches_the_oracle(dy, orc):
    from parity import check_records
    binding, ctx = dy
    w = wl.random_workload(seed=9104, R=6, nmin=3, nmax=5, kmin=2, kmax=4, B=2, M=3, L=3)
    static_path(binding, ctx, wl.make_config(0))          # a different call first
    g = static_path(binding, ctx, w)
    check_records(orc, w, g, orc.run(w), where="dyplan_compile_static")


def test_static_scratch_rejects_more_than_the_maximum(dy):
    binding, ctx = dy
    ok = wl.random_workload(seed=9105, R=binding.STATIC_MAX_REQUESTS, nmin=2, nmax=4, kmin=1, kmax=3, L=2)
    g = static_path(binding, ctx, ok)                      # exactly the maximum is accepted
    assert_same(ok, g, existing_path(binding, ctx, ok), "R = DYPLAN_STATIC_MAX_REQUESTS")
    over = wl.random_workload(seed=9106, R=binding.STATIC_MAX_REQUESTS + 1, nmin=2, nmax=3, kmin=1, kmax=2, L=2)
    dw = binding.upload(over, "cuda:0")
    with pytest.raises(binding.DyplanError) as e:
        ctx.dyplan_compile_static(dw.batch, dw.L, dw.mult, dw.out)
    assert e.value.code == binding.ERR_STATIC_LIMIT
    assert str(binding.STATIC_MAX_REQUESTS) in str(e.value) and str(over.batch.R) in str(e.value)
    assert ctx.dyplan_last_stats()["launches"] == 0


def test_static_scratch_call_allocates_no_device_memory(dy):
    import torch
    binding, _ = dy
    w = wl.random_workload(seed=9107, R=binding.STATIC_MAX_REQUESTS, nmin=4, nmax=7, kmin=2, kmax=4, B=3, M=3, L=4)
    ctx = binding.Context(0)       # a fresh ctx: it owns no scratch yet, so the existing path would have to cudaMalloc
    try:
        dw = binding.upload(w, "cuda:0")
        ctx.dyplan_compile_static(dw.batch, dw.L, dw.mult, dw.out)     # loads the kernels of this shape
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        for _ in range(3):
            ctx.dyplan_compile_static(dw.batch, dw.L, dw.mult, dw.out)
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        assert free0 - free1 < (1 << 20), (free0, free1)
        g = dw.out.host()
        # ... and the existing path on the same fresh ctx does allocate (about 15 MB for this call): the check can see it
        binding.launch(ctx, dw)
        torch.cuda.synchronize()
        free2, _ = torch.cuda.mem_get_info()
        assert free1 - free2 >= (4 << 20), (free1, free2)
        assert_same(w, g, dw.out.host(), "fresh ctx")
    finally:
        ctx.close()


def test_static_scratch_call_is_capturable_in_a_cuda_graph(dy):
    # the reason the entry point exists: nothing in it allocates, synchronises or records an event, so after one warm
    # call (symbol address, occupancy query, module load) the whole compile is capturable and replays bit for bit
    import torch
    binding, ctx = dy
    for w in (wl.random_workload(seed=9201, R=40, nmin=4, nmax=7, kmin=2, kmax=5, B=3, M=3, L=4), wl.make_config(0)):
        dw = binding.upload(w, "cuda:0")
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            ctx.dyplan_compile_static(dw.batch, dw.L, dw.mult, dw.out, s)
        s.synchronize()
        ref = {k: v.copy() for k, v in dw.out.host().items()}
        assert_same(w, ref, existing_path(binding, ctx, w), "warm static call")
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            ctx.dyplan_compile_static(dw.batch, dw.L, dw.mult, dw.out, s)
        for _ in range(3):
            for k in ("plan_idx", "corr", "lat", "status"):
                dw.out.arrays[k].fill_(0x5A if k == "status" else 77)
            g.replay()
            torch.cuda.synchronize()
            assert_same(w, dw.out.host(), ref, "graph replay")
